// generic_fft.cuh -- the transforms of H|psi> for ANY axis lengths N = 2^a 3^b (4 <= N <= 256): the general path behind
// the error contract of include/tdh.h (TDH_EUNSUPPORTED only for other prime factors or lengths outside that range).
//
// The tuned kernels (tile_kernels.cuh, xpencil_kernel.cuh) exist for the lengths of the BASELINE configs and their mixes
// (16, 32, 48, 64, 96 on every axis).  A grid with any other length (24, 36, 54, 72, 81, 108, 128, 144, ... -- the
// cutoff-derived grids of PAPER.md:106) runs the five launches below instead, each a batched 1-D transform of pencils
// staged through shared memory:
//     gfft z forward                  in   -> work
//     gfft y forward                  work -> work
//     gfft x forward, diagonal factor (kinetic + mask / Poisson / Teter), x inverse     work -> work    (as xpencil)
//     gfft y inverse                  work -> work
//     gfft z inverse + epilogue  out = alpha (T phi + V phi) + y                          work -> out     (as tile_inv)
// The non-local term uses nl_project / nl_scatter (nl_kernels.cuh), which do not depend on the grid lengths.
//
// TRANSFORM.  Stockham autosort, radices 4, 3, 2 from the factorisation of N, ping-pong between two shared-memory
// buffers [N][PT + 1] (PT pencils per CTA, one padding column: conflict-free both with the pencil index and with the
// element index fastest).  A stage of radix R with ns = product of the earlier radices: butterfly j < N/R, k = j mod ns,
//     v_t = x[j + t N/R] w^(k t N / (ns R)),  DFT_R,  y[(j - k) R + k + t ns] = v_t,      w = e^{-+2 pi i / N}
// and the result is in natural order, so the work layout of these grids is the natural one (identity row / column maps)
// and every table of the handle is in natural order.  Twiddles come from the handle's long-double tables.
#pragma once
#include "fft_codelets.cuh"
#include "tile_kernels.cuh"
#include "xpencil_kernel.cuh"

namespace tdh {

constexpr int GF_MAXFAC = 8;
constexpr int GF_THREADS = 256;

struct GAxis {
    int n;                  // transform length
    int nfac;
    int fac[GF_MAXFAC];     // radices, product = n
    int pt;                 // pencils per CTA (a power of two)
    int pt_log2;
    unsigned magic_n;       // ceil(2^32 / n): i / n = __umulhi(i, magic_n) for i < 2^24 (gfft_div)
    size_t stride;          // elements between consecutive points of a pencil
    size_t inner;           // pencil p starts at (p / inner) * outer + p % inner
    size_t outer;
    size_t npencils;
};

__host__ inline bool gfft_factor(int n, GAxis* ax) {
    if (n < 4 || n > 256) return false;
    int m = n, k = 0;
    while (m % 4 == 0 && k < GF_MAXFAC) { ax->fac[k++] = 4; m /= 4; }
    while (m % 3 == 0 && k < GF_MAXFAC) { ax->fac[k++] = 3; m /= 3; }
    while (m % 2 == 0 && k < GF_MAXFAC) { ax->fac[k++] = 2; m /= 2; }
    if (m != 1) return false;
    ax->n = n;
    ax->nfac = k;
    ax->pt = n <= 128 ? 16 : 8;
    ax->pt_log2 = n <= 128 ? 4 : 3;
    ax->magic_n = 0xFFFFFFFFu / (unsigned)n + 1u;
    return true;
}
constexpr int GF_MAXPT = 16;
// two ping-pong buffers, the twiddle table, and per pencil of the tile: its base offset and (state, ky, kz) / V offset
__host__ inline size_t gfft_smem(const GAxis& ax) {
    return ((size_t)2 * ax.n * (ax.pt + 1) + ax.n) * sizeof(cd) + GF_MAXPT * (sizeof(size_t) + sizeof(int4));
}

// Index arithmetic.  The lengths are run-time values, and a 32-bit division by one costs tens of instructions, a 64-bit
// one (pencil -> base offset) more than a hundred: per element of every load, stage and store loop that was the bound
// of these kernels (ncu r03: DRAM at 20 %, the SMs' issue slots at 58 %).  Divisions by n and by the stage's ns are
// multiplications by a precomputed reciprocal, pt is a power of two, and everything that depends on the pencil only
// (base offset, state, ky, kz) is computed once per pencil and tile into shared memory.
__device__ __forceinline__ int gfft_div(int i, unsigned magic) { return (int)__umulhi((unsigned)i, magic); }

template <int R, int DIR>
__device__ __forceinline__ void gfft_stage(const cd* __restrict__ x, cd* __restrict__ y, const cd* __restrict__ stw, int n,
                                           int ns, int pt, int ld, int npen) {
    const int nr = n / R, step = n / (ns * R);
    const unsigned mns = 0xFFFFFFFFu / (unsigned)ns + 1u;                // ns = 1: wraps to 0, handled below
    const int ptm = pt - 1, ptl = 31 - __clz(pt);
    for (int item = threadIdx.x; item < nr * pt; item += GF_THREADS) {
        const int q = item & ptm, j = item >> ptl;
        if (q >= npen) continue;
        const int k = ns == 1 ? 0 : j - gfft_div(j, mns) * ns;
        cd v[R];
        v[0] = x[j * ld + q];
#pragma unroll
        for (int t = 1; t < R; ++t) {
            const cd w = stw[k * t * step];                      // e^{+2 pi i k t / (ns R)}
            const cd a = x[(j + t * nr) * ld + q];
            v[t] = DIR > 0 ? cmul(a, w) : cmulc(a, w);
        }
        Dft<R, DIR>::run(v);
        const int j0 = (j - k) * R + k;
#pragma unroll
        for (int t = 0; t < R; ++t) y[(j0 + t * ns) * ld + q] = v[t];
    }
}

// all stages of one direction; returns the buffer that holds the result (natural order)
template <int DIR>
__device__ __forceinline__ cd* gfft_run(cd* a, cd* b, const cd* stw, const GAxis& ax, int npen) {
    const int ld = ax.pt + 1;
    int ns = 1;
    for (int f = 0; f < ax.nfac; ++f) {
        const int R = ax.fac[f];
        if (R == 4) gfft_stage<4, DIR>(a, b, stw, ax.n, ns, ax.pt, ld, npen);
        else if (R == 3) gfft_stage<3, DIR>(a, b, stw, ax.n, ns, ax.pt, ld, npen);
        else gfft_stage<2, DIR>(a, b, stw, ax.n, ns, ax.pt, ld, npen);
        __syncthreads();
        cd* t = a; a = b; b = t;
        ns *= R;
    }
    return a;
}

// load PT pencils into buf[e][q]; the thread mapping keeps global accesses contiguous for both pencil orientations
// sbase[q] = base offset of pencil q of the tile (gfft_tile_setup)
__device__ __forceinline__ void gfft_load(cd* buf, const cd* __restrict__ in, const GAxis& ax, const size_t* sbase, int npen) {
    const int ld = ax.pt + 1;
    if (ax.stride == 1) {
        for (int i = threadIdx.x; i < ax.n * npen; i += GF_THREADS) {
            const int q = gfft_div(i, ax.magic_n), e = i - q * ax.n;
            buf[e * ld + q] = lds_cd(in + sbase[q] + e);
        }
    } else {
        for (int i = threadIdx.x; i < ax.n * ax.pt; i += GF_THREADS) {
            const int q = i & (ax.pt - 1), e = i >> ax.pt_log2;
            if (q < npen) buf[e * ld + q] = lds_cd(in + sbase[q] + (size_t)e * ax.stride);
        }
    }
}

// once per tile, by the first pt threads: base offset of every pencil; with kin_nz > 0 also (state, ky, kz) of the
// x pencils for the diagonal factor; with npts > 0 the offset of the pencil's first point inside its state (index into V)
__device__ __forceinline__ void gfft_tile_setup(const GAxis& ax, size_t p0, int npen, size_t* sbase, int4* sinfo, int kin_nz,
                                                size_t npts) {
    const int q = threadIdx.x;
    if (q < npen) {
        const size_t p = p0 + q, hi = p / ax.inner, lo = p - hi * ax.inner;
        sbase[q] = hi * ax.outer + lo;
        int4 info = make_int4(0, 0, 0, 0);
        if (kin_nz > 0) { info.x = (int)hi; info.y = (int)(lo / (size_t)kin_nz); info.z = (int)(lo - (size_t)info.y * kin_nz); }
        if (npts > 0) info.w = (int)((p * (size_t)ax.n) % npts);
        sinfo[q] = info;
    }
}

// MODE -1: plain transform of direction DIR (no scaling).  Other modes (x axis only, DIR ignored) as xpencil_kernel:
// 0 forward + kinetic factor + inverse, 1 forward only, 2 inverse only times kin.scale, 3 Poisson factor, 4 Teter factor.
// in and out may be the same buffer: a CTA reads its pencils completely before it writes them.
template <int DIR, int MODE>
__global__ void __launch_bounds__(GF_THREADS)
gfft_axis_kernel(const cd* __restrict__ in, cd* __restrict__ out, const GAxis ax, const cd* __restrict__ tw, const Kinetic kin,
                 int nx)
{
    extern __shared__ __align__(16) unsigned char gsm[];
    cd* a = reinterpret_cast<cd*>(gsm);
    const int ld = ax.pt + 1;
    cd* b = a + (size_t)ax.n * ld;
    cd* stw = b + (size_t)ax.n * ld;
    size_t* sbase = reinterpret_cast<size_t*>(stw + ax.n);
    int4* sinfo = reinterpret_cast<int4*>(sbase + GF_MAXPT);
    for (int i = threadIdx.x; i < ax.n; i += GF_THREADS) stw[i] = __ldg(tw + i);
    for (size_t p0 = (size_t)blockIdx.x * ax.pt; p0 < ax.npencils; p0 += (size_t)gridDim.x * ax.pt) {
        const int npen = (int)(ax.npencils - p0 < (size_t)ax.pt ? ax.npencils - p0 : (size_t)ax.pt);
        __syncthreads();                                   // the previous tile's stores have read their buffer
        gfft_tile_setup(ax, p0, npen, sbase, sinfo, (MODE != -1 && MODE != 1 && MODE != 2) ? kin.nz : 0, 0);
        __syncthreads();
        gfft_load(a, in, ax, sbase, npen);
        __syncthreads();
        cd* res = a;
        cd* oth = b;
        if (MODE == -1) {
            res = gfft_run<DIR>(a, b, stw, ax, npen);
        } else {
            if (MODE != 2) {
                res = gfft_run<-1>(a, b, stw, ax, npen);
                oth = res == a ? b : a;
            }
            if (MODE != 1) {
                // diagonal factor: the pencil is (state, ky, kz), the element index is kx -- all in natural order
                for (int i = threadIdx.x; i < ax.n * ax.pt; i += GF_THREADS) {
                    const int q = i & (ax.pt - 1), e = i >> ax.pt_log2;
                    if (q >= npen) continue;
                    double f = kin.scale;
                    if (MODE != 2) {
                        const int4 info = sinfo[q];
                        const int st = info.x, ky = info.y, kz = info.z;
                        const double gx2 = __ldg(kin.g2x + e), gy2 = __ldg(kin.g2y_w + ky), gz2 = __ldg(kin.g2z_w + kz);
                        const double ts = MODE == 4 ? __ldg(kin.tstate + st) : 1.0;
                        f = MODE == 3 ? poisson_factor(gx2, gy2, gz2, kin.scale)
                                      : (MODE == 4 ? teter_factor(gx2, gy2, gz2, ts, kin.scale)
                                                   : kin_factor(gx2, gy2, gz2, kin.ecut, kin.scale));
                    }
                    res[e * ld + q] = cscale(res[e * ld + q], f);
                }
                __syncthreads();
                res = gfft_run<+1>(res, oth, stw, ax, npen);
            }
        }
        // store, same thread mapping as the load
        if (ax.stride == 1) {
            for (int i = threadIdx.x; i < ax.n * npen; i += GF_THREADS) {
                const int q = gfft_div(i, ax.magic_n), e = i - q * ax.n;
                sts_cd(out + sbase[q] + e, res[e * ld + q]);
            }
        } else {
            for (int i = threadIdx.x; i < ax.n * ax.pt; i += GF_THREADS) {
                const int q = i & (ax.pt - 1), e = i >> ax.pt_log2;
                if (q < npen) sts_cd(out + sbase[q] + (size_t)e * ax.stride, res[e * ld + q]);
            }
        }
    }
    (void)nx;
}

// inverse transform along z (contiguous pencils = rows of the block) with the fused epilogue of tile_inv:
//     out = alpha * (T phi + V phi) + y        (the back-projection runs as nl_scatter afterwards)
// npts = points of one state (the index into V is the block index modulo npts).
__global__ void __launch_bounds__(GF_THREADS)
gfft_zinv_epilogue_kernel(const cd* __restrict__ in, cd* __restrict__ out, const GAxis ax, const cd* __restrict__ tw,
                          const Epilogue ep, size_t npts)
{
    extern __shared__ __align__(16) unsigned char gsm[];
    cd* a = reinterpret_cast<cd*>(gsm);
    const int ld = ax.pt + 1;
    cd* b = a + (size_t)ax.n * ld;
    cd* stw = b + (size_t)ax.n * ld;
    size_t* sbase = reinterpret_cast<size_t*>(stw + ax.n);
    int4* sinfo = reinterpret_cast<int4*>(sbase + GF_MAXPT);
    for (int i = threadIdx.x; i < ax.n; i += GF_THREADS) stw[i] = __ldg(tw + i);
    for (size_t p0 = (size_t)blockIdx.x * ax.pt; p0 < ax.npencils; p0 += (size_t)gridDim.x * ax.pt) {
        const int npen = (int)(ax.npencils - p0 < (size_t)ax.pt ? ax.npencils - p0 : (size_t)ax.pt);
        __syncthreads();
        gfft_tile_setup(ax, p0, npen, sbase, sinfo, 0, npts);
        __syncthreads();
        gfft_load(a, in, ax, sbase, npen);
        __syncthreads();
        const cd* res = gfft_run<+1>(a, b, stw, ax, npen);
        for (int i = threadIdx.x; i < ax.n * npen; i += GF_THREADS) {
            const int q = gfft_div(i, ax.magic_n), e = i - q * ax.n;
            const size_t gi = sbase[q] + e;                              // rows are contiguous: index in the block
            cd x = res[e * ld + q];
            if (ep.v != nullptr) {
                const double vv = __ldg(ep.v + sinfo[q].w + e);          // a row lies inside one state: (gi mod npts)
                const cd ph = lds_cd(ep.phi + gi);
                x.x = fma(vv, ph.x, x.x);
                x.y = fma(vv, ph.y, x.y);
            }
            cd r = cmul(ep.alpha, x);
            if (ep.yv != nullptr) r = cadd(r, lds_cd(ep.yv + gi));
            sts_cd(out + gi, r);
        }
    }
}

}  // namespace tdh
