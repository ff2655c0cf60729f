// fft_kernels.cuh -- the three FFT-carrying kernels of one Hamiltonian application.
//
//   plane_fwd   : for each (state, x) plane: forward FFT along z then y            (row a1 of the scope table)
//   xpencil     : for each (state, y, z) pencil: forward x, kinetic scale+mask, inverse x   (rows a1, a2, a3)
//   plane_inv   : for each (state, x) plane: inverse FFT along y then z, then the fused epilogue
//                 out = alpha * (T psi + V psi + V_nl psi) + y                      (rows a3, a4, a5-scatter, a6, a7-axpy)
//
// Layout in global memory is always [state][x][y][z], z fastest.  A 1-D transform of length N = R1*R2 runs in two
// register stages (radix R1 on stride R2, twiddle, radix R2) with one shared-memory exchange in between.  The
// exchanges are arranged so that every stage overwrites exactly the shared-memory cells it has read ("in place per
// thread"), which removes half of the barriers; the price is a permuted order inside shared memory that the next
// stage's index arithmetic undoes.  Rows are padded to R1*(R2|1) cells so that both the contiguous and the strided
// 16-byte accesses are bank-conflict free (stride odd in units of 16 B).
#pragma once
#include "fft_codelets.cuh"

namespace tdh {

__device__ __forceinline__ cd ldg_cd(const cd* p) { return __ldg(p); }

// ------------------------------------------------------------------------------------------------------------
// plane kernels
// ------------------------------------------------------------------------------------------------------------
template <int NY, int NZ> struct PlaneCfg {
    static constexpr int R1Z = FactP<NZ>::R1, R2Z = FactP<NZ>::R2, QZ = R2Z | 1, PZ = R1Z * QZ;
    static constexpr int R1Y = FactP<NY>::R1, R2Y = FactP<NY>::R2;
    static constexpr int PPC = (NY * NZ >= 1024) ? 1 : 1024 / (NY * NZ);        // planes per CTA
    static constexpr int T = (R2Z % 3 == 0) ? 384 : ((NY * NZ >= 64 * 64) ? 512 : 256);
    static constexpr int ROWS = PPC * NY;
    static constexpr size_t SMEM = (size_t)ROWS * PZ * sizeof(cd);
    static_assert(T % R2Z == 0, "z-stage twiddles are kept in registers: T must be a multiple of R2Z");
};

// forward: in -> out (in == out allowed: a CTA reads its planes completely before it writes them)
template <int NY, int NZ>
__global__ void __launch_bounds__(PlaneCfg<NY, NZ>::T)
plane_fwd_kernel(const cd* __restrict__ in, cd* __restrict__ out, const cd* __restrict__ tw_y,
                 const cd* __restrict__ tw_z)
{
    using C = PlaneCfg<NY, NZ>;
    constexpr int R1Z = C::R1Z, R2Z = C::R2Z, QZ = C::QZ, PZ = C::PZ, R1Y = C::R1Y, R2Y = C::R2Y, T = C::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    const int tid = threadIdx.x;
    const size_t base = (size_t)blockIdx.x * C::ROWS * NZ;

    // ---- z stage A: global -> registers, radix R1Z on stride R2Z, twiddle, -> sm[row][k1*QZ + j2]
    {
        const int j2 = tid % R2Z;
        cd tw[R1Z];
#pragma unroll
        for (int k1 = 1; k1 < R1Z; ++k1) tw[k1] = ldg_cd(tw_z + k1 * j2);
        for (int row = tid / R2Z; row < C::ROWS; row += T / R2Z) {
            const cd* src = in + base + (size_t)row * NZ + j2;
            cd x[R1Z];
#pragma unroll
            for (int j1 = 0; j1 < R1Z; ++j1) x[j1] = src[j1 * R2Z];
            Dft<R1Z, -1>::run(x);
            cd* dst = sm + row * PZ + j2;
            dst[0] = x[0];
#pragma unroll
            for (int k1 = 1; k1 < R1Z; ++k1) dst[k1 * QZ] = cmulc(x[k1], tw[k1]);
        }
    }
    __syncthreads();
    // ---- z stage B, in place: X[k1 + R1Z*k2] is left at sm[row][k1*QZ + k2]
    for (int item = tid; item < C::ROWS * R1Z; item += T) {
        const int k1 = item % R1Z, row = item / R1Z;
        cd* p = sm + row * PZ + k1 * QZ;
        cd t[R2Z];
#pragma unroll
        for (int j2 = 0; j2 < R2Z; ++j2) t[j2] = p[j2];
        Dft<R2Z, -1>::run(t);
#pragma unroll
        for (int k2 = 0; k2 < R2Z; ++k2) p[k2] = t[k2];
    }
    __syncthreads();
    // ---- y stage A, in place: rows j1*R2Y + j2 of column kz -> rows k1*R2Y + j2
    for (int item = tid; item < C::PPC * NZ * R2Y; item += T) {
        const int kz = item % NZ, r = item / NZ, j2 = r % R2Y, lp = r / R2Y;
        const int col = (kz % R1Z) * QZ + kz / R1Z;
        cd* p = sm + (lp * NY + j2) * PZ + col;
        cd x[R1Y];
#pragma unroll
        for (int j1 = 0; j1 < R1Y; ++j1) x[j1] = p[j1 * R2Y * PZ];
        Dft<R1Y, -1>::run(x);
        p[0] = x[0];
#pragma unroll
        for (int k1 = 1; k1 < R1Y; ++k1) p[k1 * R2Y * PZ] = cmulc(x[k1], ldg_cd(tw_y + k1 * j2));
    }
    __syncthreads();
    // ---- y stage B -> global, natural order out[ky][kz]
    for (int item = tid; item < C::PPC * NZ * R1Y; item += T) {
        const int kz = item % NZ, r = item / NZ, k1 = r % R1Y, lp = r / R1Y;
        const int col = (kz % R1Z) * QZ + kz / R1Z;
        const cd* p = sm + (lp * NY + k1 * R2Y) * PZ + col;
        cd t[R2Y];
#pragma unroll
        for (int j2 = 0; j2 < R2Y; ++j2) t[j2] = p[j2 * PZ];
        Dft<R2Y, -1>::run(t);
        cd* dst = out + base + (size_t)lp * NY * NZ + kz;
#pragma unroll
        for (int k2 = 0; k2 < R2Y; ++k2) dst[(k1 + R1Y * k2) * NZ] = t[k2];
    }
}

// Arguments of the fused epilogue of plane_inv.
struct Epilogue {
    const cd* phi;          // input block of this application (for V*phi); NULL: no local term
    const double* v;        // V(r), n0*n1*n2; NULL: no local term
    const cd* yv;           // optional addend y (same block layout as out); NULL: none
    cd alpha;               // out = alpha * (T + V + Vnl) phi + y
    int nx;                 // planes per state
    // non-local scatter (point-centric, atomic free); nl_start == NULL: no projectors
    const int* nl_start;    // [np] index of the first entry of a grid point, -1: not covered
    const int4* nl_ent;     // per entry: {beta offset, P stride between channels, first channel, nchan | last << 16}
    const cd* nl_phase;     // per entry e^{+ik.d}; NULL at Gamma
    const double* nl_beta;  // projector values
    const cd* dpi;          // [state][nchan_tot] D * dV * <beta|phi>
    int nchan_tot;
};

template <int NY, int NZ>
__global__ void __launch_bounds__(PlaneCfg<NY, NZ>::T)
plane_inv_kernel(const cd* __restrict__ in, cd* __restrict__ out, const cd* __restrict__ tw_y,
                 const cd* __restrict__ tw_z, const Epilogue ep)
{
    using C = PlaneCfg<NY, NZ>;
    constexpr int R1Z = C::R1Z, R2Z = C::R2Z, QZ = C::QZ, PZ = C::PZ, R1Y = C::R1Y, R2Y = C::R2Y, T = C::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    const int tid = threadIdx.x;
    const size_t base = (size_t)blockIdx.x * C::ROWS * NZ;

    // ---- y stage A: global -> registers, radix R1Y, twiddle, -> sm[row k1*R2Y + j2][col(kz)],
    //      col(z) = (z / R2Z)*QZ + z % R2Z is the padded position the z stages want
    for (int item = tid; item < C::PPC * NZ * R2Y; item += T) {
        const int kz = item % NZ, r = item / NZ, j2 = r % R2Y, lp = r / R2Y;
        const cd* src = in + base + (size_t)lp * NY * NZ + (size_t)j2 * NZ + kz;
        cd x[R1Y];
#pragma unroll
        for (int j1 = 0; j1 < R1Y; ++j1) x[j1] = src[(size_t)j1 * R2Y * NZ];
        Dft<R1Y, +1>::run(x);
        const int col = (kz / R2Z) * QZ + kz % R2Z;
        cd* p = sm + (lp * NY + j2) * PZ + col;
        p[0] = x[0];
#pragma unroll
        for (int k1 = 1; k1 < R1Y; ++k1) p[k1 * R2Y * PZ] = cmul(x[k1], ldg_cd(tw_y + k1 * j2));
    }
    __syncthreads();
    // ---- y stage B, in place: row rho = k1*R2Y + k2 now holds y = k1 + R1Y*k2
    for (int item = tid; item < C::PPC * NZ * R1Y; item += T) {
        const int kz = item % NZ, r = item / NZ, k1 = r % R1Y, lp = r / R1Y;
        const int col = (kz / R2Z) * QZ + kz % R2Z;
        cd* p = sm + (lp * NY + k1 * R2Y) * PZ + col;
        cd t[R2Y];
#pragma unroll
        for (int j2 = 0; j2 < R2Y; ++j2) t[j2] = p[j2 * PZ];
        Dft<R2Y, +1>::run(t);
#pragma unroll
        for (int k2 = 0; k2 < R2Y; ++k2) p[k2 * PZ] = t[k2];
    }
    __syncthreads();
    // ---- z stage A, in place: cells j1*QZ + j2 -> k1*QZ + j2
    {
        const int j2 = tid % R2Z;
        cd tw[R1Z];
#pragma unroll
        for (int k1 = 1; k1 < R1Z; ++k1) tw[k1] = ldg_cd(tw_z + k1 * j2);
        for (int row = tid / R2Z; row < C::ROWS; row += T / R2Z) {
            cd* p = sm + row * PZ + j2;
            cd x[R1Z];
#pragma unroll
            for (int j1 = 0; j1 < R1Z; ++j1) x[j1] = p[j1 * QZ];
            Dft<R1Z, +1>::run(x);
            p[0] = x[0];
#pragma unroll
            for (int k1 = 1; k1 < R1Z; ++k1) p[k1 * QZ] = cmul(x[k1], tw[k1]);
        }
    }
    __syncthreads();
    // ---- z stage B + epilogue -> global
    const int plane0 = blockIdx.x * C::PPC;
    for (int item = tid; item < C::ROWS * R1Z; item += T) {
        const int k1 = item % R1Z, row = item / R1Z;
        const cd* p = sm + row * PZ + k1 * QZ;
        cd t[R2Z];
#pragma unroll
        for (int j2 = 0; j2 < R2Z; ++j2) t[j2] = p[j2];
        Dft<R2Z, +1>::run(t);
        const int lp = row / NY, rho = row % NY;
        const int y = rho / R2Y + R1Y * (rho % R2Y);
        const int plane = plane0 + lp;
        const int st = plane / ep.nx, x = plane % ep.nx;
        const size_t g0 = (size_t)plane * NY * NZ + (size_t)y * NZ + k1;          // index in the block
        const size_t q0 = ((size_t)x * NY + y) * NZ + k1;                           // index in the state
#pragma unroll
        for (int k2 = 0; k2 < R2Z; ++k2) {
            const size_t g = g0 + R1Z * k2, q = q0 + R1Z * k2;
            cd acc = t[k2];
            if (ep.v != nullptr) {
                const cd ph = ldg_cd(ep.phi + g);
                const double vv = __ldg(ep.v + q);
                acc.x = fma(vv, ph.x, acc.x);
                acc.y = fma(vv, ph.y, acc.y);
            }
            if (ep.nl_start != nullptr) {
                int e = __ldg(ep.nl_start + q);
                if (e >= 0) {
                    const cd* dp = ep.dpi + (size_t)st * ep.nchan_tot;
                    int last;
                    do {
                        const int4 en = __ldg(ep.nl_ent + e);
                        const int nch = en.w & 0xffff;
                        last = en.w >> 16;
                        cd s = make_double2(0.0, 0.0);
                        for (int c = 0; c < nch; ++c) {
                            const double b = __ldg(ep.nl_beta + en.x + (size_t)c * en.y);
                            const cd d = ldg_cd(dp + en.z + c);
                            s.x = fma(b, d.x, s.x);
                            s.y = fma(b, d.y, s.y);
                        }
                        if (ep.nl_phase != nullptr) s = cmulc(s, ldg_cd(ep.nl_phase + e));
                        acc = cadd(acc, s);
                        ++e;
                    } while (!last);
                }
            }
            cd o = cmul(ep.alpha, acc);
            if (ep.yv != nullptr) o = cadd(o, ldg_cd(ep.yv + g));
            out[g] = o;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// x-pencil kernel.  A CTA owns LPC = 32 consecutive (y,z) lines of one state: 512 contiguous bytes per x.
// MODE 0: forward x, kinetic scale (+ mask, + 1/N_p), inverse x.   MODE 1: forward x only.
// MODE 2: inverse x only, times `scale`.
// ------------------------------------------------------------------------------------------------------------
constexpr int XP_LPC = 32;

struct Kinetic {
    const double* g2x;   // (G_x + k_x)^2 per x index, and so on: exactly the doubles the oracle squares
    const double* g2y;
    const double* g2z;
    double ecut;         // <= 0: no mask
    double scale;        // 1 / N_p (MODE 0 and 2); unused in MODE 1
    int nz;
};

template <int NX, int MODE>
__global__ void __launch_bounds__(XP_LPC * Fact<NX>::R1)
xpencil_kernel(cd* __restrict__ w, int nynz, const cd* __restrict__ tw_x, const Kinetic kin)
{
    constexpr int R1 = Fact<NX>::R1, R2 = Fact<NX>::R2, L = XP_LPC;
    __shared__ cd sm[NX * L];
    const int tid = threadIdx.x;
    const int l = tid % L, hi = tid / L;               // hi < R1
    const int yz = blockIdx.x * L + l;
    cd* col = w + (size_t)blockIdx.y * NX * nynz + yz;  // element x at col[x * nynz]
    cd xr[R2];                                          // stage-B registers: X[hi + R1*k2]

    if (MODE != 2) {
        // ---- forward stage A (threads with hi < R2): radix R1 over x = j1*R2 + j2, j2 = hi
        if (hi < R2) {
            const int j2 = hi;
            cd x[R1];
#pragma unroll
            for (int j1 = 0; j1 < R1; ++j1) x[j1] = col[(size_t)(j1 * R2 + j2) * nynz];
            Dft<R1, -1>::run(x);
            sm[(j2)*L + l] = x[0];
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) sm[(k1 * R2 + j2) * L + l] = cmulc(x[k1], ldg_cd(tw_x + k1 * j2));
        }
        __syncthreads();
        // ---- forward stage B: thread (l, k1 = hi) -> X[k1 + R1*k2]
#pragma unroll
        for (int j2 = 0; j2 < R2; ++j2) xr[j2] = sm[(hi * R2 + j2) * L + l];
        Dft<R2, -1>::run(xr);
    } else {
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) xr[k2] = col[(size_t)(hi + R1 * k2) * nynz];
    }

    if (MODE == 1) {
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) col[(size_t)(hi + R1 * k2) * nynz] = xr[k2];
        return;
    }

    // ---- kinetic factor: t = 0.5*((gx^2 + gy^2) + gz^2) in the oracle's operation order, no contraction
    if (MODE == 0) {
        const int ky = yz / kin.nz, kz = yz % kin.nz;
        const double gy2 = __ldg(kin.g2y + ky), gz2 = __ldg(kin.g2z + kz);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) {
            const double gx2 = __ldg(kin.g2x + hi + R1 * k2);
            const double t = __dmul_rn(0.5, __dadd_rn(__dadd_rn(gx2, gy2), gz2));
            const double f = (kin.ecut > 0.0 && !(t <= kin.ecut)) ? 0.0 : t * kin.scale;
            xr[k2] = cscale(xr[k2], f);
        }
    } else {
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) xr[k2] = cscale(xr[k2], kin.scale);
    }

    // ---- inverse with the mirrored factorisation (first radix R2 on stride R1): the registers of stage B are
    //      exactly the inputs of its first stage, n = k2*R1 + hi
    Dft<R2, +1>::run(xr);
    if (MODE == 0) __syncthreads();   // every stage-B read of sm is done before sm is overwritten
    sm[hi * L + l] = xr[0];           // cell (k1' * R1 + j2'), j2' = hi
#pragma unroll
    for (int k1 = 1; k1 < R2; ++k1) sm[(k1 * R1 + hi) * L + l] = cmul(xr[k1], ldg_cd(tw_x + k1 * hi));
    __syncthreads();
    if (hi < R2) {
        const int k1 = hi;
        cd x[R1];
#pragma unroll
        for (int j2 = 0; j2 < R1; ++j2) x[j2] = sm[(k1 * R1 + j2) * L + l];
        Dft<R1, +1>::run(x);
#pragma unroll
        for (int k2 = 0; k2 < R1; ++k2) col[(size_t)(k1 + R2 * k2) * nynz] = x[k2];
    }
}

}  // namespace tdh
