// xpencil_kernel.cuh -- the x-direction kernel of one Hamiltonian application.
//
// For each (state, y, z) pencil: forward FFT along x, kinetic factor 1/2|G+k|^2 with cutoff mask and the 1/N_p of
// the inverse transform, inverse FFT along x  (rows a1, a2, a3 of the scope table; Eq. 2 first term).
// A CTA owns 32 pencils ("lines") of one state: 32 x 16 B = 512 contiguous bytes per x (S = 1), or 16 lines of
// spectrum row k and the same 16 lines of row k + NY/2 (S = 2, two 256-byte pieces).  The length-NX transform runs in
// two register stages with one shared-memory exchange each way; lanes are lines, so every access is conflict free.
//
// S = 2 (see tile_kernels.cuh): the tile kernels leave/expect half-length y transforms E_r[k] / F_r[k], r = 0, 1.
// The missing radix-2 step of the y transform commutes with the x transform, and both halves of a line pair sit in
// lanes l and l ^ 16 of one warp.  With A_h = FFT_x(E_h), w = e^{-2 pi i k / NY} and f_h the kinetic factor of
// ky = k + h NY/2:   X_0 = A_0 + w A_1,  X_1 = A_0 - w A_1,   F_0 = f_0 X_0 + f_1 X_1,  F_1 = conj(w) (f_0 X_0 - f_1 X_1)
//   =>  F_h = (f_0 + f_1) A_h + (f_0 - f_1) w_h A_(1-h),   w_0 = w, w_1 = conj(w):  one register exchange per value.
// MODE 0: forward x, kinetic, inverse x.   MODE 1: forward x only (natural spectrum out).
// MODE 2: inverse x only, times `scale` (natural spectrum in).
#pragma once
#include "fft_codelets.cuh"

namespace tdh {

constexpr int XP_LPC = 32;

struct Kinetic {
    const double* g2x;   // (G_x + k_x)^2 per x index, and so on: exactly the doubles the oracle squares
    const double* g2y;
    const double* g2z;
    double ecut;         // <= 0: no mask
    double scale;        // 1 / N_p (MODE 0 and 2); unused in MODE 1
    int nz;
    int nys;             // NY / S
};

__device__ __forceinline__ cd shfl16(cd v) {
    return make_double2(__shfl_xor_sync(0xffffffffu, v.x, 16), __shfl_xor_sync(0xffffffffu, v.y, 16));
}

template <int NX> struct XCfg {
    static constexpr int R1 = Fact<NX>::R1, R2 = Fact<NX>::R2;
    static constexpr int T = XP_LPC * R1;
    static constexpr int by_regs = 65536 / (T * 80);
    static constexpr int MINB = by_regs < 1 ? 1 : (by_regs > 8 ? 8 : by_regs);
};

// grid: (lines_per_state / 32, nst).  in == out is allowed (a CTA reads all its lines before it writes them).
template <int NX, int S, int MODE>
__global__ void __launch_bounds__(XCfg<NX>::T, XCfg<NX>::MINB)
xpencil_kernel(const cd* __restrict__ in, cd* __restrict__ out, int nynz, const cd* __restrict__ tw_x,
               const cd* __restrict__ tw_y, const Kinetic kin)
{
    constexpr int R1 = XCfg<NX>::R1, R2 = XCfg<NX>::R2, L = XP_LPC;
    __shared__ cd sm[NX * L];
    const int tid = threadIdx.x;
    const int l = tid % L, hi = tid / L;               // hi < R1
    int yz, half = 0, base = 0;
    if (S == 1) {
        yz = blockIdx.x * L + l;
    } else {
        half = l >> 4;
        base = blockIdx.x * (L / 2) + (l & 15);        // (k, kz) inside one spectrum half
        yz = half * kin.nys * kin.nz + base;
    }
    const size_t col = (size_t)blockIdx.y * NX * nynz + yz;   // element x at col + x * nynz
    cd xr[R2];                                                 // stage-B registers: X[hi + R1*k2]

    if (MODE != 2) {
        // ---- forward stage A (threads with hi < R2): radix R1 over x = j1*R2 + j2, j2 = hi
        if (hi < R2) {
            const int j2 = hi;
            cd x[R1];
#pragma unroll
            for (int j1 = 0; j1 < R1; ++j1) x[j1] = __ldcs(in + col + (size_t)(j1 * R2 + j2) * nynz);
            Dft<R1, -1>::run(x);
            sm[j2 * L + l] = x[0];
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) sm[(k1 * R2 + j2) * L + l] = cmulc(x[k1], __ldg(tw_x + k1 * j2));
        }
        __syncthreads();
        // ---- forward stage B: thread (l, k1 = hi) -> X[k1 + R1*k2]
#pragma unroll
        for (int j2 = 0; j2 < R2; ++j2) xr[j2] = sm[(hi * R2 + j2) * L + l];
        Dft<R2, -1>::run(xr);
    } else {
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) xr[k2] = __ldcs(in + col + (size_t)(hi + R1 * k2) * nynz);
    }

    // ---- kinetic factor t = 0.5*((gx^2 + gy^2) + gz^2) in the oracle's operation order, no contraction;
    //      with S = 2 also the radix-2 step of the y transform (header comment)
    if (S == 1) {
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
        } else if (MODE == 2) {
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) xr[k2] = cscale(xr[k2], kin.scale);
        }
    } else {
        const int k = base / kin.nz, kz = base % kin.nz;
        const cd w = __ldg(tw_y + k);                    // e^{+2 pi i k / NY} = conj(w of the header comment)
        if (MODE == 0) {
            const double gy2a = __ldg(kin.g2y + k), gy2b = __ldg(kin.g2y + k + kin.nys), gz2 = __ldg(kin.g2z + kz);
            const cd wh = half ? w : make_double2(w.x, -w.y);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) {
                const double gx2 = __ldg(kin.g2x + hi + R1 * k2);
                const double ta = __dmul_rn(0.5, __dadd_rn(__dadd_rn(gx2, gy2a), gz2));
                const double tb = __dmul_rn(0.5, __dadd_rn(__dadd_rn(gx2, gy2b), gz2));
                const double fa = (kin.ecut > 0.0 && !(ta <= kin.ecut)) ? 0.0 : ta * kin.scale;
                const double fb = (kin.ecut > 0.0 && !(tb <= kin.ecut)) ? 0.0 : tb * kin.scale;
                const cd other = shfl16(xr[k2]);
                const cd wo = cmul(wh, other);
                const double fs = fa + fb, fd = fa - fb;
                xr[k2] = make_double2(fma(fs, xr[k2].x, fd * wo.x), fma(fs, xr[k2].y, fd * wo.y));
            }
        } else if (MODE == 1) {
            // X_0 = A_0 + w A_1 (lane of half 0), X_1 = A_0 - w A_1 (lane of half 1), w = conj(tw_y[k])
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) {
                const cd mine = half ? cmulc(xr[k2], w) : xr[k2];      // half 1 sends w A_1, half 0 sends A_0
                const cd other = shfl16(mine);
                xr[k2] = half ? csub(other, mine) : cadd(mine, other);
            }
        } else {
            // F_0 = X_0 + X_1,  F_1 = conj(w) (X_0 - X_1), conj(w) = tw_y[k]; then the 1/N_p
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) {
                const cd other = shfl16(xr[k2]);
                const cd v = half ? cmul(w, csub(other, xr[k2])) : cadd(xr[k2], other);
                xr[k2] = cscale(v, kin.scale);
            }
        }
    }

    if (MODE == 1) {
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) __stcs(out + col + (size_t)(hi + R1 * k2) * nynz, xr[k2]);
        return;
    }

    // ---- inverse with the mirrored factorisation (first radix R2 on stride R1): the registers of stage B are
    //      exactly the inputs of its first stage, n = k2*R1 + hi
    Dft<R2, +1>::run(xr);
    if (MODE == 0) __syncthreads();   // every stage-B read of sm is done before sm is overwritten
    sm[hi * L + l] = xr[0];           // cell (k1' * R1 + j2'), j2' = hi
#pragma unroll
    for (int k1 = 1; k1 < R2; ++k1) sm[(k1 * R1 + hi) * L + l] = cmul(xr[k1], __ldg(tw_x + k1 * hi));
    __syncthreads();
    if (hi < R2) {
        const int k1 = hi;
        cd x[R1];
#pragma unroll
        for (int j2 = 0; j2 < R1; ++j2) x[j2] = sm[(k1 * R1 + j2) * L + l];
        Dft<R1, +1>::run(x);
#pragma unroll
        for (int k2 = 0; k2 < R1; ++k2) __stcs(out + col + (size_t)(k1 + R2 * k2) * nynz, x[k2]);
    }
}

}  // namespace tdh
