// xpencil_kernel.cuh -- the x-direction kernel of one Hamiltonian application (persistent, TMA-fed).
//
// For each (state, y, z) pencil: forward FFT along x, kinetic factor 1/2|G+k|^2 with cutoff mask and the 1/N_p of
// the inverse transform, inverse FFT along x  (rows a1, a2, a3 of the scope table; Eq. 2 first term).
//
// WORK LAYOUT.  The tile kernels (tile_kernels.cuh) leave the (y,z) spectrum of every (state, x) plane in the digit-
// permuted order their in-place transforms produce: plane row Y = S*rho + r, column z' = 8*k1 + k2 holds
//     kz = k1 + (NZ/8)*k2,   and   rho = k1y*R2Y + k2y  <->  k = k1y + R1Y*k2y   (index inside the spectrum part r).
// This kernel never needs the natural order: it only needs the kinetic factor of each line, which the host tabulates
// in work-layout order (g2y_w[Y], g2z_w[z'], twy_w[rho]).
//
// TILE.  A tile is 32 pencils ("lines") of one state: 16 consecutive z' of plane row Y = 2*rho2 and the same 16 z' of
// row Y + 1, for all NX planes -- one 4-D TMA box {16 cells, 1, 2 rows, NX}, landing in shared memory as [x][32 lines]
// (512 bytes per x).  Lanes are lines, so every shared-memory access is conflict free.  CTAs are persistent: each
// walks tiles blockIdx.x, blockIdx.x + gridDim.x, ... through a ring of NB buffers that one elected thread keeps
// filled with cp.async.bulk.tensor, so the loads of the next tiles are in flight while this one is transformed.
//
// THREADS.  NX = R1*R2 (R1 >= R2).  A CTA has TPL = 4 threads per line (128 threads): the R2 radix-R1 transforms of a
// line (first forward stage, last inverse stage) take ceil(R2/4) rounds, the R1 radix-R2 transforms in between
// ceil(R1/4) rounds -- for NX = 96 (12 x 8) that is 2, 3, 2 rounds with every thread busy in each.  The kernel is compiled
// for four resident CTAs per SM (<= 128 registers per thread): the barrier-separated stages of one CTA alternate between
// TMA wait, shared-memory, FP64 and store phases, and the other three fill the gaps (measured on Large: 8 threads per
// line and two CTAs 0.79 ms per 128 states, this layout 0.69 ms).  Twiddles and (G_x+k_x)^2 sit in shared memory
// behind the ring.
//
// S = 2 (see tile_kernels.cuh): the tile kernels leave/expect half-length y transforms E_r[k] / F_r[k], r = 0, 1, at
// rows Y = 2*rho + r -- lanes l and l ^ 16 of a warp.  The missing radix-2 step of the y transform commutes with the x
// transform.  With A_h = FFT_x(E_h), w = e^{-2 pi i k / NY} and f_h the kinetic factor of ky = k + h NY/2:
//   X_0 = A_0 + w A_1,  X_1 = A_0 - w A_1,   F_0 = f_0 X_0 + f_1 X_1,  F_1 = conj(w) (f_0 X_0 - f_1 X_1)
//   =>  F_h = (f_0 + f_1) A_h + (f_0 - f_1) w_h A_(1-h),   w_0 = w, w_1 = conj(w):  one register exchange per value.
// MODE 0: forward x, kinetic, inverse x.   MODE 1: forward x only (spectrum out, work layout).
// MODE 3: as MODE 0 with the Poisson factor 4 pi / |G|^2 (G = 0 dropped) in place of the kinetic one (tdh_hartree;
//         the tables in `Kinetic` are then those of the pure reciprocal vectors, without the Bloch vector).
// MODE 4: as MODE 0 with the Teter preconditioner K(t / T_s), t = 1/2|G+k|^2, T_s = kin.tstate[state] (tdh_sd_step).
// MODE 2: inverse x only, times `scale` (spectrum in, work layout).
#pragma once
#include "fft_codelets.cuh"
#include "tma.cuh"

namespace tdh {

constexpr int XP_LPC = 32;

struct Kinetic {
    const double* g2x;     // (G_x + k_x)^2 per x index: exactly the doubles the oracle squares
    const double* g2y_w;   // [NY] (G_y + k_y)^2 of the ky that plane row Y stands for (work-layout order)
    const double* g2z_w;   // [NZ] (G_z + k_z)^2 of the kz that column z' stands for
    const cd* twy_w;       // [NY/2] e^{+2 pi i k / NY} of row pair rho (S = 2 only)
    const double* tstate;  // MODE 4: kinetic energy T_s per state of this launch
    double ecut;           // <= 0: no mask
    double scale;          // 1 / N_p (MODE 0 and 2); unused in MODE 1
    int nz;
    int ny;
};

// Slab decomposition (tile_kernels.cuh, SlabDst): the pencils of this rank's Fourier-space slab (rows y0 .. y0 + ny_local - 1
// of all NX planes; `Kinetic::ny` = ny_local and the y tables start at y0) end their inverse x transform with the value
// of plane x, which belongs to rank p = x / nx_local: it is stored straight into that rank's real-space work buffer
// rs[p] = [state][nx_local][NY][NZ] -- the way back of the all-to-all, fused into the stores (peer pointers over NVLink).
struct SlabSrc {
    cd* rs[8];
    int nx_local;           // planes per state and rank
    int ny_total;           // NY
    int y0;                 // first row of this rank's Fourier-space slab
};

__device__ __forceinline__ cd shfl16(cd v) {
    return make_double2(__shfl_xor_sync(0xffffffffu, v.x, 16), __shfl_xor_sync(0xffffffffu, v.y, 16));
}

template <int NX> struct XCfg {
    static constexpr int R1 = Fact<NX>::R1, R2 = Fact<NX>::R2;
    static constexpr int TPL = 4;                                   // threads per line
    static constexpr int T = XP_LPC * TPL;
    static constexpr int CPS = 512 / T;                             // resident CTAs per SM the kernel is built for
    static constexpr int ROUNDS_A = (R2 + TPL - 1) / TPL;           // rounds of the radix-R1 stages
    static constexpr int ROUNDS_B = (R1 + TPL - 1) / TPL;           // rounds of the radix-R2 stage
    static constexpr int TILE_CELLS = NX * XP_LPC;
    static constexpr size_t TILE_BYTES = (size_t)TILE_CELLS * sizeof(cd);
    static constexpr size_t TABLE_BYTES = (size_t)NX * (sizeof(cd) + sizeof(double));
    // ring depth: what fits in 1/CPS of the SM's 228 KB beside the barriers, the tables and the 1 KB the system
    // reserves per CTA; between 2 and 4 tiles
    static constexpr int fit() { return (int)((233472 / CPS - 2048 - TABLE_BYTES) / TILE_BYTES); }
    static constexpr int NB = fit() < 1 ? 1 : (fit() > 4 ? 4 : fit());
    static constexpr size_t SMEM = 1024 + NB * TILE_BYTES + TABLE_BYTES;
};

// the kinetic factor t = 0.5*((gx^2 + gy^2) + gz^2) in the oracle's operation order (no contraction), masked, times
// the 1/N_p of the inverse transform
__device__ __forceinline__ double kin_factor(double gx2, double gy2, double gz2, double ecut, double scale) {
    const double tk = __dmul_rn(0.5, __dadd_rn(__dadd_rn(gx2, gy2), gz2));
    return (ecut > 0.0 && !(tk <= ecut)) ? 0.0 : tk * scale;
}
// the Poisson factor 4 pi / |G|^2, 0 for G = 0, times 1/N_p; |G|^2 summed in the oracle's order
__device__ __forceinline__ double poisson_factor(double gx2, double gy2, double gz2, double scale) {
    const double g2 = __dadd_rn(__dadd_rn(gx2, gy2), gz2);
    return g2 > 0.0 ? __ddiv_rn(12.566370614359172953850573533118, g2) * scale : 0.0;
}
// the Teter-Payne-Allan preconditioner K(x), x = t / T_s (reading R19), times 1/N_p
__device__ __forceinline__ double teter_factor(double gx2, double gy2, double gz2, double ts, double scale) {
    const double tk = __dmul_rn(0.5, __dadd_rn(__dadd_rn(gx2, gy2), gz2));
    // T_s <= 0 (a constant state at Gamma, up to rounding): the limit x -> infinity, K = 1 at t = 0 and 0 elsewhere (R19)
    if (!(ts > 0.0)) return tk == 0.0 ? scale : 0.0;
    const double x = tk / ts;
    const double num = 27.0 + x * (18.0 + x * (12.0 + x * 8.0));
    const double x2 = x * x;
    return num / (num + 16.0 * x2 * x2) * scale;
}
template <int MODE>
__device__ __forceinline__ double diag_factor(double gx2, double gy2, double gz2, double ecut, double scale, double ts) {
    return MODE == 3 ? poisson_factor(gx2, gy2, gz2, scale)
                     : (MODE == 4 ? teter_factor(gx2, gy2, gz2, ts, scale) : kin_factor(gx2, gy2, gz2, ecut, scale));
}

// grid: persistent CTAs; ntiles = nst * (NY/2) * (NZ/16).  in (through `map`) and out may be the same buffer: a tile
// is read completely before any of its lines is written.
template <int NX, int S, int MODE, bool SLAB = false>
__global__ void __launch_bounds__(XCfg<NX>::T, XCfg<NX>::CPS)
xpencil_kernel(const __grid_constant__ CUtensorMap map, cd* __restrict__ out, int ntiles,
               const cd* __restrict__ tw_x, const Kinetic kin, const SlabSrc slab)
{
    static_assert(!SLAB || MODE == 0 || MODE == 2, "the slab stores exist for the modes that end in real space");
    using C = XCfg<NX>;
    constexpr int R1 = C::R1, R2 = C::R2, L = XP_LPC, NB = C::NB, TPL = C::TPL, RA = C::ROUNDS_A, RB = C::ROUNDS_B;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);            // NB barriers in the first 1024 bytes
    cd* ring = reinterpret_cast<cd*>(smem_raw + 1024);
    cd* stw = ring + (size_t)NB * C::TILE_CELLS;                        // e^{+2 pi i m / NX}
    double* sg2x = reinterpret_cast<double*>(stw + NX);                 // (G_x + k_x)^2
    const int tid = threadIdx.x;
    const int l = tid % L, hi = tid / L;               // hi < TPL, warp-uniform
    const int half = l >> 4;
    const int zc = kin.nz >> 4;                         // 16-column chunks per plane row
    const int tiles_per_state = (kin.ny >> 1) * zc;
    const size_t nynz = (size_t)kin.ny * kin.nz;

    uint64_t pol = 0;
    if (tid == 0) {
        tma_prefetch_desc(&map);
        pol = policy_evict_first();
        for (int b = 0; b < NB; ++b) mbar_init(full + b, 1);
        mbar_fence_init();
    }
    for (int i = tid; i < NX; i += C::T) {
        stw[i] = __ldg(tw_x + i);
        sg2x[i] = (MODE == 0 || MODE >= 3) ? __ldg(kin.g2x + i) : 0.0;
    }
    __syncthreads();
    auto issue = [&](int t, int b) {                    // thread 0 only
        const int st = t / tiles_per_state, rem = t % tiles_per_state;
        const int rho2 = rem / zc, ch = rem % zc;
        mbar_arrive_expect_tx(full + b, (uint32_t)C::TILE_BYTES);
        tma_load_4d(ring + (size_t)b * C::TILE_CELLS, &map, full + b, 0, ch, 2 * rho2, st * NX, pol);
    };
    if (tid == 0)
        for (int b = 0; b < NB; ++b) {
            const int t = blockIdx.x + b * gridDim.x;
            if (t < ntiles) issue(t, b);
        }

    int it = 0;
    for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++it) {
        const int b = it % NB;
        const uint32_t parity = (uint32_t)(it / NB) & 1u;
        cd* sm = ring + (size_t)b * C::TILE_CELLS;
        const int st = t / tiles_per_state, rem = t % tiles_per_state;
        const int rho2 = rem / zc, ch = rem % zc;
        const int Y = 2 * rho2 + half, zp = ch * 16 + (l & 15);
        cd* gcol = out + (size_t)st * NX * nynz + (size_t)Y * kin.nz + zp;   // element x at gcol + x * nynz
        // address of the value of plane x of this pencil
        auto xdst = [&](int x) -> cd* {
            if (SLAB) {
                const int p = x / slab.nx_local;
                return slab.rs[p] + (((size_t)st * slab.nx_local + (x - p * slab.nx_local)) * slab.ny_total + slab.y0 + Y) * kin.nz + zp;
            }
            return gcol + (size_t)x * nynz;
        };
        // per-line constants of this tile (in flight while the tile arrives)
        double gy2a = 0.0, gy2b = 0.0, gz2 = 0.0;
        cd w = make_double2(1.0, 0.0);
        if (MODE == 0 || MODE >= 3) {
            gz2 = __ldg(kin.g2z_w + zp);
            gy2a = __ldg(kin.g2y_w + (S == 2 ? 2 * rho2 : Y));
            if (S == 2) gy2b = __ldg(kin.g2y_w + 2 * rho2 + 1);
        }
        if (S == 2) w = __ldg(kin.twy_w + rho2);                 // e^{+2 pi i k / NY} = conj(w of the header comment)
        const double ts = MODE == 4 ? __ldg(kin.tstate + st) : 1.0;
        // a ring of one buffer cannot prefetch into shared memory: start the CTA's next tile towards L2 instead
        // (measured: +3 % for the 48 KB tiles of NX = 96, -4 % for the 32 KB tiles of NX = 64, so only the former)
        if (NB == 1 && NX >= 96 && tid == 0 && t + (int)gridDim.x < ntiles) {
            const int tn = t + gridDim.x, stn = tn / tiles_per_state, remn = tn % tiles_per_state;
            tma_prefetch_l2_4d(&map, 0, remn % zc, 2 * (remn / zc), stn * NX);
        }
        mbar_wait(full + b, parity);

        if (MODE != 2) {
            // ---- forward stage A: radix R1 over x = j1*R2 + j2, transforms j2 = hi, hi + TPL, ... < R2, in place
#pragma unroll
            for (int ra = 0; ra < RA; ++ra) {
                const int j2 = hi + ra * TPL;
                if (j2 < R2) {
                    cd x[R1];
#pragma unroll
                    for (int j1 = 0; j1 < R1; ++j1) x[j1] = sm[(j1 * R2 + j2) * L + l];
                    Dft<R1, -1>::run(x);
                    sm[j2 * L + l] = x[0];
#pragma unroll
                    for (int k1 = 1; k1 < R1; ++k1) sm[(k1 * R2 + j2) * L + l] = cmulc(x[k1], stw[k1 * j2]);
                }
            }
            __syncthreads();
        }

        if (MODE == 2) {
            // ---- inverse only: X[k1 + R1*k2] sits in slot k1 + R1*k2; every thread reads all its inputs, then the
            //      intermediate values go to slots k1*R2 + n2 (other threads' inputs: barrier in between)
            cd xr[RB][R2];
#pragma unroll
            for (int rd = 0; rd < RB; ++rd) {
                const int k1 = hi + rd * TPL;
                if (k1 < R1) {
#pragma unroll
                    for (int k2 = 0; k2 < R2; ++k2) xr[rd][k2] = sm[(k1 + R1 * k2) * L + l];
                }
            }
            __syncthreads();
#pragma unroll
            for (int rd = 0; rd < RB; ++rd) {
                const int k1 = hi + rd * TPL;
                if (k1 < R1) {
#pragma unroll
                    for (int k2 = 0; k2 < R2; ++k2) {
                        if (S == 2) {
                            // F_0 = X_0 + X_1,  F_1 = conj(w) (X_0 - X_1), conj(w) = twy_w[rho]; then the 1/N_p
                            const cd other = shfl16(xr[rd][k2]);
                            const cd v = half ? cmul(w, csub(other, xr[rd][k2])) : cadd(xr[rd][k2], other);
                            xr[rd][k2] = cscale(v, kin.scale);
                        } else {
                            xr[rd][k2] = cscale(xr[rd][k2], kin.scale);
                        }
                    }
                    Dft<R2, +1>::run(xr[rd]);
                    sm[(k1 * R2) * L + l] = xr[rd][0];
#pragma unroll
                    for (int n2 = 1; n2 < R2; ++n2) sm[(k1 * R2 + n2) * L + l] = cmul(xr[rd][n2], stw[n2 * k1]);
                }
            }
        } else {
            // ---- forward stage B: the transform of slots k1*R2 + j2 gives X[k1 + R1*k2]; MODE 0 continues in registers
            //      with the kinetic factor and the first inverse stage, whose output n2 goes back to slot k1*R2 + n2 --
            //      a slot this thread read itself, so no barrier is needed inside the stage
#pragma unroll
            for (int rd = 0; rd < RB; ++rd) {
                const int k1 = hi + rd * TPL;
                if (k1 < R1) {                                             // warp-uniform
                    cd xr[R2];
#pragma unroll
                    for (int j2 = 0; j2 < R2; ++j2) xr[j2] = sm[(k1 * R2 + j2) * L + l];
                    Dft<R2, -1>::run(xr);
                    if (MODE == 0 || MODE >= 3) {
                        // Without a cutoff mask no decision hangs on the bits of t, and the kinetic factor is affine in
                        // (G_x+k_x)^2: f = fx * gx2 + f0 with per-line constants (one FMA per value instead of the
                        // masked evaluation in the oracle's order); for the split y transform f_0 + f_1 is affine in
                        // gx2 as well and f_0 - f_1 does not depend on it.
                        const bool affine = MODE == 0 && !(kin.ecut > 0.0);
                        const double hs = 0.5 * kin.scale;
                        const double f0a = hs * (gy2a + gz2), f0b = hs * (gy2b + gz2);
                        const cd wh = half ? w : make_double2(w.x, -w.y);
#pragma unroll
                        for (int k2 = 0; k2 < R2; ++k2) {
                            const double gx2 = sg2x[k1 + R1 * k2];
                            if (S == 1) {
                                const double f = affine ? fma(hs, gx2, f0a) : diag_factor<MODE>(gx2, gy2a, gz2, kin.ecut, kin.scale, ts);
                                xr[k2] = cscale(xr[k2], f);
                            } else {
                                // the radix-2 step of the y transform folded into the factor (header comment)
                                double fs, fd;
                                if (affine) {
                                    fs = fma(kin.scale, gx2, f0a + f0b);
                                    fd = f0a - f0b;
                                } else {
                                    const double fa = diag_factor<MODE>(gx2, gy2a, gz2, kin.ecut, kin.scale, ts);
                                    const double fb = diag_factor<MODE>(gx2, gy2b, gz2, kin.ecut, kin.scale, ts);
                                    fs = fa + fb;
                                    fd = fa - fb;
                                }
                                const cd other = shfl16(xr[k2]);
                                const cd wo = cmul(wh, other);
                                xr[k2] = make_double2(fma(fs, xr[k2].x, fd * wo.x), fma(fs, xr[k2].y, fd * wo.y));
                            }
                        }
                        Dft<R2, +1>::run(xr);
                        sm[(k1 * R2) * L + l] = xr[0];
#pragma unroll
                        for (int n2 = 1; n2 < R2; ++n2) sm[(k1 * R2 + n2) * L + l] = cmul(xr[n2], stw[n2 * k1]);
                    } else {
                        if (S == 2) {
                            // X_0 = A_0 + w A_1 (lane of half 0), X_1 = A_0 - w A_1 (lane of half 1), w = conj(twy_w[rho])
#pragma unroll
                            for (int k2 = 0; k2 < R2; ++k2) {
                                const cd mine = half ? cmulc(xr[k2], w) : xr[k2];  // half 1 sends w A_1, half 0 sends A_0
                                const cd other = shfl16(mine);
                                xr[k2] = half ? csub(other, mine) : cadd(mine, other);
                            }
                        }
#pragma unroll
                        for (int k2 = 0; k2 < R2; ++k2) __stcs(gcol + (size_t)(k1 + R1 * k2) * nynz, xr[k2]);
                    }
                }
            }
        }

        if (MODE == 1) {
            // all reads of the buffer are done: hand it back to the TMA
            fence_proxy_async();
            __syncthreads();
            if (tid == 0 && t + NB * (int)gridDim.x < ntiles) issue(t + NB * gridDim.x, b);
            continue;
        }

        // ---- last inverse stage: transforms n2 = hi, hi + TPL, ... < R2 over the slots k1*R2 + n2 -> x = n2 + R2*n1.
        //      The buffer is handed back to the TMA as soon as the inputs of the last round are in registers.
        __syncthreads();
#pragma unroll
        for (int ra = 0; ra + 1 < RA; ++ra) {
            const int n2 = hi + ra * TPL;
            if (n2 < R2) {
                cd x[R1];
#pragma unroll
                for (int k1 = 0; k1 < R1; ++k1) x[k1] = sm[(k1 * R2 + n2) * L + l];
                Dft<R1, +1>::run(x);
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) __stcs(xdst(n2 + R2 * n1), x[n1]);
            }
        }
        const int n2 = hi + (RA - 1) * TPL;
        cd x[R1];
        if (n2 < R2) {
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) x[k1] = sm[(k1 * R2 + n2) * L + l];
        }
        fence_proxy_async();
        __syncthreads();                  // every read of this buffer is done: refill it
        if (tid == 0 && t + NB * (int)gridDim.x < ntiles) issue(t + NB * gridDim.x, b);
        if (n2 < R2) {
            Dft<R1, +1>::run(x);
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) __stcs(xdst(n2 + R2 * n1), x[n1]);
        }
    }
}

}  // namespace tdh
