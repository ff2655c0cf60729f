// small_kernels.cuh -- H|psi> of a small grid in ONE launch, the whole state on chip (SURVEY.md section 7 "Hard parts",
// section 8(d) "on-chip whole-state plan"; rows a1-a7 of the scope table, Eq. 2 / Eq. 9 / Eq. 8's axpy).
//
// For the grids whose state fits in shared memory -- 16^3 (64 KB: one CTA) and 32^3 (512 KB: a cluster of four CTAs, 128 KB
// each) -- the four launches of the tiled path (nl_project, tile_fwd, xpencil, tile_inv) are bound by launch latency, not
// by bytes.  Here one CTA (cluster) owns one state from the load of psi to the store of
//     out = alpha * (T psi + V psi + V_nl psi) + y
// and nothing but psi, V, y and the projector tables is read from global memory, nothing but `out` written.
//
// LAYOUT.  CTA c of the cluster (c < CS) holds the planes x = CS*j + c, j < NJ = N/CS, each in the swizzled 128-byte-line
// layout of tile_kernels.cuh (cell of (y, z) = swz(y*N/8 + (z >> 3), z & 7)), so the (z, y) stages are the tile kernels'
// stages on a tile of NJ planes and the back-projection uses the handle's per-plane record lists unchanged.
//
// x TRANSFORM.  x = CS*j + c splits X[k1 + NJ*k2] = sum_c w_CS^(c k2) [ w_N^(c k1) A_c[k1] ],  A_c = FFT_NJ over j.
// CS = 1: one in-register radix-16 pass per pencil with the kinetic factor between forward and inverse.  CS = 4: local
// radix-8 + twiddle; cluster barrier; the radix-4 across the four CTAs runs over distributed shared memory -- a thread
// owns a group (k1, cell), reads its four values (one local, three remote), transforms, applies the kinetic factor
// 1/2|G+k|^2 (work-layout tables of the handle) with the 1/N_p of the inverse, transforms back and writes the four
// values where it found them; cluster barrier; inverse twiddle + radix-8.  Every value crosses the cluster once each way.
//
// PROJECTORS.  <beta|psi> is taken from the planes in shared memory before the first butterfly: a warp per atom over the
// atom's sorted sphere list (points of other CTAs' planes skipped), fixed-order shuffle reduction, the CTAs' partial sums
// added in rank order through distributed shared memory (bitwise the same on every CTA), times D dV.
#pragma once
#include <cooperative_groups.h>

#include "nl_kernels.cuh"
#include "tile_kernels.cuh"
#include "xpencil_kernel.cuh"

namespace tdh {

namespace cg = cooperative_groups;

constexpr int SMALL_T = 512;               // threads of the 16^3 kernel; SmallCfg<N, CS>::T for each kernel
#ifndef TDH_SMALL_T32
#define TDH_SMALL_T32 512
#endif
constexpr int SMALL_MAX_CHAN = 1024;
constexpr int SMALL_HEADER = 2048;        // twiddle tables

template <int N, int CS> struct SmallCfg {
    static constexpr int NJ = N / CS;
    static constexpr int R1Z = N / 8;
    static constexpr int R1Y = FactY<N>::R1, R2Y = FactY<N>::R2;
    static constexpr int PLANE = N * N;
    static constexpr int ROWS = NJ * N;
    static constexpr int CELLS = ROWS * N;
    static constexpr int T = N == 32 ? TDH_SMALL_T32 : SMALL_T;
    static_assert(NJ == 16 || NJ == 8 || NJ == 4, "local x transform is one radix-16, radix-8 or radix-4 pass");
    static_assert(CS == 1 || CS == 4, "cluster of one or four CTAs");
    static_assert((2 * N + NJ) * sizeof(cd) <= SMALL_HEADER, "twiddle tables must fit in the header");
};
constexpr int SMALL_MAX_SEG = 8;          // an atom's sphere list is split over up to 8 warps
constexpr int SMALL_SEG_ENTRIES = 2048;   // bound of (segments x channels) partial sums kept in shared memory
// segments per atom: enough to give every warp work, bounded by the partial-sum buffer
__host__ __device__ constexpr int small_segments(int natoms, int nchan) {
    int g = natoms > 0 ? (SMALL_T / 32 + natoms - 1) / natoms : 1;
    if (g > SMALL_MAX_SEG) g = SMALL_MAX_SEG;
    while (g > 1 && g * nchan > SMALL_SEG_ENTRIES) --g;
    return g < 1 ? 1 : g;
}
// dynamic shared memory: header, the planes, segment partials, partial and summed projections (+ 16 zeroed entries)
__host__ __device__ constexpr size_t small_smem(int cells, int natoms, int nchan) {
    return SMALL_HEADER + (size_t)cells * sizeof(cd) +
           (size_t)(small_segments(natoms, nchan) * nchan + 2 * nchan + 16) * sizeof(cd);
}

struct SmallProj {
    const AtomDesc* atoms;
    const int* sidx;
    const double* sbeta;
    const cd* sphase;       // NULL at Gamma
    const double* dscale;   // D dV per channel
    int natoms;
    int nchan_tot;
};

template <int N, int CS>
__global__ void __launch_bounds__(SmallCfg<N, CS>::T, 1)
small_h_kernel(const cd* __restrict__ psi, cd* __restrict__ out, const cd* __restrict__ tw_x, const cd* __restrict__ tw_y,
               const cd* __restrict__ tw_z, const Kinetic kin, const Epilogue ep, const SmallProj pj)
{
    using C = SmallCfg<N, CS>;
    constexpr int NJ = C::NJ, R1Z = C::R1Z, R1Y = C::R1Y, R2Y = C::R2Y, PLANE = C::PLANE, ROWS = C::ROWS, T = C::T;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    cd* stw_z = reinterpret_cast<cd*>(smem_raw);                        // [k1][j2] = e^{+2 pi i k1 j2 / N}
    cd* stw_y = stw_z + N;                                              // e^{+2 pi i m / N}
    cd* stw_x = stw_y + N;                                              // e^{+2 pi i c k1 / N}, k1 < NJ
    cd* sm = reinterpret_cast<cd*>(smem_raw + SMALL_HEADER);
    const int nseg = small_segments(pj.natoms, pj.nchan_tot);
    cd* dseg = sm + C::CELLS;                                           // [segment][nchan_tot] partial projections of this CTA
    cd* dpart = dseg + nseg * pj.nchan_tot;                             // this CTA's partial projections [nchan_tot]
    cd* dsum = dpart + pj.nchan_tot;                                    // D dV <beta|psi> [nchan_tot] + 16 zeros
    __shared__ int rec_pref[2 * 16 + 1];                                // record ranges of the planes of one layer
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int crank = CS > 1 ? (int)cg::this_cluster().block_rank() : 0;
    const int st = blockIdx.x / CS;
    const cd* psi_s = psi + (size_t)st * N * PLANE;
    const bool have_nl = ep.nl_off != nullptr;
    const bool have_v = ep.v != nullptr;

    for (int i = tid; i < N; i += T) {
        stw_z[i] = ldg_cd(tw_z + (i >> 3) * (i & 7));
        stw_y[i] = ldg_cd(tw_y + i);
    }
    for (int i = tid; i < NJ; i += T) stw_x[i] = ldg_cd(tw_x + (crank * i) % N);
    for (int i = tid; i < pj.nchan_tot + 16; i += T) dsum[i] = make_double2(0.0, 0.0);
    // ---- load the CTA's planes, natural (y, z) order into swizzled cells; sixteen loads in flight per thread
    {
        constexpr int U = 16;
        for (int i0 = tid; i0 < C::CELLS; i0 += U * T) {
            cd v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * T, j = i / PLANE, yz = i % PLANE;
                if (i < C::CELLS) v[u] = lds_cd(psi_s + (size_t)(CS * j + crank) * PLANE + yz);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * T, j = i / PLANE, yz = i % PLANE, y = yz / N, z = yz % N;
                if (i < C::CELLS) sm[j * PLANE + swz(y * R1Z + (z >> 3), z & 7)] = v[u];
            }
        }
    }
    __syncthreads();

    // ---- projections over this CTA's planes: work item = (atom, segment of its sorted sphere list), one warp each;
    //      four points per lane in flight; fixed-order sums (lanes by shuffle, segments in order): deterministic
    if (have_nl) {
        for (int item = warp; item < pj.natoms * nseg; item += T / 32) {
            const int a = item / nseg, sg = item % nseg;
            const AtomDesc at = pj.atoms[a];
            const int per = ((at.np + nseg - 1) / nseg + 31) / 32 * 32;
            const int q0 = sg * per, q1 = min(at.np, q0 + per);
            for (int c0 = 0; c0 < at.nchan; c0 += 4) {
                cd acc[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[c] = make_double2(0.0, 0.0);
                for (int qb = q0 + lane; qb < q1; qb += 4 * 32) {
                    int pp[4];
                    double bb[4][4];
                    cd ph[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int q = qb + 32 * u;
                        const bool ok = q < q1;
                        pp[u] = ok ? __ldg(pj.sidx + at.q0 + q) : -1;
#pragma unroll
                        for (int c = 0; c < 4; ++c)
                            bb[u][c] = (ok && c0 + c < at.nchan) ? __ldg(pj.sbeta + at.boff + (size_t)(c0 + c) * at.np + q) : 0.0;
                        if (pj.sphase != nullptr) ph[u] = ok ? __ldg(pj.sphase + at.q0 + q) : make_double2(1.0, 0.0);
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int p = pp[u], x = p / PLANE;
                        if (p >= 0 && (CS == 1 || x % CS == crank)) {
                            const int yz = p % PLANE, y = yz / N, z = yz % N;
                            cd v = sm[(x / CS) * PLANE + swz(y * R1Z + (z >> 3), z & 7)];
                            if (pj.sphase != nullptr) v = cmul(v, ph[u]);
#pragma unroll
                            for (int c = 0; c < 4; ++c) {
                                acc[c].x = fma(bb[u][c], v.x, acc[c].x);
                                acc[c].y = fma(bb[u][c], v.y, acc[c].y);
                            }
                        }
                    }
                }
#pragma unroll
                for (int c = 0; c < 4; ++c) {
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        acc[c].x += __shfl_xor_sync(0xffffffffu, acc[c].x, o);
                        acc[c].y += __shfl_xor_sync(0xffffffffu, acc[c].y, o);
                    }
                    if (lane == 0 && c0 + c < at.nchan) dseg[sg * pj.nchan_tot + at.chan0 + c0 + c] = acc[c];
                }
            }
        }
        __syncthreads();
        for (int i = tid; i < pj.nchan_tot; i += T) {
            cd t = dseg[i];
            for (int sg = 1; sg < nseg; ++sg) t = cadd(t, dseg[sg * pj.nchan_tot + i]);
            dpart[i] = t;
            if (CS == 1) dsum[i] = cscale(t, __ldg(pj.dscale + i));
        }
        __syncthreads();
    }

    // ---- forward z: radix N/8 over j1 (lines), twiddle; radix 8 inside a line (tile_fwd's stages, all in place)
    {
        const int j2 = tid & 7;
        for (int lr = tid >> 3; lr < ROWS; lr += T / 8) {
            const int l0 = lr * R1Z;
            cd x[R1Z];
#pragma unroll
            for (int j1 = 0; j1 < R1Z; ++j1) x[j1] = sm[swz(l0 + j1, j2)];
            Dft<R1Z, -1>::run(x);
            sm[swz(l0, j2)] = x[0];
#pragma unroll
            for (int k1 = 1; k1 < R1Z; ++k1) sm[swz(l0 + k1, j2)] = cmulc(x[k1], stw_z[8 * k1 + j2]);
        }
    }
    __syncthreads();
    for (int g = tid; g < ROWS * R1Z; g += T) {
        cd* p = sm + 8 * g;
        const int s = g & 7;
        cd v[8];
#pragma unroll
        for (int j2 = 0; j2 < 8; ++j2) v[j2] = p[j2 ^ s];
        Dft<8, -1>::run(v);
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) p[k2 ^ s] = v[k2];
    }
    __syncthreads();
    // ---- forward y: rows j1*R2Y + j2 -> k1y*R2Y + j2 with twiddle, then radix R2Y inside each group of R2Y rows
    for (int item = tid; item < NJ * N * R2Y; item += T) {
        const int c = item % N, rr = item / N, j2 = rr % R2Y, lp = rr / R2Y;
        const int k1 = c >> 3, k2 = c & 7;
        const int row0 = lp * N + j2;
        cd x[R1Y];
#pragma unroll
        for (int j1 = 0; j1 < R1Y; ++j1) x[j1] = sm[swz((row0 + j1 * R2Y) * R1Z + k1, k2)];
        Dft<R1Y, -1>::run(x);
        sm[swz(row0 * R1Z + k1, k2)] = x[0];
#pragma unroll
        for (int k1y = 1; k1y < R1Y; ++k1y) sm[swz((row0 + k1y * R2Y) * R1Z + k1, k2)] = cmulc(x[k1y], stw_y[k1y * j2]);
    }
    __syncthreads();
    for (int item = tid; item < NJ * N * R1Y; item += T) {
        const int c = item % N, rr = item / N, k1y = rr % R1Y, lp = rr / R1Y;
        const int k1 = c >> 3, k2 = c & 7;
        const int row0 = lp * N + k1y * R2Y;
        cd v[R2Y];
#pragma unroll
        for (int j2 = 0; j2 < R2Y; ++j2) v[j2] = sm[swz((row0 + j2) * R1Z + k1, k2)];
        Dft<R2Y, -1>::run(v);
#pragma unroll
        for (int k2y = 0; k2y < R2Y; ++k2y) sm[swz((row0 + k2y) * R1Z + k1, k2)] = v[k2y];
    }
    __syncthreads();

    // ---- x: forward, kinetic factor (work-layout tables: physical cell -> plane row Y, column z'), inverse
    auto factor = [&](int kx, int pc) -> double {
        const int ln = pc >> 3, pos = (pc & 7) ^ (ln & 7);
        const int Y = ln / R1Z, zp = 8 * (ln % R1Z) + pos;
        const double gx2 = __ldg(kin.g2x + kx), gy2 = __ldg(kin.g2y_w + Y), gz2 = __ldg(kin.g2z_w + zp);
        return kin_factor(gx2, gy2, gz2, kin.ecut, kin.scale);
    };
    if (CS == 1) {
        for (int pc = tid; pc < PLANE; pc += T) {
            cd x[NJ];
#pragma unroll
            for (int j = 0; j < NJ; ++j) x[j] = sm[j * PLANE + pc];
            Dft<NJ, -1>::run(x);
#pragma unroll
            for (int kx = 0; kx < NJ; ++kx) x[kx] = cscale(x[kx], factor(kx, pc));
            Dft<NJ, +1>::run(x);
#pragma unroll
            for (int j = 0; j < NJ; ++j) sm[j * PLANE + pc] = x[j];
        }
        __syncthreads();
    } else {
        cg::cluster_group cl = cg::this_cluster();
        for (int pc = tid; pc < PLANE; pc += T) {
            cd x[NJ];
#pragma unroll
            for (int j = 0; j < NJ; ++j) x[j] = sm[j * PLANE + pc];
            Dft<NJ, -1>::run(x);
            sm[pc] = x[0];
#pragma unroll
            for (int k1 = 1; k1 < NJ; ++k1) sm[k1 * PLANE + pc] = cmulc(x[k1], stw_x[k1]);
        }
        cl.sync();
        cd* peer[4];
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) peer[cc] = cl.map_shared_rank(sm, cc);
        if (have_nl) {                    // sum of the CTAs' partial projections, rank order, times D dV
            const cd* dp[4];
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) dp[cc] = cl.map_shared_rank(dpart, cc);
            for (int i = tid; i < pj.nchan_tot; i += T) {
                cd s = dp[0][i];
#pragma unroll
                for (int cc = 1; cc < 4; ++cc) s = cadd(s, dp[cc][i]);
                dsum[i] = cscale(s, __ldg(pj.dscale + i));
            }
        }
        // groups (k1, cell) of this CTA's quarter of the plane cells
        constexpr int QUARTER = PLANE / 4;
        for (int item = tid; item < NJ * QUARTER; item += T) {
            const int k1 = item / QUARTER, pc = crank * QUARTER + item % QUARTER;
            const int off = k1 * PLANE + pc;
            cd v[4];
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) v[cc] = peer[cc][off];
            Dft<4, -1>::run(v);
#pragma unroll
            for (int k2 = 0; k2 < 4; ++k2) v[k2] = cscale(v[k2], factor(k1 + NJ * k2, pc));
            Dft<4, +1>::run(v);
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) peer[cc][off] = v[cc];
        }
        cl.sync();
        for (int pc = tid; pc < PLANE; pc += T) {
            cd x[NJ];
            x[0] = sm[pc];
#pragma unroll
            for (int k1 = 1; k1 < NJ; ++k1) x[k1] = cmul(sm[k1 * PLANE + pc], stw_x[k1]);
            Dft<NJ, +1>::run(x);
#pragma unroll
            for (int j = 0; j < NJ; ++j) sm[j * PLANE + pc] = x[j];
        }
        __syncthreads();
    }

    // ---- inverse y, inverse z (tile_inv's stages), ending in natural order in place
    for (int item = tid; item < NJ * N * R1Y; item += T) {
        const int c = item % N, rr = item / N, k1y = rr % R1Y, lp = rr / R1Y;
        const int k1 = c >> 3, k2 = c & 7;
        const int row0 = lp * N + k1y * R2Y;
        cd v[R2Y];
#pragma unroll
        for (int k2y = 0; k2y < R2Y; ++k2y) v[k2y] = sm[swz((row0 + k2y) * R1Z + k1, k2)];
        Dft<R2Y, +1>::run(v);
        sm[swz(row0 * R1Z + k1, k2)] = v[0];
#pragma unroll
        for (int j2 = 1; j2 < R2Y; ++j2) sm[swz((row0 + j2) * R1Z + k1, k2)] = cmul(v[j2], stw_y[j2 * k1y]);
    }
    __syncthreads();
    for (int item = tid; item < NJ * N * R2Y; item += T) {
        const int c = item % N, rr = item / N, j2 = rr % R2Y, lp = rr / R2Y;
        const int k1 = c >> 3, k2 = c & 7;
        const int row0 = lp * N + j2;
        cd x[R1Y];
#pragma unroll
        for (int k1y = 0; k1y < R1Y; ++k1y) x[k1y] = sm[swz((row0 + k1y * R2Y) * R1Z + k1, k2)];
        Dft<R1Y, +1>::run(x);
#pragma unroll
        for (int j1 = 0; j1 < R1Y; ++j1) sm[swz((row0 + j1 * R2Y) * R1Z + k1, k2)] = x[j1];
    }
    __syncthreads();
    for (int g = tid; g < ROWS * R1Z; g += T) {
        cd* p = sm + 8 * g;
        const int s = g & 7;
        cd v[8];
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) v[k2] = p[k2 ^ s];
        Dft<8, +1>::run(v);
#pragma unroll
        for (int j2 = 0; j2 < 8; ++j2) p[j2 ^ s] = v[j2];
    }
    __syncthreads();
    {
        const int j2 = tid & 7;
        for (int lr = tid >> 3; lr < ROWS; lr += T / 8) {
            const int l0 = lr * R1Z;
            cd x[R1Z];
            x[0] = sm[swz(l0, j2)];
#pragma unroll
            for (int k1 = 1; k1 < R1Z; ++k1) x[k1] = cmul(sm[swz(l0 + k1, j2)], stw_z[8 * k1 + j2]);
            Dft<R1Z, +1>::run(x);
#pragma unroll
            for (int j1 = 0; j1 < R1Z; ++j1) sm[swz(l0 + j1, j2)] = x[j1];
        }
    }
    __syncthreads();

    // ---- back-projection from the handle's per-plane record lists, layer by layer (a layer holds a cell at most once).
    //      The record ranges of the CTA's NJ planes are gathered first, then the threads run over their concatenation.
    if (have_nl) {
        const int cm = ep.cmax;
        for (int layer = 0; layer < ep.nl_layers; ++layer) {
            if (tid < NJ) {
                const int* off = ep.nl_off + (size_t)(CS * tid + crank) * (ep.nl_layers + 1) + layer;
                rec_pref[tid] = __ldg(off);                      // first record of plane tid
                rec_pref[16 + tid] = __ldg(off + 1) - __ldg(off);   // count
            }
            __syncthreads();
            int total = 0;
#pragma unroll
            for (int j = 0; j < NJ; ++j) total += rec_pref[16 + j];
            for (int e = tid; e < total; e += T) {
                int j = 0, r = e;
                while (r >= rec_pref[16 + j]) { r -= rec_pref[16 + j]; ++j; }
                const int i = rec_pref[j] + r;
                const unsigned cc = __ldg(ep.nl_cc + i);
                const cd* d = dsum + (cc >> 16);
                cd sacc = make_double2(0.0, 0.0);
                for (int c = 0; c < cm; ++c) {
                    const double b = __ldg(ep.nl_beta + (size_t)c * ep.nrec + i);
                    sacc.x = fma(b, d[c].x, sacc.x);
                    sacc.y = fma(b, d[c].y, sacc.y);
                }
                if (ep.nl_phase != nullptr) sacc = cmulc(sacc, __ldg(ep.nl_phase + i));
                cd* cell = sm + j * PLANE + (cc & 0xffffu);
                *cell = cadd(*cell, sacc);
            }
            __syncthreads();
        }
    }

    // ---- epilogue: out = alpha * (tile + V psi) + y, natural order, coalesced; eight points per thread in flight
    cd* out_s = out + (size_t)st * N * PLANE;
    const cd* yv_s = ep.yv != nullptr ? ep.yv + (size_t)st * N * PLANE : nullptr;
    {
        constexpr int U = 8;
        for (int i0 = tid; i0 < C::CELLS; i0 += U * T) {
            double vv[U];
            cd ph[U], ya[U];
            size_t gi[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * T, j = i / PLANE, yz = i % PLANE;
                gi[u] = (size_t)(CS * j + crank) * PLANE + yz;
                if (i >= C::CELLS) continue;
                if (have_v) { vv[u] = __ldg(ep.v + gi[u]); ph[u] = lds_cd(psi_s + gi[u]); }
                if (yv_s != nullptr) ya[u] = lds_cd(yv_s + gi[u]);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * T, j = i / PLANE, yz = i % PLANE, y = yz / N, z = yz % N;
                if (i >= C::CELLS) continue;
                cd x = sm[j * PLANE + swz(y * R1Z + (z >> 3), z & 7)];
                if (have_v) {
                    x.x = fma(vv[u], ph[u].x, x.x);
                    x.y = fma(vv[u], ph[u].y, x.y);
                }
                cd r = cmul(ep.alpha, x);
                if (yv_s != nullptr) r = cadd(r, ya[u]);
                sts_cd(out_s + gi[u], r);
            }
        }
    }
    if (CS > 1) cg::this_cluster().sync();          // no CTA leaves while a peer may still address its shared memory
}

}  // namespace tdh
