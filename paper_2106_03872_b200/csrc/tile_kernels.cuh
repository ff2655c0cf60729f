// tile_kernels.cuh -- the two (y,z)-transform kernels of one Hamiltonian application.
//
//   tile_fwd : per tile: forward FFT along z then y                                   (row a1 of the scope table)
//   tile_inv : per tile: inverse FFT along y then z, then the fused epilogue
//              out = alpha * (T psi + V psi + V_nl psi) + y           (rows a3, a4, a5 back-projection, a6, a7 axpy)
//
// TILE.  Global layout is [state][x][y][z], z fastest.  A tile is the set of rows y = S*m + r (m = 0..NY/S-1) of one
// (state, x) plane: the whole plane when S = 1, the even or the odd rows when S = 2.  S = 2 is used for the large
// planes (96x96, 96x64, 64x96) so that a tile is at most 73,728 bytes and three CTAs fit in the 227 KB of one SM
// (a 96x96 plane is 147 KB: one CTA per SM and no overlap of the load, FFT and store phases).  With S = 2 the tile
// transforms only length-NY/2 sequences along y; the remaining radix-2 butterfly of the y transform commutes with the
// x transform and is done in registers by the x-pencil kernel (xpencil_kernel.cuh), which sees both halves of a line
// pair in one warp.  The spectrum halves are stored at rows r*(NY/2) + k.
//
// SHARED-MEMORY LAYOUT.  One complex128 is a 16-byte cell; a quarter-warp (8 lanes) of a 128-bit access is
// conflict free when its 8 cells are distinct modulo 8.  A row of NZ cells is NZ/8 groups of 8 cells; group index
// g = row*(NZ/8) + k1, cell address 8*g + ((p + g) & 7): the position p inside a group is rotated by g.  Then
//   * the first z stage (radix NZ/8 across groups, fixed p) touches 8 consecutive p of one group per quarter-warp,
//   * the second z stage (radix 8 inside a group) runs over consecutive g with a fixed p,
//   * the y stages run over the 8 positions of one group of one row,
// and all of them are conflict free WITHOUT padding: a 48x96 tile is exactly 73,728 bytes.  Only the final sweep in
// natural z order (8 consecutive z straddle two rotation offsets for NZ = 48, 96) has some 2-way conflicts.
// Every stage overwrites exactly the cells it has read, so one barrier per stage suffices.
//
// 1-D transforms: length N = R1*R2 in two register stages (radix R1 on stride R2, twiddle, radix R2), with
// z: R2 = 8, R1 = NZ/8;  y (length NY/S): 16 = 4x4, 32 = 8x4, 48 = 8x6, 64 = 8x8.
#pragma once
#include "fft_codelets.cuh"

namespace tdh {

__device__ __forceinline__ cd ldg_cd(const cd* p) { return __ldg(p); }
// streaming (evict-first) accesses for the state blocks: they are touched once per kernel and must not push the
// potential, the twiddles and the projector tables out of L2
__device__ __forceinline__ cd lds_cd(const cd* p) { return __ldcs(p); }
__device__ __forceinline__ void sts_cd(cd* p, cd v) { __stcs(p, v); }

template <int N> struct FactY;
template <> struct FactY<16> { static constexpr int R1 = 4, R2 = 4; };
template <> struct FactY<32> { static constexpr int R1 = 8, R2 = 4; };
template <> struct FactY<48> { static constexpr int R1 = 8, R2 = 6; };
template <> struct FactY<64> { static constexpr int R1 = 8, R2 = 8; };
template <> struct FactY<96> { static constexpr int R1 = 12, R2 = 8; };

constexpr int tile_round_up(int a, int b) { return (a + b - 1) / b * b; }

template <int NY, int NZ> struct TileCfg {
    static constexpr int S = (NY * NZ >= 6144) ? 2 : 1;            // y-split (96x96, 96x64, 64x96)
    static constexpr int NYS = NY / S;                              // rows of one plane part
    static constexpr int R1Z = NZ / 8, R2Z = 8;
    static constexpr int R1Y = FactY<NYS>::R1, R2Y = FactY<NYS>::R2;
    static constexpr int PART = NYS * NZ;                           // cells of one plane part
    static constexpr int PPC = PART <= 1152 ? 4 : (PART <= 2304 ? 2 : 1);   // parts per CTA: at most 4608 cells
    static constexpr int ROWS = PPC * NYS;
    static constexpr int CELLS = ROWS * NZ;
    static constexpr size_t SMEM = (size_t)CELLS * sizeof(cd);
    // work items of the four stages
    static constexpr int I_ZA = ROWS * 8, I_ZB = ROWS * R1Z, I_YA = PPC * NZ * R2Y, I_YB = PPC * NZ * R1Y;
    static constexpr int cost(int t) {
        return tile_round_up(I_ZA, t) + tile_round_up(I_ZB, t) + tile_round_up(I_YA, t) + tile_round_up(I_YB, t);
    }
    static constexpr int pick_t() {
        int best = 64;
        const int cand[5] = {64, 96, 128, 192, 256};
        for (int i = 0; i < 5; ++i)
            if (cand[i] * 2 <= I_ZA && cost(cand[i]) <= cost(best)) best = cand[i];
        return best;
    }
    static constexpr int T = pick_t();
    // resident CTAs per SM the launch bounds ask for: limited by shared memory (227 KB, 1 KB reserved per CTA) and by
    // a register budget of >= 80 per thread (>= 104 when the first z stage holds 12 values + 11 twiddles)
    static constexpr int REGS = R1Z > 8 ? 104 : 80;
    static constexpr int by_smem = (int)(232448 / (SMEM + 1024));
    static constexpr int by_regs = 65536 / (T * REGS);
    static constexpr int MINB = by_smem < by_regs ? (by_smem < 1 ? 1 : by_smem) : (by_regs < 1 ? 1 : by_regs);
    static_assert(NZ % 8 == 0 && T % 8 == 0, "z stage mapping");
    static_assert((NYS * R1Z) % 8 == 0, "group rotation must not depend on the plane part");
};

// cell address of (row lr of the tile, group k1, position p): 8*g + ((p + g) & 7), g = lr*R1Z + k1
template <int R1Z> __device__ __forceinline__ int cell_addr(int lr, int k1, int p) {
    const int g = lr * R1Z + k1;
    return 8 * g + ((p + g) & 7);
}

// ------------------------------------------------------------------------------------------------------------
// forward: in -> out (must not alias when S = 2).  Grid: nst * NX * S / PPC tiles.
// ------------------------------------------------------------------------------------------------------------
template <int NY, int NZ>
__global__ void __launch_bounds__(TileCfg<NY, NZ>::T, TileCfg<NY, NZ>::MINB)
tile_fwd_kernel(const cd* __restrict__ in, cd* __restrict__ out, const cd* __restrict__ tw_y,
                const cd* __restrict__ tw_z)
{
    using C = TileCfg<NY, NZ>;
    constexpr int S = C::S, NYS = C::NYS, R1Z = C::R1Z, R1Y = C::R1Y, R2Y = C::R2Y, T = C::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    const int tid = threadIdx.x;
    const int part0 = blockIdx.x * C::PPC;

    // ---- z stage A: global -> registers, radix R1Z over j1 (stride 8 cells), twiddle w^(k1*j2) -> cell (lr, k1, j2)
    {
        const int j2 = tid & 7;
        cd tw[R1Z];
#pragma unroll
        for (int k1 = 1; k1 < R1Z; ++k1) tw[k1] = ldg_cd(tw_z + k1 * j2);
        for (int lr = tid >> 3; lr < C::ROWS; lr += T / 8) {
            const int lp = lr / NYS, m = lr % NYS;
            const int part = part0 + lp, plane = part / S, r = part % S;
            const cd* src = in + (size_t)plane * NY * NZ + (size_t)(S * m + r) * NZ + j2;
            cd x[R1Z];
#pragma unroll
            for (int j1 = 0; j1 < R1Z; ++j1) x[j1] = lds_cd(src + j1 * 8);
            Dft<R1Z, -1>::run(x);
            sm[cell_addr<R1Z>(lr, 0, j2)] = x[0];
#pragma unroll
            for (int k1 = 1; k1 < R1Z; ++k1) sm[cell_addr<R1Z>(lr, k1, j2)] = cmulc(x[k1], tw[k1]);
        }
    }
    __syncthreads();
    // ---- z stage B, in place inside group g: position k2 then holds kz = k1 + R1Z*k2
    for (int g = tid; g < C::I_ZB; g += T) {
        cd* p = sm + 8 * g;
        const int s = g & 7;
        cd t[8];
#pragma unroll
        for (int j2 = 0; j2 < 8; ++j2) t[j2] = p[(j2 + s) & 7];
        Dft<8, -1>::run(t);
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) p[(k2 + s) & 7] = t[k2];
    }
    __syncthreads();
    // ---- y stage A, in place: rows j1*R2Y + j2 of column c = (k1, k2) -> rows k1y*R2Y + j2
    for (int item = tid; item < C::I_YA; item += T) {
        const int c = item % NZ, rr = item / NZ, j2 = rr % R2Y, lp = rr / R2Y;
        const int k1 = c >> 3, k2 = c & 7;
        const int row0 = lp * NYS + j2;
        cd x[R1Y];
#pragma unroll
        for (int j1 = 0; j1 < R1Y; ++j1) x[j1] = sm[cell_addr<R1Z>(row0 + j1 * R2Y, k1, k2)];
        Dft<R1Y, -1>::run(x);
        sm[cell_addr<R1Z>(row0, k1, k2)] = x[0];
#pragma unroll
        for (int k1y = 1; k1y < R1Y; ++k1y)
            sm[cell_addr<R1Z>(row0 + k1y * R2Y, k1, k2)] = cmulc(x[k1y], ldg_cd(tw_y + S * k1y * j2));
    }
    __syncthreads();
    // ---- y stage B -> global, natural kz order; spectrum half r goes to rows r*NYS + ky
    for (int item = tid; item < C::I_YB; item += T) {
        const int kz = item % NZ, rr = item / NZ, k1y = rr % R1Y, lp = rr / R1Y;
        const int k1 = kz % R1Z, k2 = kz / R1Z;
        const int row0 = lp * NYS + k1y * R2Y;
        cd t[R2Y];
#pragma unroll
        for (int j2 = 0; j2 < R2Y; ++j2) t[j2] = sm[cell_addr<R1Z>(row0 + j2, k1, k2)];
        Dft<R2Y, -1>::run(t);
        const int part = part0 + lp, plane = part / S, r = part % S;
        cd* dst = out + (size_t)plane * NY * NZ + (size_t)(r * NYS) * NZ + kz;
#pragma unroll
        for (int k2y = 0; k2y < R2Y; ++k2y) dst[(size_t)(k1y + R1Y * k2y) * NZ] = t[k2y];
    }
}

// Arguments of the fused epilogue of tile_inv.
struct Epilogue {
    const cd* phi;          // input block of this application (for V*phi); used only when v != NULL
    const double* v;        // V(r), n0*n1*n2; NULL: no local term
    const cd* yv;           // optional addend y (same block layout as out); NULL: none
    cd alpha;               // out = alpha * (T + V + Vnl) phi + y
    int nx;                 // planes per state
    // Kleinman-Bylander back-projection (second half of Eq. 9), as per-tile record lists; nl_off == NULL: none.
    // Tile (x, r) owns records nl_off[(x*S + r)*(nl_layers+1) + l] .. [.. + l + 1) of layer l; within one layer every
    // grid point appears at most once, so the shared-memory read-modify-write needs no atomics.
    const int* nl_off;
    int nl_layers;
    const unsigned* nl_cc;  // per record: cell address inside the plane part | first channel << 16
    const double* nl_beta;  // [cmax][nrec] projector values, zero padded above the atom's channel count
    const cd* nl_phase;     // per record e^{+ik.d}; NULL at Gamma
    const cd* dpi;          // [state][nchan_tot] D * dV * <beta|phi>  (+ cmax zeroed entries of padding)
    int nrec;
    int cmax;
    int nchan_tot;
};

// ------------------------------------------------------------------------------------------------------------
// inverse + epilogue: in -> out (must not alias when S = 2)
// ------------------------------------------------------------------------------------------------------------
template <int NY, int NZ>
__global__ void __launch_bounds__(TileCfg<NY, NZ>::T, TileCfg<NY, NZ>::MINB)
tile_inv_kernel(const cd* __restrict__ in, cd* __restrict__ out, const cd* __restrict__ tw_y,
                const cd* __restrict__ tw_z, const Epilogue ep)
{
    using C = TileCfg<NY, NZ>;
    constexpr int S = C::S, NYS = C::NYS, R1Z = C::R1Z, R1Y = C::R1Y, R2Y = C::R2Y, T = C::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* sm = reinterpret_cast<cd*>(smem_raw);
    const int tid = threadIdx.x;
    const int part0 = blockIdx.x * C::PPC;

    // ---- y stage A: global rows r*NYS + n1*R2Y + n2 -> registers, radix R1Y, twiddle -> rows m1*R2Y + n2
    for (int item = tid; item < C::I_YA; item += T) {
        const int kz = item % NZ, rr = item / NZ, n2 = rr % R2Y, lp = rr / R2Y;
        const int part = part0 + lp, plane = part / S, r = part % S;
        const cd* src = in + (size_t)plane * NY * NZ + (size_t)(r * NYS + n2) * NZ + kz;
        cd x[R1Y];
#pragma unroll
        for (int n1 = 0; n1 < R1Y; ++n1) x[n1] = lds_cd(src + (size_t)n1 * R2Y * NZ);
        Dft<R1Y, +1>::run(x);
        const int row0 = lp * NYS + n2, grp = kz >> 3, pos = kz & 7;
        sm[cell_addr<R1Z>(row0, grp, pos)] = x[0];
#pragma unroll
        for (int m1 = 1; m1 < R1Y; ++m1)
            sm[cell_addr<R1Z>(row0 + m1 * R2Y, grp, pos)] = cmul(x[m1], ldg_cd(tw_y + S * m1 * n2));
    }
    __syncthreads();
    // ---- y stage B, in place: row m1*R2Y + m2 then holds m = m1 + R1Y*m2, i.e. y = S*m + r
    for (int item = tid; item < C::I_YB; item += T) {
        const int c = item % NZ, rr = item / NZ, m1 = rr % R1Y, lp = rr / R1Y;
        const int grp = c >> 3, pos = c & 7;
        const int row0 = lp * NYS + m1 * R2Y;
        cd t[R2Y];
#pragma unroll
        for (int n2 = 0; n2 < R2Y; ++n2) t[n2] = sm[cell_addr<R1Z>(row0 + n2, grp, pos)];
        Dft<R2Y, +1>::run(t);
#pragma unroll
        for (int m2 = 0; m2 < R2Y; ++m2) sm[cell_addr<R1Z>(row0 + m2, grp, pos)] = t[m2];
    }
    __syncthreads();
    // ---- z stage A, in place: input kz = 8*n1 + n2 sits at (group n1, position n2); radix R1Z over n1, twiddle
    {
        const int n2 = tid & 7;
        cd tw[R1Z];
#pragma unroll
        for (int m1 = 1; m1 < R1Z; ++m1) tw[m1] = ldg_cd(tw_z + m1 * n2);
        for (int lr = tid >> 3; lr < C::ROWS; lr += T / 8) {
            cd x[R1Z];
#pragma unroll
            for (int n1 = 0; n1 < R1Z; ++n1) x[n1] = sm[cell_addr<R1Z>(lr, n1, n2)];
            Dft<R1Z, +1>::run(x);
            sm[cell_addr<R1Z>(lr, 0, n2)] = x[0];
#pragma unroll
            for (int m1 = 1; m1 < R1Z; ++m1) sm[cell_addr<R1Z>(lr, m1, n2)] = cmul(x[m1], tw[m1]);
        }
    }
    __syncthreads();
    // ---- z stage B, in place: (group m1, position m2) then holds z = m1 + R1Z*m2 of the kinetic term
    for (int g = tid; g < C::I_ZB; g += T) {
        cd* p = sm + 8 * g;
        const int s = g & 7;
        cd t[8];
#pragma unroll
        for (int n2 = 0; n2 < 8; ++n2) t[n2] = p[(n2 + s) & 7];
        Dft<8, +1>::run(t);
#pragma unroll
        for (int m2 = 0; m2 < 8; ++m2) p[(m2 + s) & 7] = t[m2];
    }
    __syncthreads();
    // ---- Kleinman-Bylander back-projection into the tile (layer by layer: no two records of a layer share a cell)
    if (ep.nl_off != nullptr) {
        for (int layer = 0; layer < ep.nl_layers; ++layer) {
#pragma unroll
            for (int lp = 0; lp < C::PPC; ++lp) {
                const int part = part0 + lp, plane = part / S, r = part % S;
                const int st = plane / ep.nx, x = plane % ep.nx;
                const int* off = ep.nl_off + (size_t)(x * S + r) * (ep.nl_layers + 1) + layer;
                const int i1 = __ldg(off + 1);
                const cd* dp = ep.dpi + (size_t)st * ep.nchan_tot;
                cd* base = sm + lp * C::PART;
                for (int i = __ldg(off) + tid; i < i1; i += T) {
                    const unsigned cc = __ldg(ep.nl_cc + i);
                    const cd* d = dp + (cc >> 16);
                    const double* b = ep.nl_beta + i;
                    cd s = make_double2(0.0, 0.0);
                    for (int c = 0; c < ep.cmax; ++c) {
                        const double bv = __ldg(b + (size_t)c * ep.nrec);
                        const cd dv = ldg_cd(d + c);
                        s.x = fma(bv, dv.x, s.x);
                        s.y = fma(bv, dv.y, s.y);
                    }
                    if (ep.nl_phase != nullptr) s = cmulc(s, ldg_cd(ep.nl_phase + i));
                    cd* cell = base + (cc & 0xffffu);
                    *cell = cadd(*cell, s);
                }
            }
            __syncthreads();
        }
    }
    // ---- sweep in natural z order: out = alpha * (T phi + V phi + Vnl phi) + y
    for (int item = tid; item < C::CELLS; item += T) {
        const int z = item % NZ, lr = item / NZ;
        const int lp = lr / NYS, rho = lr % NYS;
        const int part = part0 + lp, plane = part / S, r = part % S;
        const int y = S * (rho / R2Y + R1Y * (rho % R2Y)) + r;
        cd acc = sm[cell_addr<R1Z>(lr, z % R1Z, z / R1Z)];
        const size_t gi = (size_t)plane * NY * NZ + (size_t)y * NZ + z;                    // index in the block
        if (ep.v != nullptr) {
            const size_t q = ((size_t)(plane % ep.nx) * NY + y) * NZ + z;                 // index in the state
            const cd ph = lds_cd(ep.phi + gi);
            const double vv = __ldg(ep.v + q);
            acc.x = fma(vv, ph.x, acc.x);
            acc.y = fma(vv, ph.y, acc.y);
        }
        cd o = cmul(ep.alpha, acc);
        if (ep.yv != nullptr) o = cadd(o, lds_cd(ep.yv + gi));
        sts_cd(out + gi, o);
    }
}

}  // namespace tdh
