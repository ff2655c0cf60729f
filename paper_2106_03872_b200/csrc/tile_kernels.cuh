// tile_kernels.cuh -- the two (y,z)-transform kernels of one Hamiltonian application (persistent, TMA-fed).
//
//   tile_fwd : per tile: forward FFT along z then y                                   (row a1 of the scope table)
//   tile_inv : per tile: inverse FFT along y then z, then the fused epilogue
//              out = alpha * (T psi + V psi [+ V_nl psi]) + y         (rows a3, a4, a5 back-projection, a6, a7 axpy)
// Both kernels run two independent warp groups per CTA on a ring of three tiles (see tile_fwd_kernel).
//
// TILE.  Global layout is [state][x][y][z], z fastest.  A tile is the set of rows y = S*m + r (m = 0..NY/S-1) of one
// (state, x) plane: the whole plane when S = 1 (PPC consecutive planes when they are small), the even or the odd rows
// when S = 2.  S = 2 is used for the large planes (96x96, 96x64, 64x96) so that a tile is at most 73,728 bytes and a
// ring of three tiles fits in the 227 KB of one SM.  With S = 2 the tile transforms only length-NY/2 sequences along
// y; the remaining radix-2 butterfly of the y transform commutes with the x transform and is done in registers by the
// x-pencil kernel (xpencil_kernel.cuh), which sees both parts of a row pair in one warp.
//
// TMA + SWIZZLE.  A tile is one 4-D box {16 doubles, NZ/8, NY/S, PPC} of a tensor map with 128-byte swizzling
// (tensor_maps.h): the 128-byte line Ln = row*(NZ/8) + (z >> 3) lands at byte 128*Ln of a 1024-byte aligned buffer
// and complex value p = z & 7 of the line at chunk p ^ (Ln & 7).  With that hardware XOR swizzle every stage below is
// free of bank conflicts without padding: a quarter-warp always touches 8 distinct 16-byte chunks modulo 128 bytes
// (8 positions of one line, or one position of 8 consecutive lines).  CTAs are persistent; the thread that releases a
// buffer refills it with cp.async.bulk.tensor, so the next tiles stream in while this one is transformed.
//
// ORDER.  1-D transforms of length N = R1*R2 run as two in-place register stages.  Forward (natural in): radix R1 over
// j1 (stride R2), twiddle, radix R2 over j2; position k1*R2 + k2 then holds index k1 + R1*k2.  The inverse takes
// exactly that digit-permuted order as input (radix R2 over k2, twiddle, radix R1 over k1) and ends in natural order,
// so no reordering pass exists anywhere: the x-pencil kernel works on permuted lines.  z: R2 = 8, R1 = NZ/8;
// y (length NY/S): 16 = 4x4, 32 = 8x4, 48 = 8x6, 64 = 8x8.
#pragma once
#include "fft_codelets.cuh"
#include "tma.cuh"

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
constexpr int TILE_MAX_CELLS = 4608;
constexpr int TILE_HEADER_FWD = 4096;  // barriers (64 bytes), then the z and y twiddle tables; keeps the buffers 1024-byte aligned
constexpr int TILE_TW_OFF = 64;

template <int NY, int NZ> struct TileCfg {
    static constexpr int S = (NY * NZ >= 6144) ? 2 : 1;            // y-split (96x96, 96x64, 64x96)
    static constexpr int NYS = NY / S;                              // rows of one plane part
    static constexpr int R1Z = NZ / 8, R2Z = 8;
    static constexpr int R1Y = FactY<NYS>::R1, R2Y = FactY<NYS>::R2;
    static constexpr int PART = NYS * NZ;                           // cells of one plane part
    static constexpr int pick_ppc() {
        if (S == 2) return 1;
        int p = 1;
        while (p < 16 && 2 * p * PART <= TILE_MAX_CELLS) p *= 2;
        return p;
    }
    static constexpr int PPC = pick_ppc();                          // plane parts per tile (divides NX: NX % 16 == 0)
    static constexpr int ROWS = PPC * NYS;
    static constexpr int CELLS = ROWS * NZ;
    static constexpr size_t TILE_BYTES = (size_t)CELLS * sizeof(cd);
    static constexpr int NB_FWD = 3;                                // ring depth of tile_fwd
    static constexpr size_t SMEM_FWD = TILE_HEADER_FWD + NB_FWD * TILE_BYTES;
    static constexpr size_t SMEM_INV = SMEM_FWD;                       // tile_inv: the same ring of three tiles
    // work items of the four stages
    static constexpr int I_ZA = ROWS * 8, I_ZB = ROWS * R1Z, I_YA = PPC * NZ * R2Y, I_YB = PPC * NZ * R1Y;
    static constexpr int cost(int t) {
        return tile_round_up(I_ZA, t) + tile_round_up(I_ZB, t) + tile_round_up(I_YA, t) + tile_round_up(I_YB, t);
    }
    static constexpr int pick_t() {
        int best = 256;
        const int cand[5] = {256, 320, 384, 448, 512};
        for (int i = 0; i < 5; ++i)
            if (cost(cand[i]) <= cost(best)) best = cand[i];
        return best;
    }
#ifdef TDH_TILE_THREADS
    static constexpr int T = TDH_TILE_THREADS;
#else
    static constexpr int T = pick_t();
#endif
    static_assert(NZ % 16 == 0 && T % 8 == 0, "z stage mapping");
    static_assert(PART % 64 == 0, "plane parts must keep the 1024-byte swizzle phase");
    static_assert(CELLS <= TILE_MAX_CELLS, "tile too large");
    static_assert(TILE_TW_OFF + (NY + NZ) * sizeof(cd) <= TILE_HEADER_FWD, "twiddle tables must fit in the header");
};

// cell (in complex values) of position p of 128-byte line ln in a swizzled tile buffer
__device__ __forceinline__ int swz(int ln, int p) { return 8 * ln + (p ^ (ln & 7)); }

// named barrier of one warp group (ids 1, 2; id 0 is __syncthreads)
template <int NTHREADS>
__device__ __forceinline__ void group_sync(int grp) {
    asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "n"(NTHREADS) : "memory");
}

// armed[b] of the tile ring (see ARMED FLAGS at tile_fwd_kernel): set by the thread that armed full[b] for tile k ...
__device__ __forceinline__ void ring_set_armed(volatile int* armed, int b, int k) {
    __threadfence_block();                      // the mbarrier arrival before the flag
    armed[b] = k;
}
// ... and awaited by every thread that is about to wait on the parity of tile k
__device__ __forceinline__ void ring_wait_armed(const volatile int* armed, int b, int k) {
    while (armed[b] < k) {}
    __threadfence_block();                      // the flag before the mbarrier wait
}
constexpr int TILE_ARMED_OFF = 32;             // byte offset of armed[3] in the header (full[3] occupies bytes 0..23)

// Slab decomposition (Fig. 6): with the grid split over `world` ranks, a rank holds the planes
// x0 .. x0 + nx_local - 1 of every state in real space and the rows y0 .. y0 + ny_local - 1 (work-layout order) of ALL
// planes in Fourier space.  The redistribution between the two ("all-to-all") is fused into the stores of the producing
// kernels: tile_fwd writes every spectrum row straight into the Fourier-space slab buffer of the rank that owns it
// (fs[q] is that rank's buffer [state][NX][ny_local][NZ]: a peer pointer over NVLink, or another buffer of the same
// device when the ranks are emulated on one GPU).
constexpr int SLAB_MAX_WORLD = 8;
struct SlabDst {
    cd* fs[SLAB_MAX_WORLD];
    int ny_local;           // rows per rank, NY / world (even)
    int nx_local;           // planes per state on this rank, NX / world
    int nx_total;           // NX
    int x0;                 // first plane of this rank
};

// ------------------------------------------------------------------------------------------------------------
// forward: `map_in` describes the input block, `out` is the work block (same geometry, digit-permuted spectrum).
// Persistent grid; ntiles = nst * NX * S / PPC.
//
// WARP GROUPS.  The CTA is two independent groups of TG = T/2 threads that share the ring of NB = 3 tile buffers: the
// CTA's k-th tile (tile blockIdx.x + k*gridDim.x) lives in buffer k % 3 and is transformed by group k % 2, whose thread 0
// refills the buffer with tile k + 3 when the group is done with it.  The groups only meet at the mbarriers of the
// ring, so while one group sits in a shared-memory-bound or store-bound stage the other one keeps the FP64 pipe busy.
//
// ARMED FLAGS.  Buffer b is filled with tile k + 3 by the group that consumed tile k, but tile k + 3 is consumed by the
// OTHER group, and an mbarrier wait carries one bit of phase.  A group that runs two tiles ahead of the other one
// (a slow TMA load on one side is enough) would reach its wait for tile k + 6 while the barrier is still in tile k + 3's
// phase, whose parity says "tile k's phase is complete": the wait would pass at once, the group would transform a
// buffer that is being loaded or worked on, and would then arm the barrier a second time in one phase.  So every
// buffer has a flag armed[b] = the last k whose load was armed on full[b] (written after the arrival that opens
// the phase), and a group spins on armed[b] >= k before it waits on the parity of tile k: from then on the barrier is
// in tile k's phase and the parity is unambiguous.  The spin cannot deadlock: the flag for tile k is set by the group
// that finished tile k - 3, which only needed flags of earlier tiles.
// ------------------------------------------------------------------------------------------------------------
template <int NY, int NZ, bool SLAB>
__global__ void __launch_bounds__(TileCfg<NY, NZ>::T, 1)
tile_fwd_kernel(const __grid_constant__ CUtensorMap map_in, cd* __restrict__ out, int ntiles,
                const cd* __restrict__ tw_y, const cd* __restrict__ tw_z, const SlabDst slab)
{
    using C = TileCfg<NY, NZ>;
    constexpr int S = C::S, NYS = C::NYS, R1Z = C::R1Z, R1Y = C::R1Y, R2Y = C::R2Y, T = C::T, NB = C::NB_FWD;
    constexpr int TG = T / 2;
    static_assert(NB == 3 && TG % 32 == 0, "ring of three buffers shared by two warp groups");
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);
    volatile int* armed = reinterpret_cast<volatile int*>(smem_raw + TILE_ARMED_OFF);
    cd* stw_z = reinterpret_cast<cd*>(smem_raw + TILE_TW_OFF);          // [k1][j2] = e^{+2 pi i k1 j2 / NZ}: a quarter-warp
                                                                        // reads 8 consecutive entries (no bank conflict)
    cd* stw_y = stw_z + NZ;                                             // e^{+2 pi i m / NY}
    cd* ring = reinterpret_cast<cd*>(smem_raw + TILE_HEADER_FWD);
    const int grp = threadIdx.x / TG, tid = threadIdx.x % TG;           // tid: index inside the group

    uint64_t pol = policy_evict_first();
    if (threadIdx.x == 0) {
        tma_prefetch_desc(&map_in);
        for (int b = 0; b < NB; ++b) { mbar_init(full + b, 1); armed[b] = -1; }
        mbar_fence_init();
    }
    for (int i = threadIdx.x; i < NZ; i += T) stw_z[i] = ldg_cd(tw_z + (i >> 3) * (i & 7));   // [k1][j2]: w^(k1*j2)
    for (int i = threadIdx.x; i < NY; i += T) stw_y[i] = ldg_cd(tw_y + i);
    __syncthreads();
    auto issue = [&](int k) {                            // one thread; tile k of this CTA into buffer k % NB
        const int t = blockIdx.x + k * gridDim.x;
        if (t >= ntiles) return;
        const int b = k % NB;
        const int part0 = t * C::PPC, plane = part0 / S, r = part0 % S;
        mbar_arrive_expect_tx(full + b, (uint32_t)C::TILE_BYTES);
        ring_set_armed(armed, b, k);
        tma_load_4d(ring + (size_t)b * C::CELLS, &map_in, full + b, 0, r * R1Z, 0, plane, pol);
    };
    if (threadIdx.x == 0)
        for (int k = 0; k < NB; ++k) issue(k);

    for (int k = grp;; k += 2) {
        const int t = blockIdx.x + k * gridDim.x;
        if (t >= ntiles) break;
        const int b = k % NB;
        cd* sm = ring + (size_t)b * C::CELLS;
        const int part0 = t * C::PPC;
        ring_wait_armed(armed, b, k);
        mbar_wait(full + b, (uint32_t)(k / NB) & 1u);

        // ---- z stage A, in place: radix R1Z over j1 (lines lr*R1Z + j1, position j2), twiddle w^(k1*j2)
        {
            const int j2 = tid & 7;
            for (int lr = tid >> 3; lr < C::ROWS; lr += TG / 8) {
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
        group_sync<TG>(grp);
        // ---- z stage B, in place inside line g: position k2 then holds kz = k1 + R1Z*k2
        for (int g = tid; g < C::I_ZB; g += TG) {
            cd* p = sm + 8 * g;
            const int s = g & 7;
            cd v[8];
#pragma unroll
            for (int j2 = 0; j2 < 8; ++j2) v[j2] = p[j2 ^ s];
            Dft<8, -1>::run(v);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) p[k2 ^ s] = v[k2];
        }
        group_sync<TG>(grp);
        // ---- y stage A, in place: rows j1*R2Y + j2 of column c = (k1, k2) -> rows k1y*R2Y + j2
        for (int item = tid; item < C::I_YA; item += TG) {
            const int c = item % NZ, rr = item / NZ, j2 = rr % R2Y, lp = rr / R2Y;
            const int k1 = c >> 3, k2 = c & 7;
            const int row0 = lp * NYS + j2;
            cd x[R1Y];
#pragma unroll
            for (int j1 = 0; j1 < R1Y; ++j1) x[j1] = sm[swz((row0 + j1 * R2Y) * R1Z + k1, k2)];
            Dft<R1Y, -1>::run(x);
            sm[swz(row0 * R1Z + k1, k2)] = x[0];
#pragma unroll
            for (int k1y = 1; k1y < R1Y; ++k1y)
                sm[swz((row0 + k1y * R2Y) * R1Z + k1, k2)] = cmulc(x[k1y], stw_y[S * k1y * j2]);
        }
        group_sync<TG>(grp);
        // ---- y stage B -> global at the in-place position: row rho = k1y*R2Y + k2y (plane row S*rho + r), column c
        for (int item = tid; item < C::I_YB; item += TG) {
            const int c = item % NZ, rr = item / NZ, k1y = rr % R1Y, lp = rr / R1Y;
            const int k1 = c >> 3, k2 = c & 7;
            const int row0 = lp * NYS + k1y * R2Y;
            cd res[R2Y];
#pragma unroll
            for (int j2 = 0; j2 < R2Y; ++j2) res[j2] = sm[swz((row0 + j2) * R1Z + k1, k2)];
            Dft<R2Y, -1>::run(res);
            const int part = part0 + lp, plane = part / S, r = part % S;
            if (SLAB) {
                // row Y of plane (st, x0 + xl) belongs to rank q = Y / ny_local: local row Y - q * ny_local of its slab
                const int st = plane / slab.nx_local, xl = plane - st * slab.nx_local;
                const size_t prow = ((size_t)st * slab.nx_total + slab.x0 + xl) * slab.ny_local;
#pragma unroll
                for (int k2y = 0; k2y < R2Y; ++k2y) {
                    const int Y = S * (k1y * R2Y + k2y) + r;
                    const int q = Y / slab.ny_local;
                    sts_cd(slab.fs[q] + (prow + (Y - q * slab.ny_local)) * NZ + c, res[k2y]);
                }
            } else {
                cd* dst = out + (size_t)plane * NY * NZ + (size_t)(S * (k1y * R2Y) + r) * NZ + c;
#pragma unroll
                for (int k2y = 0; k2y < R2Y; ++k2y) sts_cd(dst + (size_t)(S * k2y) * NZ, res[k2y]);
            }
        }
        // every read of this buffer is done: hand it back to the TMA
        fence_proxy_async();
        group_sync<TG>(grp);
        if (tid == 0) issue(k + NB);
    }
}

// Arguments of the fused epilogue of tile_inv.
struct Epilogue {
    const double* v;        // V(r), n0*n1*n2; NULL: no local term (then phi is not read, unless nl_off != NULL)
    const cd* phi;          // input block of this Hamiltonian application (read with V and with projectors)
    const cd* yv;           // optional addend y (same block layout as out); NULL: none
    cd alpha;               // out = alpha * (T + V + Vnl) phi + y
    int nx;                 // planes per state
    // Kleinman-Bylander back-projection (second half of Eq. 9), as per-tile record lists; nl_off == NULL: none.
    // Tile (x, r) owns records nl_off[(x*S + r)*(nl_layers+1) + l] .. [.. + l + 1) of layer l; within one layer every
    // grid point appears at most once, so the shared-memory read-modify-write needs no atomics.  With projectors, v must
    // not be NULL (the handle passes its zero-filled potential when none was set).
    const int* nl_off;
    int nl_layers;
    const unsigned* nl_cc;  // per record: swizzled cell inside the plane part | first channel << 16
    const double* nl_beta;  // [cmax][nrec] projector values, zero padded above the atom's channel count
    const cd* nl_phase;     // per record e^{+ik.d}; NULL at Gamma
    const cd* dpi;          // [state][nchan_tot] D * dV * <beta|phi>  (+ cmax zeroed entries of padding)
    int nrec;
    int cmax;               // padded channel count of a record: 1, 4, 9 or 16 (nl_pad_cmax) = the kernel's CM
    int nchan_tot;
};

// channel counts the record loop is compiled for; the host pads nl_beta (zeros) and dpi (zeros) to this
__host__ __device__ constexpr int nl_pad_cmax(int c) { return c <= 1 ? 1 : (c <= 4 ? 4 : (c <= 9 ? 9 : 16)); }
// index of a padded channel count in the table of tile_inv instantiations (0: no projectors)
__host__ __device__ constexpr int nl_cm_index(int cm) { return cm == 0 ? 0 : (cm == 1 ? 1 : (cm == 4 ? 2 : (cm == 9 ? 3 : 4))); }
constexpr int NL_NCM = 5;
// records of one thread in flight together
template <int CM> struct NlUnroll { static constexpr int U = CM <= 1 ? 8 : (CM <= 4 ? 6 : (CM <= 9 ? 3 : 2)); };

// One layer of the back-projection of one plane part: records [i0, i1) add  e^{-ik.d} sum_c beta_c[i] * dpi[chan0 + c]
// into cell (cc & 0xffff) of `base`.  U records per thread are in flight together: the loop is bound by the latency of
// the record loads (L2), not by arithmetic.  dp points at dpi of this state (global memory; the few hundred bytes a
// tile touches stay in L1).
template <int CM, int U>
__device__ __forceinline__ void nl_scatter_layer(cd* base, const cd* __restrict__ dp, const unsigned* __restrict__ nl_cc,
                                                 const double* __restrict__ nl_beta, const cd* __restrict__ nl_phase,
                                                 size_t nrec, int i0, int i1, int tid, int nthreads)
{
    for (int ib = i0 + tid; ib < i1; ib += U * nthreads) {
        unsigned cc[U];
        double bv[U][CM > 0 ? CM : 1];
        cd ph[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = ib + u * nthreads;
            const bool ok = i < i1;
            cc[u] = ok ? __ldg(nl_cc + i) : 0u;
#pragma unroll
            for (int c = 0; c < CM; ++c) bv[u][c] = ok ? __ldg(nl_beta + (size_t)c * nrec + i) : 0.0;
            if (nl_phase != nullptr) ph[u] = ok ? __ldg(nl_phase + i) : make_double2(1.0, 0.0);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (ib + u * nthreads < i1) {
                const cd* d = dp + (cc[u] >> 16);
                cd sacc = make_double2(0.0, 0.0);
#pragma unroll
                for (int c = 0; c < CM; ++c) {
                    const cd dv = ldg_cd(d + c);
                    sacc.x = fma(bv[u][c], dv.x, sacc.x);
                    sacc.y = fma(bv[u][c], dv.y, sacc.y);
                }
                if (nl_phase != nullptr) sacc = cmulc(sacc, ph[u]);
                cd* cell = base + (cc[u] & 0xffffu);
                *cell = cadd(*cell, sacc);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// inverse + epilogue: `map_spec` describes the work block (digit-permuted spectrum), `out` the output block; `map_phi`
// and `map_yv` describe the input block ep.phi of this Hamiltonian application and the addend block ep.yv (same
// geometry) and are only used to start their tiles towards L2 when a tile's turn begins -- the epilogue reads both
// straight from global memory.  CM = padded channel count of the projector records (0: no projectors; ep.cmax == CM).
// Persistent grid; ntiles = nst * NX * S / PPC.
//
// WARP GROUPS as in tile_fwd: two groups of TG = T/2 threads, a ring of three spectrum buffers, the CTA's k-th tile in
// buffer k % 3 handled by group k % 2.  Per tile: inverse y (two stages), inverse z (two stages), then
//   without projectors: the last z stage ends in registers, out = alpha * (x + V phi) + y goes straight to global;
//   with projectors:    the last z stage is written back in place (natural order), the record lists add V_nl phi into
//                       the tile layer by layer, and a final pass forms out = alpha * (tile + V phi) + y.
// A stage of one group that waits on L2 (records, phi, V, y) or on the store queue overlaps with the other group's
// butterflies.
// ------------------------------------------------------------------------------------------------------------
template <int NY, int NZ, int CM>
__global__ void __launch_bounds__(TileCfg<NY, NZ>::T, 1)
tile_inv_kernel(const __grid_constant__ CUtensorMap map_spec, const __grid_constant__ CUtensorMap map_phi,
                const __grid_constant__ CUtensorMap map_yv, cd* __restrict__ out, int ntiles,
                const cd* __restrict__ tw_y, const cd* __restrict__ tw_z, const Epilogue ep)
{
    using C = TileCfg<NY, NZ>;
    constexpr int S = C::S, NYS = C::NYS, R1Z = C::R1Z, R1Y = C::R1Y, R2Y = C::R2Y, T = C::T, NB = C::NB_FWD;
    constexpr int TG = T / 2;
    constexpr bool HAVE_NL = CM > 0;
    static_assert(NB == 3 && TG % 32 == 0, "ring of three buffers shared by two warp groups");
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);
    volatile int* armed = reinterpret_cast<volatile int*>(smem_raw + TILE_ARMED_OFF);
    cd* stw_z = reinterpret_cast<cd*>(smem_raw + TILE_TW_OFF);          // [k1][j2] = e^{+2 pi i k1 j2 / NZ}: a quarter-warp
                                                                        // reads 8 consecutive entries (no bank conflict)
    cd* stw_y = stw_z + NZ;                                             // e^{+2 pi i m / NY}
    cd* ring = reinterpret_cast<cd*>(smem_raw + TILE_HEADER_FWD);
    const int grp = threadIdx.x / TG, tid = threadIdx.x % TG;           // tid: index inside the group
    const bool have_v = HAVE_NL || ep.v != nullptr;

    uint64_t pol = policy_evict_first();
    if (threadIdx.x == 0) {
        tma_prefetch_desc(&map_spec);
        if (have_v) tma_prefetch_desc(&map_phi);
        if (ep.yv != nullptr) tma_prefetch_desc(&map_yv);
        for (int b = 0; b < NB; ++b) { mbar_init(full + b, 1); armed[b] = -1; }
        mbar_fence_init();
    }
    for (int i = threadIdx.x; i < NZ; i += T) stw_z[i] = ldg_cd(tw_z + (i >> 3) * (i & 7));   // [k1][j2]: w^(k1*j2)
    for (int i = threadIdx.x; i < NY; i += T) stw_y[i] = ldg_cd(tw_y + i);
    __syncthreads();
    auto issue = [&](int k) {                            // one thread; tile k of this CTA into buffer k % NB
        const int t = blockIdx.x + k * gridDim.x;
        if (t >= ntiles) return;
        const int b = k % NB;
        const int part0 = t * C::PPC, plane = part0 / S, r = part0 % S;
        mbar_arrive_expect_tx(full + b, (uint32_t)C::TILE_BYTES);
        ring_set_armed(armed, b, k);
        tma_load_4d(ring + (size_t)b * C::CELLS, &map_spec, full + b, 0, r * R1Z, 0, plane, pol);
    };
    if (threadIdx.x == 0)
        for (int k = 0; k < NB; ++k) issue(k);
    for (int k = grp;; k += 2) {
        const int t = blockIdx.x + k * gridDim.x;
        if (t >= ntiles) break;
        const int b = k % NB;
        cd* sm = ring + (size_t)b * C::CELLS;
        const int part0 = t * C::PPC;
        // the tiles of phi and of the addend that the epilogue will read: start them towards L2 now
        if (tid == 0) {
            if (have_v) tma_prefetch_l2_4d(&map_phi, 0, (part0 % S) * R1Z, 0, part0 / S);
            if (ep.yv != nullptr) tma_prefetch_l2_4d(&map_yv, 0, (part0 % S) * R1Z, 0, part0 / S);
        }
        ring_wait_armed(armed, b, k);
        mbar_wait(full + b, (uint32_t)(k / NB) & 1u);

        // ---- y stage A', in place: rows k1y*R2Y + k2y (contiguous) hold k = k1y + R1Y*k2y; radix R2Y over k2y -> j2,
        //      twiddle w^(-j2*k1y)
        for (int item = tid; item < C::I_YB; item += TG) {
            const int c = item % NZ, rr = item / NZ, k1y = rr % R1Y, lp = rr / R1Y;
            const int k1 = c >> 3, k2 = c & 7;
            const int row0 = lp * NYS + k1y * R2Y;
            cd v[R2Y];
#pragma unroll
            for (int k2y = 0; k2y < R2Y; ++k2y) v[k2y] = sm[swz((row0 + k2y) * R1Z + k1, k2)];
            Dft<R2Y, +1>::run(v);
            sm[swz(row0 * R1Z + k1, k2)] = v[0];
#pragma unroll
            for (int j2 = 1; j2 < R2Y; ++j2) sm[swz((row0 + j2) * R1Z + k1, k2)] = cmul(v[j2], stw_y[S * j2 * k1y]);
        }
        group_sync<TG>(grp);
        // ---- y stage B', in place: rows k1y*R2Y + j2, radix R1Y over k1y -> j1: row j1*R2Y + j2 = m, y = S*m + r
        for (int item = tid; item < C::I_YA; item += TG) {
            const int c = item % NZ, rr = item / NZ, j2 = rr % R2Y, lp = rr / R2Y;
            const int k1 = c >> 3, k2 = c & 7;
            const int row0 = lp * NYS + j2;
            cd x[R1Y];
#pragma unroll
            for (int k1y = 0; k1y < R1Y; ++k1y) x[k1y] = sm[swz((row0 + k1y * R2Y) * R1Z + k1, k2)];
            Dft<R1Y, +1>::run(x);
#pragma unroll
            for (int j1 = 0; j1 < R1Y; ++j1) sm[swz((row0 + j1 * R2Y) * R1Z + k1, k2)] = x[j1];
        }
        group_sync<TG>(grp);
        // ---- z stage A', in place inside line g = (row, k1): positions k2 hold kz = k1 + R1Z*k2; radix 8 -> j2
        for (int g = tid; g < C::I_ZB; g += TG) {
            cd* p = sm + 8 * g;
            const int s = g & 7;
            cd v[8];
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) v[k2] = p[k2 ^ s];
            Dft<8, +1>::run(v);
#pragma unroll
            for (int j2 = 0; j2 < 8; ++j2) p[j2 ^ s] = v[j2];
        }
        group_sync<TG>(grp);
        const int j2 = tid & 7;
        if (HAVE_NL) {
            // ---- z stage B', in place: thread (row lr, j2): twiddle w^(-k1*j2), radix R1Z over k1 -> cell (lr, 8*j1 + j2)
            for (int lr = tid >> 3; lr < C::ROWS; lr += TG / 8) {
                const int l0 = lr * R1Z;
                cd x[R1Z];
                x[0] = sm[swz(l0, j2)];
#pragma unroll
                for (int k1 = 1; k1 < R1Z; ++k1) x[k1] = cmul(sm[swz(l0 + k1, j2)], stw_z[8 * k1 + j2]);
                Dft<R1Z, +1>::run(x);
#pragma unroll
                for (int j1 = 0; j1 < R1Z; ++j1) sm[swz(l0 + j1, j2)] = x[j1];
            }
            group_sync<TG>(grp);
            // ---- back-projection: the tile now holds T phi in natural order; add V_nl phi layer by layer
            const int st = (part0 / S) / ep.nx;                           // PPC divides NX: one state per tile
            const cd* dp = ep.dpi + (size_t)st * ep.nchan_tot;
            for (int layer = 0; layer < ep.nl_layers; ++layer) {
#pragma unroll
                for (int lp = 0; lp < C::PPC; ++lp) {
                    const int part = part0 + lp, plane = part / S, r = part % S;
                    const int x = plane % ep.nx;
                    const int* off = ep.nl_off + (size_t)(x * S + r) * (ep.nl_layers + 1) + layer;
                    nl_scatter_layer<CM, NlUnroll<CM>::U>(sm + lp * C::PART, dp, ep.nl_cc, ep.nl_beta, ep.nl_phase,
                                                          (size_t)ep.nrec, __ldg(off), __ldg(off + 1), tid, TG);
                }
                group_sync<TG>(grp);
            }
        }
        // ---- epilogue, thread (row lr, j2), cells z = 8*j1 + j2:  out = alpha * (T phi [+ V_nl phi] + V phi) + y.
        //      phi, V and y come straight from global memory (their tiles were started towards L2 above); all their
        //      loads are issued before the first store because out may alias y.
        for (int lr = tid >> 3; lr < C::ROWS; lr += TG / 8) {
            const int l0 = lr * R1Z;
            const int lp = lr / NYS, m = lr % NYS;
            const int part = part0 + lp, plane = part / S, r = part % S;
            const int y = S * m + r;
            const size_t gi = (size_t)plane * NY * NZ + (size_t)y * NZ + j2;               // index in the block
            double vv[R1Z];
            cd ph[R1Z];
            if (have_v) {
                const double* vrow = ep.v + ((size_t)(plane % ep.nx) * NY + y) * NZ + j2;
#pragma unroll
                for (int j1 = 0; j1 < R1Z; ++j1) {
                    vv[j1] = __ldg(vrow + 8 * j1);
                    ph[j1] = lds_cd(ep.phi + gi + 8 * j1);
                }
            }
            cd x[R1Z];
            if (HAVE_NL) {
#pragma unroll
                for (int j1 = 0; j1 < R1Z; ++j1) x[j1] = sm[swz(l0 + j1, j2)];
            } else {
                x[0] = sm[swz(l0, j2)];
#pragma unroll
                for (int k1 = 1; k1 < R1Z; ++k1) x[k1] = cmul(sm[swz(l0 + k1, j2)], stw_z[8 * k1 + j2]);   // w_NZ^(-k1*j2)
                Dft<R1Z, +1>::run(x);
            }
            if (have_v) {
#pragma unroll
                for (int j1 = 0; j1 < R1Z; ++j1) {
                    x[j1].x = fma(vv[j1], ph[j1].x, x[j1].x);
                    x[j1].y = fma(vv[j1], ph[j1].y, x[j1].y);
                }
            }
            if (ep.yv != nullptr) {
                cd ya[R1Z];
#pragma unroll
                for (int j1 = 0; j1 < R1Z; ++j1) ya[j1] = lds_cd(ep.yv + gi + 8 * j1);
#pragma unroll
                for (int j1 = 0; j1 < R1Z; ++j1) sts_cd(out + gi + 8 * j1, cadd(cmul(ep.alpha, x[j1]), ya[j1]));
            } else {
#pragma unroll
                for (int j1 = 0; j1 < R1Z; ++j1) sts_cd(out + gi + 8 * j1, cmul(ep.alpha, x[j1]));
            }
        }
        // every read of this buffer is done: hand it back to the TMA
        fence_proxy_async();
        group_sync<TG>(grp);
        if (tid == 0) issue(k + NB);
    }
}

}  // namespace tdh
