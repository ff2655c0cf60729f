// nl_kernels.cuh -- Kleinman-Bylander projection (first half of Eq. 9) on FP64 tensor cores.
//
// For atom I and state s:   dpi[s][c] = D_{I,c} dV sum_q beta_{I,c}[q] e^{+ik.d_q} psi_s[S_I[q]]
// This is a real (C_I x P_I) matrix times a complex (P_I x n_st) block, gathered from the sphere's grid points.
// A CTA owns one atom and 8 states; its NLP_WARPS warps split the sphere's points in blocks of 32.  Per block a lane
// issues 8 independent 16-byte gathers (8 k-steps of 4 points), then for each tile of 8 channels
//     mma.sync.m8n8k4.f64   D(8 chan x 8 states) += A(8 chan x 4 points) * B(4 points x 8 states)
// twice per k-step (real and imaginary parts of psi).  Fragment layout of m8n8k4 (PTX ISA): lane l holds A[l/4][l%4],
// B[l%4][l/4] and C[l/4][2*(l%4) + {0,1}].  So lane l gathers ONE complex value psi_{s0 + l/4}[S[q0 + l%4]] per k-step
// and that is both B fragments.  The partial sums of the warps are combined through shared memory in warp order:
// deterministic, no atomics.  The second half of Eq. 9 (back-projection) is nl_scatter_kernel below, or, on whole-plane
// tiles, the record lists inside tile_inv (tile_kernels.cuh).  The indices and projector values of the next block are
// requested while the gathers of the current one are in flight.
#pragma once
#include "fft_codelets.cuh"

namespace tdh {

struct AtomDesc {
    int q0;      // first entry in the (sorted) sphere arrays
    int np;      // P_I
    int boff;    // offset of beta_{I,0}[0]; channel c at boff + c*np
    int chan0;   // first channel in the global channel list
    int nchan;   // C_I
    int sc0;     // first chunk of the atom in the chunk table of nl_scatter_bulk_kernel
    int scn;     // number of chunks
};

__device__ __forceinline__ void dmma_m8n8k4(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c[0]), "+d"(c[1])
                 : "d"(a), "d"(b));
}

constexpr int NLP_WARPS = 8;     // warps per CTA, splitting the sphere
constexpr int NLP_STATES = 8;    // states per CTA (the N of the MMA)
constexpr int NLP_KSTEPS = 8;    // k-steps (of 4 points) per block: 32 points, 8 gathers in flight per lane

// grid: (ceil(nst / 8), natoms) -- the state groups of one atom are neighbours in launch order, run together and share
// the atom's index and projector tables through L2; MT = number of 8-channel tiles (C_I <= 8*MT)
template <int MT>
__global__ void __launch_bounds__(32 * NLP_WARPS)
nl_project_kernel(const cd* __restrict__ psi, size_t npts, int nst, const AtomDesc* __restrict__ atoms,
                  const int* __restrict__ sidx, const double* __restrict__ sbeta, const cd* __restrict__ sphase,
                  const double* __restrict__ dscale, cd* __restrict__ dpi, int nchan_tot)
{
    constexpr int KS = MT == 1 ? NLP_KSTEPS : NLP_KSTEPS / 2;   // two channel tiles: half the k-steps in flight (registers)
    __shared__ double part[NLP_WARPS][MT][4][32];
    const AtomDesc at = atoms[blockIdx.x];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kq = lane & 3, r8 = lane >> 2;
    const int s0 = blockIdx.y * NLP_STATES;
    const int s = s0 + r8;                                      // this lane's state (B fragment column)
    const bool s_ok = s < nst;
    const cd* ps = psi + (size_t)(s_ok ? s : 0) * npts;
    const int* idx = sidx + at.q0;
    const cd* phs = sphase ? sphase + at.q0 : nullptr;

    double cre[MT][2], cim[MT][2];
#pragma unroll
    for (int m = 0; m < MT; ++m) cre[m][0] = cre[m][1] = cim[m][0] = cim[m][1] = 0.0;

    // Software pipeline over the warp's blocks of 32 points: the sphere indices and the projector values (A fragments)
    // of block i+1 are requested while the gathers of block i are in flight, so a block costs one DRAM round trip
    // instead of three dependent ones (index -> psi, beta).
    constexpr int STRIDE = NLP_WARPS * 4 * KS;
    int ix[KS];
    double af[KS][MT];
    auto load_meta = [&](int q0, int (&ixo)[KS], double (&afo)[KS][MT]) {
#pragma unroll
        for (int u = 0; u < KS; ++u) {
            const int q = q0 + 4 * u + kq;
            const bool q_ok = q < at.np;
            ixo[u] = q_ok ? __ldg(idx + q) : -1;
#pragma unroll
            for (int m = 0; m < MT; ++m) {
                const int c = 8 * m + r8;                                   // A fragment row = channel
                afo[u][m] = (q_ok && c < at.nchan) ? __ldg(sbeta + at.boff + (size_t)c * at.np + q) : 0.0;
            }
        }
    };
    int q0 = warp * 4 * KS;
    if (q0 < at.np) load_meta(q0, ix, af);
    for (; q0 < at.np; q0 += STRIDE) {
        cd b[KS];
#pragma unroll
        for (int u = 0; u < KS; ++u) {
            b[u] = make_double2(0.0, 0.0);
            if (ix[u] >= 0 && s_ok) b[u] = __ldcs(ps + ix[u]);
        }
        int ixn[KS];
        double afn[KS][MT];
        if (q0 + STRIDE < at.np) load_meta(q0 + STRIDE, ixn, afn);
#pragma unroll
        for (int u = 0; u < KS; ++u) {
            cd bv = b[u];
            if (phs != nullptr && ix[u] >= 0) bv = cmul(bv, __ldg(phs + q0 + 4 * u + kq));
#pragma unroll
            for (int m = 0; m < MT; ++m) {
                dmma_m8n8k4(cre[m], af[u][m], bv.x);
                dmma_m8n8k4(cim[m], af[u][m], bv.y);
            }
        }
#pragma unroll
        for (int u = 0; u < KS; ++u) {
            ix[u] = ixn[u];
#pragma unroll
            for (int m = 0; m < MT; ++m) af[u][m] = afn[u][m];
        }
    }
#pragma unroll
    for (int m = 0; m < MT; ++m) {
        part[warp][m][0][lane] = cre[m][0];
        part[warp][m][1][lane] = cre[m][1];
        part[warp][m][2][lane] = cim[m][0];
        part[warp][m][3][lane] = cim[m][1];
    }
    __syncthreads();
    // C fragment: row = channel 8m + lane/4, columns = states 2*(lane%4) + {0,1}.  Warp m < MT sums tile m.
    if (warp < MT) {
        const int m = warp;
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        for (int w = 0; w < NLP_WARPS; ++w)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[j] += part[w][m][j][lane];
        const int c = 8 * m + r8;
        if (c < at.nchan) {
            const double d = __ldg(dscale + at.chan0 + c);
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int so = s0 + 2 * kq + j;
                if (so < nst) dpi[(size_t)so * nchan_tot + at.chan0 + c] = make_double2(d * acc[j], d * acc[2 + j]);
            }
        }
    }
}


// ------------------------------------------------------------------------------------------------------------
// Back-projection (second half of Eq. 9):   out_s[S_I[q]] += alpha e^{-ik.d_q} sum_c beta_{I,c}[q] dpi[s][c]
// The mirror image of the projection: a real (P_I x C_I) matrix times the complex (C_I x n_st) coefficients, added
// into the sphere's grid points of the output block.  A CTA owns one atom and 8 states, its warps split the sphere in
// blocks of 8 points; per block and per tile of 4 channels
//     mma.sync.m8n8k4.f64   D(8 points x 8 states) += A(8 points x 4 chan) * B(4 chan x 8 states)
// twice (real and imaginary parts of dpi; B is loop invariant and stays in registers).  Lane l then holds the sums of
// point q0 + l/4 for the two states s0 + 2*(l%4) + {0,1} and read-modify-writes those two values: for one state the 8
// lanes l/4 = 0..7 touch 8 consecutive sphere points = up to 128 contiguous bytes (a sphere is z-runs of grid points).
// NLS_BLOCKS blocks are in flight per warp, and the indices / projector values of the next iteration are requested
// while this iteration's loads travel (one DRAM round trip per iteration).
// ATOMIC FREE: one launch covers a set of atoms whose spheres share no grid point (the host colours the atoms), a
// point appears once per sphere, CTAs of one atom own different states -- plain loads and stores, deterministic.
// ------------------------------------------------------------------------------------------------------------
constexpr int NLS_WARPS = 8;
constexpr int NLS_BLOCKS = 4;

// grid: (ceil(nst / 8), atoms of this colour); KT = number of 4-channel tiles (C_I <= 4*KT)
template <int KT>
__global__ void __launch_bounds__(32 * NLS_WARPS)
nl_scatter_kernel(cd* __restrict__ out, size_t npts, int nst, const AtomDesc* __restrict__ atoms,
                  const int* __restrict__ sidx, const double* __restrict__ sbeta, const cd* __restrict__ sphase,
                  const cd* __restrict__ dpi, int nchan_tot, cd alpha)
{
    const AtomDesc at = atoms[blockIdx.x];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kq = lane & 3, r8 = lane >> 2;
    const int s0 = blockIdx.y * NLP_STATES;
    // B fragments: B[k = kq][n = r8] = alpha * dpi[s0 + r8][chan0 + 4*kt + kq]
    double bre[KT], bim[KT];
#pragma unroll
    for (int kt = 0; kt < KT; ++kt) {
        const int c = 4 * kt + kq, s = s0 + r8;
        cd v = make_double2(0.0, 0.0);
        if (c < at.nchan && s < nst) v = cmul(alpha, __ldg(dpi + (size_t)s * nchan_tot + at.chan0 + c));
        bre[kt] = v.x;
        bim[kt] = v.y;
    }
    // C fragment: row = point q0 + 8u + r8, columns = states sa, sa + 1
    const int sa = s0 + 2 * kq;
    const bool ok0 = sa < nst, ok1 = sa + 1 < nst;
    cd* o0 = out + (size_t)(ok0 ? sa : 0) * npts;
    cd* o1 = out + (size_t)(ok1 ? sa + 1 : 0) * npts;
    const int* idx = sidx + at.q0;
    const cd* phs = sphase ? sphase + at.q0 : nullptr;

    constexpr int STRIDE = NLS_WARPS * 8 * NLS_BLOCKS;
    int ix[NLS_BLOCKS];
    double af[NLS_BLOCKS][KT];
    auto load_meta = [&](int q0, int (&ixo)[NLS_BLOCKS], double (&afo)[NLS_BLOCKS][KT]) {
#pragma unroll
        for (int u = 0; u < NLS_BLOCKS; ++u) {
            const int q = q0 + 8 * u + r8;
            const bool q_ok = q < at.np;
            ixo[u] = q_ok ? __ldg(idx + q) : -1;
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) {
                const int c = 4 * kt + kq;                                  // A fragment column = channel
                afo[u][kt] = (q_ok && c < at.nchan) ? __ldg(sbeta + at.boff + (size_t)c * at.np + q) : 0.0;
            }
        }
    };
    int q0 = warp * 8 * NLS_BLOCKS;
    if (q0 < at.np) load_meta(q0, ix, af);
    for (; q0 < at.np; q0 += STRIDE) {
        cd v0[NLS_BLOCKS], v1[NLS_BLOCKS];
#pragma unroll
        for (int u = 0; u < NLS_BLOCKS; ++u) {
            v0[u] = v1[u] = make_double2(0.0, 0.0);
            if (ix[u] >= 0 && ok0) v0[u] = o0[ix[u]];
            if (ix[u] >= 0 && ok1) v1[u] = o1[ix[u]];
        }
        int ixn[NLS_BLOCKS];
        double afn[NLS_BLOCKS][KT];
        if (q0 + STRIDE < at.np) load_meta(q0 + STRIDE, ixn, afn);
#pragma unroll
        for (int u = 0; u < NLS_BLOCKS; ++u) {
            double cre[2] = {0.0, 0.0}, cim[2] = {0.0, 0.0};
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) {
                dmma_m8n8k4(cre, af[u][kt], bre[kt]);
                dmma_m8n8k4(cim, af[u][kt], bim[kt]);
            }
            cd a0 = make_double2(cre[0], cim[0]), a1 = make_double2(cre[1], cim[1]);
            if (phs != nullptr && ix[u] >= 0) {
                const cd ph = __ldg(phs + q0 + 8 * u + r8);
                a0 = cmulc(a0, ph);
                a1 = cmulc(a1, ph);
            }
            if (ix[u] >= 0 && ok0) o0[ix[u]] = cadd(v0[u], a0);
            if (ix[u] >= 0 && ok1) o1[ix[u]] = cadd(v1[u], a1);
        }
#pragma unroll
        for (int u = 0; u < NLS_BLOCKS; ++u) {
            ix[u] = ixn[u];
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) af[u][kt] = afn[u][kt];
        }
    }
}


// ------------------------------------------------------------------------------------------------------------
// The same back-projection with the read-modify-write done by the L2: cp.reduce.async.bulk ... .add.f64 (TMA, no tensor
// map).  nl_scatter_kernel above loads every output value, adds and stores it, and waits on those loads (ncu,
// profiles/r02_summary.md: 16 of 18 warp-cycles per issue on long_scoreboard, DRAM 56 % busy).  Here the kernel never
// reads `out`: the contributions alpha e^{-ik.d} sum_c beta_c D pi_c of a chunk of the sphere go to shared memory, laid out
// [state][point], and one bulk reduce-add per (z-run, state) adds them to the output block in the L2 -- a sphere is z-runs
// of consecutive grid points, i.e. of consecutive addresses.  Measured on B200 (Large geometry, 296 states): plain RMW
// 3.55 TB/s, bulk reduce-add 4.6 TB/s of the 32 B per point and state.
// A chunk is up to SC_RC runs / SC_MAXPTS points (longer runs are cut); two chunk buffers: the TMA reads one while the warps
// fill the other.  Rounding is that of one IEEE addition per point, as in the RMW kernel; the launches per colour keep the
// order of the additions fixed where spheres overlap.
// ------------------------------------------------------------------------------------------------------------
constexpr int SC_RC = 32;          // runs per chunk: one bulk operation per (run, state) = 256 threads
#ifndef TDH_SC_MAXPTS
#define TDH_SC_MAXPTS 352
#endif
#ifndef TDH_SC_NBUF
#define TDH_SC_NBUF 2
#endif
constexpr int SC_MAXPTS = TDH_SC_MAXPTS;     // points per chunk: two CTAs of 90 KB per SM
constexpr int SC_NBUF = TDH_SC_NBUF;
constexpr size_t SC_SMEM = (size_t)SC_NBUF * NLP_STATES * SC_MAXPTS * sizeof(cd);
struct ScRun { int p0, len, off; };         // first grid point, points, offset (points) inside the chunk
struct ScChunk { int r0, nr, q0, np; };     // first run, runs, first point in the atom's sorted list, points

__device__ __forceinline__ void bulk_reduce_add_f64(void* gdst, const void* ssrc, unsigned bytes) {
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;" ::"l"(gdst),
                 "r"((unsigned)__cvta_generic_to_shared(ssrc)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit_group() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_group_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_group() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }

// grid: (atoms of this colour, ceil(nst / 8)); KT = number of 4-channel tiles (C_I <= 4*KT)
template <int KT>
__global__ void __launch_bounds__(32 * NLS_WARPS)
nl_scatter_bulk_kernel(cd* __restrict__ out, size_t npts, int nst, const AtomDesc* __restrict__ atoms,
                       const ScRun* __restrict__ runs, const ScChunk* __restrict__ chunks, const double* __restrict__ sbeta,
                       const cd* __restrict__ sphase, const cd* __restrict__ dpi, int nchan_tot, cd alpha)
{
    extern __shared__ __align__(128) unsigned char sc_smem[];
    cd* buf = reinterpret_cast<cd*>(sc_smem);
    const AtomDesc at = atoms[blockIdx.x];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kq = lane & 3, r8 = lane >> 2;
    const int s0 = blockIdx.y * NLP_STATES;
    // B fragments: B[k = kq][n = r8] = alpha * dpi[s0 + r8][chan0 + 4*kt + kq]
    double bre[KT], bim[KT];
#pragma unroll
    for (int kt = 0; kt < KT; ++kt) {
        const int c = 4 * kt + kq, s = s0 + r8;
        cd v = make_double2(0.0, 0.0);
        if (c < at.nchan && s < nst) v = cmul(alpha, __ldg(dpi + (size_t)s * nchan_tot + at.chan0 + c));
        bre[kt] = v.x;
        bim[kt] = v.y;
    }
    const cd* phs = sphase ? sphase + at.q0 : nullptr;
    const int prun = threadIdx.x >> 3, pst = threadIdx.x & 7;       // this thread's bulk operation: (run, state) of a chunk
    cd* orow = out + (size_t)min(s0 + pst, nst - 1) * npts;
    const bool pst_ok = s0 + pst < nst;
    constexpr int U = 4;                                            // 8-point blocks of one warp in flight
    for (int c = 0; c < at.scn; ++c) {
        const ScChunk ch = chunks[at.sc0 + c];
        cd* bb = buf + (size_t)(c % SC_NBUF) * NLP_STATES * SC_MAXPTS;
        if (c >= SC_NBUF) bulk_wait_group_read<SC_NBUF - 1>();     // the TMA has read this buffer (chunk c - 2)
        __syncthreads();
        const int nblk = (ch.np + 7) >> 3;
        for (int b0 = warp; b0 < nblk; b0 += U * NLS_WARPS) {
            double af[U][KT];
            cd ph[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = 8 * (b0 + u * NLS_WARPS) + r8;        // row of the MMA: point i of the chunk
                const bool ok = i < ch.np;
#pragma unroll
                for (int kt = 0; kt < KT; ++kt) {
                    const int cc = 4 * kt + kq;                     // column of the A fragment: channel
                    af[u][kt] = (ok && cc < at.nchan) ? __ldg(sbeta + at.boff + (size_t)cc * at.np + ch.q0 + i) : 0.0;
                }
                if (phs != nullptr) ph[u] = ok ? __ldg(phs + ch.q0 + i) : make_double2(1.0, 0.0);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = 8 * (b0 + u * NLS_WARPS) + r8;
                double cre[2] = {0.0, 0.0}, cim[2] = {0.0, 0.0};
#pragma unroll
                for (int kt = 0; kt < KT; ++kt) {
                    dmma_m8n8k4(cre, af[u][kt], bre[kt]);
                    dmma_m8n8k4(cim, af[u][kt], bim[kt]);
                }
                cd a0 = make_double2(cre[0], cim[0]), a1 = make_double2(cre[1], cim[1]);
                if (phs != nullptr) {
                    a0 = cmulc(a0, ph[u]);
                    a1 = cmulc(a1, ph[u]);
                }
                if (i < ch.np) {                                    // C fragment: point i, states 2*kq and 2*kq + 1
                    bb[(size_t)(2 * kq) * SC_MAXPTS + i] = a0;
                    bb[(size_t)(2 * kq + 1) * SC_MAXPTS + i] = a1;
                }
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the generic-proxy writes above before the TMA's reads
        __syncthreads();
        if (prun < ch.nr && pst_ok) {
            const ScRun ru = runs[ch.r0 + prun];
            bulk_reduce_add_f64(orow + ru.p0, bb + (size_t)pst * SC_MAXPTS + ru.off, (unsigned)ru.len * 16u);
        }
        bulk_commit_group();
    }
    bulk_wait_group_read<0>();                                  // the buffers may be released; the kernel boundary completes the additions
}

}  // namespace tdh
