// overlap_kernels.cuh -- overlap / subspace matrix of two state blocks on FP64 tensor cores (first block of NEXT-3).
//
//     S[i][j] = dV sum_p conj(a_i[p]) b_j[p],   i < na, j < nb
//
// A complex "TN" GEMM with M = na, N = nb and K = N_p (both operands contiguous along K: a state is a contiguous
// array of grid points).  Unlike the projector contractions this one is flop bound: 8 na nb N_p flop against
// 16 (na + nb) N_p bytes.
//
// CTA = 64 x 64 tile of S and one slice of K (split-K: partial tiles go to a workspace and are summed in slice order
// by overlap_reduce_kernel -- deterministic, no atomics).  256 threads = 8 warps as 2 x 4, a warp owns 32 x 16 of the
// tile = 4 x 2 MMA tiles.  K advances in chunks of 16 points: the chunk of all 128 states (32 KB) is loaded with
// 16-byte loads (16 lanes = 256 contiguous bytes of one state) into registers while the previous chunk is multiplied,
// then stored to shared memory as separate re / im planes [state][20 doubles] -- the padding to 20 makes the fragment
// reads (lane l: state l/4, point l%4, 8 bytes) conflict free.  Per step of 4 points and per MMA tile
//     mma.sync.m8n8k4.f64 x 4:   Cre += Ar Br + Ai Bi,   Cim += Ar Bi - Ai Br          (conj on the left operand)
// with A[row = state i][k = point] and B[k = point][n = state j], i.e. the same fragment addressing for both.
#pragma once
#include "fft_codelets.cuh"
#include "nl_kernels.cuh"

namespace tdh {

constexpr int OV_T = 64;          // tile edge (states)
constexpr int OV_KC = 16;         // points per chunk
constexpr int OV_KCP = 20;        // padded row length (doubles) of a state in shared memory
constexpr int OV_THREADS = 256;

// grid: (tiles_i * tiles_j, ksplit).  part: [ksplit][na_pad][nb_pad] complex, na_pad = tiles_i*64, nb_pad = tiles_j*64.
// Slice ks covers the chunks [ks*chunks_per_slice, (ks+1)*chunks_per_slice) of the N_p/16 chunks.
__global__ void __launch_bounds__(OV_THREADS)
overlap_kernel(const cd* __restrict__ a, int na, const cd* __restrict__ b, int nb, size_t npts, int tiles_j,
               int chunks_per_slice, cd* __restrict__ part)
{
    __shared__ double sre[2 * OV_T][OV_KCP];     // rows 0..63: A tile (states of a), rows 64..127: B tile (states of b)
    __shared__ double sim[2 * OV_T][OV_KCP];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wi = warp >> 2, wj = warp & 3;                    // warp grid 2 x 4
    const int fr = lane >> 2, fk = lane & 3;                    // fragment row (state) and k (point)
    const int ti = blockIdx.x / tiles_j, tj = blockIdx.x % tiles_j;
    const int i0 = ti * OV_T, j0 = tj * OV_T;
    const size_t nchunks = npts / OV_KC;
    const size_t c_begin = (size_t)blockIdx.y * chunks_per_slice;
    const size_t c_end = c_begin + chunks_per_slice < nchunks ? c_begin + chunks_per_slice : nchunks;

    // this thread's 8 load slots: slot r -> row (tid + 256 r) / 16 of the 128-row tile, point (tid + 256 r) % 16
    const cd* src[8];
    bool ok[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int idx = tid + OV_THREADS * r, row = idx >> 4, pt = idx & 15;
        const bool isb = row >= OV_T;
        const int st = isb ? j0 + row - OV_T : i0 + row;
        ok[r] = isb ? st < nb : st < na;
        src[r] = (isb ? b : a) + (size_t)(ok[r] ? st : 0) * npts + pt;
    }
    double cre[4][2][2], cim[4][2][2];
#pragma unroll
    for (int it = 0; it < 4; ++it)
#pragma unroll
        for (int jt = 0; jt < 2; ++jt) cre[it][jt][0] = cre[it][jt][1] = cim[it][jt][0] = cim[it][jt][1] = 0.0;

    cd v[8];
    auto load = [&](size_t c) {
#pragma unroll
        for (int r = 0; r < 8; ++r) v[r] = ok[r] ? __ldcs(src[r] + c * OV_KC) : make_double2(0.0, 0.0);
    };
    if (c_begin < c_end) load(c_begin);
    for (size_t c = c_begin; c < c_end; ++c) {
        __syncthreads();                                         // the previous chunk has been consumed
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int idx = tid + OV_THREADS * r, row = idx >> 4, pt = idx & 15;
            sre[row][pt] = v[r].x;
            sim[row][pt] = v[r].y;
        }
        __syncthreads();
        if (c + 1 < c_end) load(c + 1);                          // in flight during the multiplications below
#pragma unroll
        for (int k4 = 0; k4 < OV_KC / 4; ++k4) {
            double ar[4], ai[4], br[2], bi[2];
#pragma unroll
            for (int it = 0; it < 4; ++it) {
                ar[it] = sre[wi * 32 + it * 8 + fr][k4 * 4 + fk];
                ai[it] = sim[wi * 32 + it * 8 + fr][k4 * 4 + fk];
            }
#pragma unroll
            for (int jt = 0; jt < 2; ++jt) {
                br[jt] = sre[OV_T + wj * 16 + jt * 8 + fr][k4 * 4 + fk];
                bi[jt] = sim[OV_T + wj * 16 + jt * 8 + fr][k4 * 4 + fk];
            }
#pragma unroll
            for (int it = 0; it < 4; ++it)
#pragma unroll
                for (int jt = 0; jt < 2; ++jt) {
                    dmma_m8n8k4(cre[it][jt], ar[it], br[jt]);
                    dmma_m8n8k4(cre[it][jt], ai[it], bi[jt]);
                    dmma_m8n8k4(cim[it][jt], ar[it], bi[jt]);
                    dmma_m8n8k4(cim[it][jt], -ai[it], br[jt]);
                }
        }
    }
    // C fragment: row = lane/4, columns 2*(lane%4) + {0,1}
    const int nb_pad = tiles_j * OV_T;
    const size_t na_pad = (size_t)gridDim.x / tiles_j * OV_T;
    cd* dst = part + (size_t)blockIdx.y * na_pad * nb_pad;
#pragma unroll
    for (int it = 0; it < 4; ++it)
#pragma unroll
        for (int jt = 0; jt < 2; ++jt) {
            const int i = i0 + wi * 32 + it * 8 + fr, j = j0 + wj * 16 + jt * 8 + 2 * fk;
            dst[(size_t)i * nb_pad + j] = make_double2(cre[it][jt][0], cim[it][jt][0]);
            dst[(size_t)i * nb_pad + j + 1] = make_double2(cre[it][jt][1], cim[it][jt][1]);
        }
}

// s[i][j] = dv * sum over slices (in order) of part[ks][i][j]
__global__ void overlap_reduce_kernel(const cd* __restrict__ part, int ksplit, int na, int nb, int na_pad, int nb_pad,
                                      double dv, cd* __restrict__ s)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= na * nb) return;
    const int i = idx / nb, j = idx % nb;
    double re = 0.0, im = 0.0;
    for (int ks = 0; ks < ksplit; ++ks) {
        const cd v = part[((size_t)ks * na_pad + i) * nb_pad + j];
        re += v.x;
        im += v.y;
    }
    s[idx] = make_double2(dv * re, dv * im);
}

}  // namespace tdh
