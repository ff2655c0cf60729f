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
// Slice ks covers the chunks [ks*chunks_per_slice, (ks+1)*chunks_per_slice) of the ceil(N_p/16) chunks.
// hermitian != 0 (a and b are the same block): tiles below the diagonal are skipped, the reduction mirrors them.
__global__ void __launch_bounds__(OV_THREADS)
overlap_kernel(const cd* __restrict__ a, int na, const cd* __restrict__ b, int nb, size_t npts, int tiles_j,
               int chunks_per_slice, cd* __restrict__ part, int hermitian)
{
    if (hermitian && (int)(blockIdx.x % tiles_j) < (int)(blockIdx.x / tiles_j)) return;
    __shared__ double sre[2 * OV_T][OV_KCP];     // rows 0..63: A tile (states of a), rows 64..127: B tile (states of b)
    __shared__ double sim[2 * OV_T][OV_KCP];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wi = warp >> 2, wj = warp & 3;                    // warp grid 2 x 4
    const int fr = lane >> 2, fk = lane & 3;                    // fragment row (state) and k (point)
    const int ti = blockIdx.x / tiles_j, tj = blockIdx.x % tiles_j;
    const int i0 = ti * OV_T, j0 = tj * OV_T;
    const size_t nchunks = (npts + OV_KC - 1) / OV_KC;           // the last chunk may be ragged (loads predicated)
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
        const bool inside = c * OV_KC + (tid & 15) < npts;       // every slot of this thread has point tid % 16
#pragma unroll
        for (int r = 0; r < 8; ++r) v[r] = (ok[r] && inside) ? __ldcs(src[r] + c * OV_KC) : make_double2(0.0, 0.0);
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

// s[i][j] = dv * sum over slices (in order) of part[ks][i][j]; hermitian: elements in tiles below the diagonal are the
// conjugates of their mirror images (which were computed)
__global__ void overlap_reduce_kernel(const cd* __restrict__ part, int ksplit, int na, int nb, int na_pad, int nb_pad,
                                      double dv, cd* __restrict__ s, int hermitian)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= na * nb) return;
    int i = idx / nb, j = idx % nb;
    const bool mirror = hermitian && (j / OV_T) < (i / OV_T);
    if (mirror) { const int t = i; i = j; j = t; }
    double re = 0.0, im = 0.0;
    for (int ks = 0; ks < ksplit; ++ks) {
        const cd v = part[((size_t)ks * na_pad + i) * nb_pad + j];
        re += v.x;
        im += v.y;
    }
    s[idx] = make_double2(dv * re, mirror ? -dv * im : dv * im);
}

// ------------------------------------------------------------------------------------------------------------
// Rotation in the space of states:   out_j[p] = sum_i psi_i[p] m[i][j],   i < n_in, j < n_out
// A complex "NN" GEMM with M = N_p (contiguous), K = n_in, N = n_out.  CTA = 64 points x 64 output states, 8 warps as
// 2 (points) x 4 (states), a warp owns 32 points x 16 states = 4 x 2 MMA tiles; K advances in chunks of 16 input states.
// Fragments: A[row = point][k = state i] from the psi tile [i][64 points] (re / im planes, rows padded to 68 doubles),
// B[k = state i][n = state j] from the m tile [i][64 j] (padded to 68): lane l reads (row l/4, k l%4) of either -- both
// conflict free.  The C fragment (point l/4, states 2*(l%4) + {0,1}) is stored straight to out: for one output state
// 8 lanes write 8 consecutive points.  upper != 0: m is upper triangular (m[i][j] = 0 for i > j, the Cholesky case),
// input states beyond the tile's last column are skipped.
// ------------------------------------------------------------------------------------------------------------
constexpr int RT_P = 64;          // points per tile
constexpr int RT_J = 64;          // output states per tile
constexpr int RT_KC = 16;         // input states per chunk
constexpr int RT_LD = 68;         // padded row length (doubles)

// grid: (ceil(N_p / 64), ceil(n_out / 64)); loads and stores of the last tile of points are predicated
__global__ void __launch_bounds__(OV_THREADS)
rotate_kernel(const cd* __restrict__ psi, int n_in, const cd* __restrict__ m, int n_out, size_t npts, int upper,
              cd* __restrict__ out)
{
    __shared__ double are[RT_KC][RT_LD], aim[RT_KC][RT_LD];      // psi tile: [state i][point]
    __shared__ double bre[RT_KC][RT_LD], bim[RT_KC][RT_LD];      // m tile:   [state i][state j]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wp = warp >> 2, wj = warp & 3;                    // warp grid 2 x 4
    const int fr = lane >> 2, fk = lane & 3;
    const size_t p0 = (size_t)blockIdx.x * RT_P;
    const int j0 = blockIdx.y * RT_J;
    const int k_end = upper ? (n_in < j0 + RT_J ? n_in : j0 + RT_J) : n_in;

    double cre[4][2][2], cim[4][2][2];
#pragma unroll
    for (int it = 0; it < 4; ++it)
#pragma unroll
        for (int jt = 0; jt < 2; ++jt) cre[it][jt][0] = cre[it][jt][1] = cim[it][jt][0] = cim[it][jt][1] = 0.0;

    // load slots: 16 x 64 values of each tile = 1024 per tile, 4 + 4 per thread; slot r -> row (tid + 256 r) / 64
    cd va[4], vb[4];
    auto load = [&](int k0) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int idx = tid + OV_THREADS * r, row = idx >> 6, col = idx & 63;
            const int i = k0 + row;
            va[r] = (i < k_end && p0 + col < npts) ? __ldcs(psi + (size_t)i * npts + p0 + col) : make_double2(0.0, 0.0);
            vb[r] = (i < k_end && j0 + col < n_out) ? __ldg(m + (size_t)i * n_out + j0 + col) : make_double2(0.0, 0.0);
        }
    };
    if (k_end > 0) load(0);
    for (int k0 = 0; k0 < k_end; k0 += RT_KC) {
        __syncthreads();
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int idx = tid + OV_THREADS * r, row = idx >> 6, col = idx & 63;
            are[row][col] = va[r].x; aim[row][col] = va[r].y;
            bre[row][col] = vb[r].x; bim[row][col] = vb[r].y;
        }
        __syncthreads();
        if (k0 + RT_KC < k_end) load(k0 + RT_KC);
#pragma unroll
        for (int k4 = 0; k4 < RT_KC / 4; ++k4) {
            double ar[4], ai[4], br[2], bi[2];
#pragma unroll
            for (int it = 0; it < 4; ++it) {
                ar[it] = are[k4 * 4 + fk][wp * 32 + it * 8 + fr];
                ai[it] = aim[k4 * 4 + fk][wp * 32 + it * 8 + fr];
            }
#pragma unroll
            for (int jt = 0; jt < 2; ++jt) {
                br[jt] = bre[k4 * 4 + fk][wj * 16 + jt * 8 + fr];
                bi[jt] = bim[k4 * 4 + fk][wj * 16 + jt * 8 + fr];
            }
#pragma unroll
            for (int it = 0; it < 4; ++it)
#pragma unroll
                for (int jt = 0; jt < 2; ++jt) {
                    dmma_m8n8k4(cre[it][jt], ar[it], br[jt]);
                    dmma_m8n8k4(cre[it][jt], -ai[it], bi[jt]);
                    dmma_m8n8k4(cim[it][jt], ar[it], bi[jt]);
                    dmma_m8n8k4(cim[it][jt], ai[it], br[jt]);
                }
        }
    }
#pragma unroll
    for (int it = 0; it < 4; ++it)
#pragma unroll
        for (int jt = 0; jt < 2; ++jt) {
            const size_t p = p0 + wp * 32 + it * 8 + fr;
            const int j = j0 + wj * 16 + jt * 8 + 2 * fk;
            if (p >= npts) continue;                             // ragged last tile of points
            if (j < n_out) __stcs(out + (size_t)j * npts + p, make_double2(cre[it][jt][0], cim[it][jt][0]));
            if (j + 1 < n_out) __stcs(out + (size_t)(j + 1) * npts + p, make_double2(cre[it][jt][1], cim[it][jt][1]));
        }
}

// ------------------------------------------------------------------------------------------------------------
// Small dense kernels of the Cholesky orthonormalisation (n <= 1024; O(n^3 / 3) flop against the O(n^2 N_p) of the two
// GEMMs): s (n x n, row-major, Hermitian) -> lower Cholesky factor L in place (upper part untouched), then
// m = L^{-H} (upper triangular), the rotation matrix of psi' = psi L^{-H}.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ cd warp_sum(cd v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
    }
    return v;
}

// Left-looking Cholesky in the L D L^H form, cooperative launch (all CTAs resident), one grid barrier per column.
// Column k: every row i >= k (one warp per row, lanes over j) subtracts sum_{j<k} u[i][j] conj(u[k][j]) / d_j from
// s[i][k], where u are the not yet scaled columns and d_j the pivots; after the barrier every CTA reads the pivot
// d_k = s[k][k] into its own shared copy of 1/d.  A final pass scales column j by 1/sqrt(d_j).
// *status = k + 1 if pivot k is not positive or has lost more than 13 digits against the diagonal element it started
// from (s not positive definite to working precision: linearly dependent states), else 0.
__global__ void __launch_bounds__(256)
cholesky_kernel(cd* __restrict__ s, int n, int* __restrict__ status, unsigned* __restrict__ barrier)
{
    __shared__ double invd[1024];
    __shared__ double orig[1024];
    __shared__ int bad;
    const int tid = threadIdx.x, lane = tid & 31;
    const int gw = (blockIdx.x * blockDim.x + tid) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    if (tid == 0) bad = 0;
    for (int i = tid; i < n; i += blockDim.x) orig[i] = s[(size_t)i * n + i].x;
    __syncthreads();
    // sense-free grid barrier on a monotonically increasing counter (cooperative launch: every CTA is resident)
    unsigned epoch = 0;
    auto grid_barrier = [&]() {
        __syncthreads();
        if (tid == 0) {
            epoch += gridDim.x;
            __threadfence();
            atomicAdd(barrier, 1u);
            while (*((volatile unsigned*)barrier) < epoch) {}
            __threadfence();
        }
        __syncthreads();
    };
    for (int k = 0; k < n; ++k) {
        for (int i = k + gw; i < n; i += nw) {
            const cd* ri = s + (size_t)i * n;
            const cd* rk = s + (size_t)k * n;
            cd acc = make_double2(0.0, 0.0);
            for (int j = lane; j < k; j += 32) {
                const cd a = __ldcg(ri + j), b = __ldcg(rk + j);
                const double w = invd[j];
                acc.x += w * (a.x * b.x + a.y * b.y);
                acc.y += w * (a.y * b.x - a.x * b.y);
            }
            acc = warp_sum(acc);
            if (lane == 0) {
                cd v = __ldcg(ri + k);
                v.x -= acc.x;
                v.y -= acc.y;
                __stcg(s + (size_t)i * n + k, v);
            }
        }
        grid_barrier();
        if (tid == 0) {
            const double d = __ldcg(s + (size_t)k * n + k).x;
            if (!(d > 1e-13 * orig[k])) { bad = k + 1; invd[k] = 1.0; } else { invd[k] = 1.0 / d; }
        }
        __syncthreads();
        if (bad) break;                       // every CTA sees the same pivot and leaves together
    }
    if (bad) { if (blockIdx.x == 0 && tid == 0) *status = bad; return; }
    if (blockIdx.x == 0 && tid == 0) *status = 0;
    // scale: L[i][j] = u[i][j] / sqrt(d_j), L[j][j] = sqrt(d_j)
    for (size_t e = (size_t)blockIdx.x * blockDim.x + tid; e < (size_t)n * n; e += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / n), j = (int)(e % n);
        if (j <= i) {
            const cd u = __ldcg(s + e);
            const double r = sqrt(invd[j]);
            s[e] = (i == j) ? make_double2(1.0 / r, 0.0) : make_double2(u.x * r, u.y * r);
        }
    }
}

// m = L^{-H}: one warp per column j of W = L^{-1} (forward substitution, the column kept in shared memory):
//   w_jj = 1 / L_jj,   w_ij = -(sum_{k=j}^{i-1} L[i][k] w_kj) / L_ii,   m[j][i] = conj(w_ij),   m[i][j] = 0 for i > j.
// dynamic shared memory: (blockDim.x / 32) * n complex values.
__global__ void inverse_lower_conjtrans_kernel(const cd* __restrict__ l, int n, cd* __restrict__ m)
{
    extern __shared__ __align__(16) unsigned char smem_inv[];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    cd* w = reinterpret_cast<cd*>(smem_inv) + (size_t)wl * n;
    const int j = blockIdx.x * (blockDim.x >> 5) + wl;
    if (j >= n) return;
    for (int i = lane; i < j; i += 32) m[(size_t)j * n + i] = make_double2(0.0, 0.0);
    if (lane == 0) {
        const double dj = 1.0 / l[(size_t)j * n + j].x;
        w[j] = make_double2(dj, 0.0);
        m[(size_t)j * n + j] = make_double2(dj, 0.0);
    }
    __syncwarp();
    for (int i = j + 1; i < n; ++i) {
        const cd* li = l + (size_t)i * n;
        cd acc = make_double2(0.0, 0.0);
        for (int k = j + lane; k < i; k += 32) acc = cfma(__ldg(li + k), w[k], acc);
        acc = warp_sum(acc);
        if (lane == 0) {
            const double di = -1.0 / __ldg(li + i).x;
            const cd v = cscale(acc, di);
            w[i] = v;
            m[(size_t)j * n + i] = make_double2(v.x, -v.y);
        }
        __syncwarp();
    }
}

}  // namespace tdh
