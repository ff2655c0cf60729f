// eigh_kernels.cuh -- Hermitian eigensolver of the n_st x n_st subspace matrix (subspace diagonalisation).
//
// Parallel two-sided Jacobi with a round-robin (tournament) ordering: every step rotates n/2 disjoint pairs (p, q) at
// once, a sweep is n - 1 steps.  For a pair with a_pq = |a_pq| e^{i phi}, tau = (a_qq - a_pp) / (2 |a_pq|),
// t = sign(tau) / (|tau| + sqrt(1 + tau^2)), c = 1 / sqrt(1 + t^2), s = t c, the unitary
//     J_pp = c,  J_pq = s,  J_qp = -s e^{-i phi},  J_qq = c e^{-i phi}
// zeroes a_pq in J^H A J.  One cooperative launch (every CTA resident) runs all sweeps; a step is three phases
// separated by grid barriers: the rotation parameters of the step's pairs from the current matrix, the column update
// A <- A J and V <- V J, the row update A <- J^H A.  The matrix (16 MB at n = 1024) lives in L2; every access that
// crosses CTAs goes through ld.global.cg / st.global.cg.  Sweeps stop when the largest rotated |a_pq| of a sweep is
// below 1e-15 of the largest matrix element (checked identically by every CTA), at most 40 sweeps.
// The O(n^3) work of this kernel is small beside the O(n^2 N_p) of the GEMMs around it.
#pragma once
#include "fft_codelets.cuh"

namespace tdh {

// pair k (0 <= k < m/2) of step r (0 <= r < m-1) of the round-robin tournament on m (even) players
__device__ __forceinline__ void jacobi_pair(int m, int r, int k, int& p, int& q) {
    int i, j;
    if (k == 0) { i = m - 1; j = r; }
    else { i = (r + k) % (m - 1); j = (r - k + (m - 1)) % (m - 1); }
    p = i < j ? i : j;
    q = i < j ? j : i;
}

struct __align__(16) JacobiRot { double c, s, cph, sph; };      // e^{i phi} = cph + i sph
// the rotations are written by one CTA and read by all others in the next phase: through L2
__device__ __forceinline__ JacobiRot ld_rot(const JacobiRot* p) {
    const double2 a = __ldcg(reinterpret_cast<const double2*>(p)), b = __ldcg(reinterpret_cast<const double2*>(p) + 1);
    JacobiRot r;
    r.c = a.x; r.s = a.y; r.cph = b.x; r.sph = b.y;
    return r;
}
__device__ __forceinline__ void st_rot(JacobiRot* p, const JacobiRot& r) {
    __stcg(reinterpret_cast<double2*>(p), make_double2(r.c, r.s));
    __stcg(reinterpret_cast<double2*>(p) + 1, make_double2(r.cph, r.sph));
}

// a: n x n Hermitian (row-major), overwritten; v: n x n, receives the eigenvectors as columns (not yet sorted);
// rot: scratch [m/2]; ctl (8 words, zeroed): [0] grid-barrier counter, [2..3] (64-bit) largest |a_pq| of the sweep,
// [4] sweeps used
__global__ void __launch_bounds__(256)
jacobi_eigh_kernel(cd* __restrict__ a, cd* __restrict__ v, int n, JacobiRot* __restrict__ rot, unsigned* __restrict__ ctl)
{
    const int tid = threadIdx.x;
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + tid, gsize = (size_t)gridDim.x * blockDim.x;
    const int m = n + (n & 1), half = m / 2;
    unsigned long long* sweep_max = reinterpret_cast<unsigned long long*>(ctl + 2);
    unsigned epoch = 0;
    auto grid_barrier = [&]() {
        __syncthreads();
        if (tid == 0) {
            epoch += gridDim.x;
            __threadfence();
            atomicAdd(ctl, 1u);
            while (*((volatile unsigned*)ctl) < epoch) {}
            __threadfence();
        }
        __syncthreads();
    };
    // v = identity; scale = largest |a_ij|
    double mx = 0.0;
    for (size_t e = gtid; e < (size_t)n * n; e += gsize) {
        v[e] = make_double2((e / n == e % n) ? 1.0 : 0.0, 0.0);
        const cd x = __ldcg(a + e);
        mx = fmax(mx, fmax(fabs(x.x), fabs(x.y)));
    }
    atomicMax(sweep_max, (unsigned long long)__double_as_longlong(mx));
    grid_barrier();
    const double scale = __longlong_as_double((long long)*((volatile unsigned long long*)sweep_max));
    grid_barrier();
    if (gtid == 0) *sweep_max = 0ull;
    grid_barrier();
    int sweep = 0;
    for (; sweep < 40; ++sweep) {
        for (int r = 0; r < m - 1; ++r) {
            // ---- phase 0: rotation parameters of this step's pairs
            for (size_t k = gtid; k < (size_t)half; k += gsize) {
                int p, q;
                jacobi_pair(m, r, (int)k, p, q);
                JacobiRot jr = {1.0, 0.0, 1.0, 0.0};
                if (q < n) {
                    const double app = __ldcg(a + (size_t)p * n + p).x, aqq = __ldcg(a + (size_t)q * n + q).x;
                    const cd apq = __ldcg(a + (size_t)p * n + q);
                    const double mag = hypot(apq.x, apq.y);
                    if (mag > 0.0) {
                        atomicMax(sweep_max, (unsigned long long)__double_as_longlong(mag));
                        const double tau = (aqq - app) / (2.0 * mag);
                        const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                        jr.c = 1.0 / sqrt(1.0 + t * t);
                        jr.s = t * jr.c;
                        jr.cph = apq.x / mag;
                        jr.sph = apq.y / mag;
                    }
                }
                st_rot(rot + k, jr);
            }
            grid_barrier();
            // ---- phase 1: columns p, q of A and of V:  [x, y] <- [c x - s e^{-i phi} y,  s x + c e^{-i phi} y]
            for (size_t e = gtid; e < (size_t)n * half; e += gsize) {
                const int row = (int)(e / half), k = (int)(e % half);
                int p, q;
                jacobi_pair(m, r, k, p, q);
                if (q >= n) continue;
                const JacobiRot jr = ld_rot(rot + k);
                if (jr.s == 0.0) continue;
#pragma unroll
                for (int which = 0; which < 2; ++which) {
                    cd* mat = which ? v : a;
                    const cd x = __ldcg(mat + (size_t)row * n + p), y = __ldcg(mat + (size_t)row * n + q);
                    const cd ey = make_double2(y.x * jr.cph + y.y * jr.sph, y.y * jr.cph - y.x * jr.sph);   // e^{-i phi} y
                    __stcg(mat + (size_t)row * n + p, make_double2(jr.c * x.x - jr.s * ey.x, jr.c * x.y - jr.s * ey.y));
                    __stcg(mat + (size_t)row * n + q, make_double2(jr.s * x.x + jr.c * ey.x, jr.s * x.y + jr.c * ey.y));
                }
            }
            grid_barrier();
            // ---- phase 2: rows p, q of A:  [x; y] <- [c x - s e^{i phi} y;  s x + c e^{i phi} y]
            for (size_t e = gtid; e < (size_t)half * n; e += gsize) {
                const int k = (int)(e / n), col = (int)(e % n);
                int p, q;
                jacobi_pair(m, r, k, p, q);
                if (q >= n) continue;
                const JacobiRot jr = ld_rot(rot + k);
                if (jr.s == 0.0) continue;
                const cd x = __ldcg(a + (size_t)p * n + col), y = __ldcg(a + (size_t)q * n + col);
                const cd ey = make_double2(y.x * jr.cph - y.y * jr.sph, y.y * jr.cph + y.x * jr.sph);       // e^{+i phi} y
                __stcg(a + (size_t)p * n + col, make_double2(jr.c * x.x - jr.s * ey.x, jr.c * x.y - jr.s * ey.y));
                __stcg(a + (size_t)q * n + col, make_double2(jr.s * x.x + jr.c * ey.x, jr.s * x.y + jr.c * ey.y));
            }
            grid_barrier();
        }
        // ---- end of the sweep: every CTA reads the same maximum, then it is reset behind a barrier
        const double big = __longlong_as_double((long long)*((volatile unsigned long long*)sweep_max));
        grid_barrier();
        if (gtid == 0) *sweep_max = 0ull;
        grid_barrier();
        if (big <= 1e-15 * scale) { ++sweep; break; }
    }
    if (gtid == 0) ctl[4] = (unsigned)sweep;
}

// eigenvalues ascending and the matching column permutation of v: w[rank] = a[i][i], vout[:, rank] = v[:, i]
__global__ void eigh_sort_kernel(const cd* __restrict__ a, const cd* __restrict__ v, int n, double* __restrict__ w,
                                 cd* __restrict__ vout)
{
    extern __shared__ double ev[];
    for (int i = threadIdx.x; i < n; i += blockDim.x) ev[i] = a[(size_t)i * n + i].x;
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double e = ev[i];
        int rank = 0;
        for (int j = 0; j < n; ++j) rank += (ev[j] < e) || (ev[j] == e && j < i);
        w[rank] = e;
        for (int row = 0; row < n; ++row) vout[(size_t)row * n + rank] = v[(size_t)row * n + i];
    }
}

// m <- (m + m^H) / 2 into out (the subspace matrix is Hermitian up to rounding)
__global__ void symmetrize_kernel(const cd* __restrict__ m, int n, cd* __restrict__ out) {
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < (size_t)n * n; e += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / n), j = (int)(e % n);
        const cd x = m[e], y = m[(size_t)j * n + i];
        out[e] = make_double2(0.5 * (x.x + y.x), 0.5 * (x.y - y.y));
    }
}

}  // namespace tdh
