// eigh_kernels.cuh -- Hermitian eigensolver of the n_st x n_st subspace matrix (subspace diagonalisation).
//
// Parallel two-sided Jacobi with a round-robin (tournament) ordering: every step rotates n/2 disjoint pairs (p, q) at
// once, a sweep is n - 1 steps.  For a pair with a_pq = |a_pq| e^{i phi}, tau = (a_qq - a_pp) / (2 |a_pq|),
// t = sign(tau) / (|tau| + sqrt(1 + tau^2)), c = 1 / sqrt(1 + t^2), s = t c, the unitary
//     J_pp = c,  J_pq = s,  J_qp = -s e^{-i phi},  J_qq = c e^{-i phi}
// zeroes a_pq in J^H A J.  One cooperative launch (every CTA resident) runs all sweeps with ONE grid barrier per step:
//   * every CTA computes the rotations of all n/2 pairs of the step itself (three matrix elements per pair, into shared
//     memory) -- redundant arithmetic instead of a phase and a barrier of its own; the largest rotated |a_pq| of a sweep
//     is therefore known to every CTA without any communication;
//   * the two-sided update is done per 2 x 2 block (row pair P, column pair C): B' = J_P^H B J_C, read from one copy of
//     the matrix and written to the other (ping-pong), so no CTA can read an element another CTA has already replaced;
//     V <- V J in place (no CTA reads V).
// The arithmetic per element (column rotation, then row rotation) is that of the three-phase version of round 1 (65 ms
// for n = 512: three barriers per step).  The matrices (2 x 4 MB + 4 MB at n = 512) live in L2; every access that
// crosses CTAs goes through ld.global.cg / st.global.cg.  Threshold Jacobi: elements below JACOBI_TOL of the largest
// matrix element are not rotated, a step without any rotation costs no update and no barrier (the last, verifying sweep
// is therefore cheap), and the sweeps stop after one in which nothing was rotated; at most JACOBI_MAX_SWEEPS sweeps;
// ctl[4] receives the sweeps used and ctl[5] = 1 when the last sweep still rotated (the host reports that as an error).
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
constexpr int JACOBI_MAX_SWEEPS = 40;
constexpr int JACOBI_T = 512;
constexpr double JACOBI_TOL = 1e-14;      // off-diagonal elements below JACOBI_TOL * max|a_ij| are not rotated

// a: n x n Hermitian (row-major), overwritten; a2: second n x n buffer (ping-pong); v: n x n, receives the eigenvectors as
// columns (not yet sorted); ctl (8 words, zeroed): [0] grid-barrier counter, [2..3] (64-bit) largest |a_ij| of the input,
// [4] sweeps used, [5] not converged.  On return the diagonal of `a` holds the eigenvalues.
// Dynamic shared memory: (n + 1) / 2 JacobiRot.
__global__ void __launch_bounds__(JACOBI_T)
jacobi_eigh_kernel(cd* __restrict__ a, cd* __restrict__ a2, cd* __restrict__ v, int n, unsigned* __restrict__ ctl)
{
    extern __shared__ __align__(16) unsigned char jsm[];
    JacobiRot* srot = reinterpret_cast<JacobiRot*>(jsm);
    __shared__ double red[JACOBI_T / 32];
    const int tid = threadIdx.x;
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + tid, gsize = (size_t)gridDim.x * blockDim.x;
    const int m = n + (n & 1), half = m / 2;
    unsigned long long* scale_word = reinterpret_cast<unsigned long long*>(ctl + 2);
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
        // fmax drops a NaN and the threshold test below never rotates one: a non-finite element is recorded as an
        // infinite scale instead, which ends the solve as "not converged"
        if (!(fabs(x.x) <= 1.7976931348623157e308) || !(fabs(x.y) <= 1.7976931348623157e308))
            mx = __longlong_as_double(0x7ff0000000000000LL);
    }
    atomicMax(scale_word, (unsigned long long)__double_as_longlong(mx));
    grid_barrier();
    const double scale = __longlong_as_double((long long)*((volatile unsigned long long*)scale_word));
    const bool finite = scale <= 1.7976931348623157e308;     // the same value in every CTA
    const double thr = JACOBI_TOL * scale;
    cd* cur = a;
    cd* nxt = a2;
    int sweep = 0;
    bool converged = false;
    for (; finite && sweep < JACOBI_MAX_SWEEPS && !converged; ++sweep) {
        double tmax = 0.0;                                   // this thread's largest rotated |a_pq| of the sweep
        for (int r = 0; r < m - 1; ++r) {
            // ---- rotations of this step's pairs, computed by every CTA from the current matrix
            int any = 0;
            for (int k = tid; k < half; k += JACOBI_T) {
                int p, q;
                jacobi_pair(m, r, k, p, q);
                JacobiRot jr = {1.0, 0.0, 1.0, 0.0};
                if (q < n) {
                    const double app = __ldcg(cur + (size_t)p * n + p).x, aqq = __ldcg(cur + (size_t)q * n + q).x;
                    const cd apq = __ldcg(cur + (size_t)p * n + q);
                    const double mag = sqrt(apq.x * apq.x + apq.y * apq.y);
                    if (mag > thr) {                         // threshold Jacobi: smaller elements are left alone
                        tmax = fmax(tmax, mag);
                        any = 1;
                        const double tau = (aqq - app) / (2.0 * mag);
                        const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                        jr.c = 1.0 / sqrt(1.0 + t * t);
                        jr.s = t * jr.c;
                        jr.cph = apq.x / mag;
                        jr.sph = apq.y / mag;
                    }
                }
                srot[k] = jr;
            }
            // a step without any rotation changes nothing: no update, no barrier (every CTA takes the same decision, it
            // has computed the same rotations from the same matrix)
            if (!__syncthreads_or(any)) continue;
            // ---- one pass per thread over its items: 2 x 2 blocks of A (row pair kp, column pair kc), B' = J_P^H (B J_C),
            //      cur -> nxt, and (row, column pair) items of V <- V J in place.  All loads of an item pair are issued
            //      before the arithmetic (one L2 round trip per pass).
            const int na_items = half * half, nv_items = n * half;         // n <= 1024: 32-bit index arithmetic
            for (int e = (int)gtid; e < na_items || e < nv_items; e += (int)gsize) {
                const bool do_a = e < na_items, do_v = e < nv_items;
                int p = 0, q = 0, cr = 0, cs = 0, vp = 0, vq = 0, vrow = 0;
                bool qv = false, sv = false;
                JacobiRot jp = {1.0, 0.0, 1.0, 0.0}, jc = jp, jv = jp;
                const cd z0 = make_double2(0.0, 0.0);
                cd b11 = z0, b12 = z0, b21 = z0, b22 = z0, vx = z0, vy = z0;
                if (do_a) {
                    const int kp = e / half, kc = e % half;
                    jacobi_pair(m, r, kp, p, q);
                    jacobi_pair(m, r, kc, cr, cs);
                    qv = q < n; sv = cs < n;
                    jp = srot[kp]; jc = srot[kc];
                    b11 = __ldcg(cur + (size_t)p * n + cr);
                    if (sv) b12 = __ldcg(cur + (size_t)p * n + cs);
                    if (qv) b21 = __ldcg(cur + (size_t)q * n + cr);
                    if (qv && sv) b22 = __ldcg(cur + (size_t)q * n + cs);
                }
                bool v_on = false;
                if (do_v) {
                    vrow = e / half;
                    const int k = e % half;
                    jacobi_pair(m, r, k, vp, vq);
                    jv = srot[k];
                    v_on = vq < n && jv.s != 0.0;
                    if (v_on) { vx = __ldcg(v + (size_t)vrow * n + vp); vy = __ldcg(v + (size_t)vrow * n + vq); }
                }
                if (do_a) {
                    if (jc.s != 0.0) {       // columns: [x, y] <- [c x - s e^{-i phi} y,  s x + c e^{-i phi} y]
                        const cd e1 = make_double2(b12.x * jc.cph + b12.y * jc.sph, b12.y * jc.cph - b12.x * jc.sph);
                        const cd e2 = make_double2(b22.x * jc.cph + b22.y * jc.sph, b22.y * jc.cph - b22.x * jc.sph);
                        const cd n11 = make_double2(jc.c * b11.x - jc.s * e1.x, jc.c * b11.y - jc.s * e1.y);
                        const cd n12 = make_double2(jc.s * b11.x + jc.c * e1.x, jc.s * b11.y + jc.c * e1.y);
                        const cd n21 = make_double2(jc.c * b21.x - jc.s * e2.x, jc.c * b21.y - jc.s * e2.y);
                        const cd n22 = make_double2(jc.s * b21.x + jc.c * e2.x, jc.s * b21.y + jc.c * e2.y);
                        b11 = n11; b12 = n12; b21 = n21; b22 = n22;
                    }
                    if (jp.s != 0.0) {       // rows: [x; y] <- [c x - s e^{+i phi} y;  s x + c e^{+i phi} y]
                        const cd e1 = make_double2(b21.x * jp.cph - b21.y * jp.sph, b21.y * jp.cph + b21.x * jp.sph);
                        const cd e2 = make_double2(b22.x * jp.cph - b22.y * jp.sph, b22.y * jp.cph + b22.x * jp.sph);
                        const cd n11 = make_double2(jp.c * b11.x - jp.s * e1.x, jp.c * b11.y - jp.s * e1.y);
                        const cd n21 = make_double2(jp.s * b11.x + jp.c * e1.x, jp.s * b11.y + jp.c * e1.y);
                        const cd n12 = make_double2(jp.c * b12.x - jp.s * e2.x, jp.c * b12.y - jp.s * e2.y);
                        const cd n22 = make_double2(jp.s * b12.x + jp.c * e2.x, jp.s * b12.y + jp.c * e2.y);
                        b11 = n11; b21 = n21; b12 = n12; b22 = n22;
                    }
                    __stcg(nxt + (size_t)p * n + cr, b11);
                    if (sv) __stcg(nxt + (size_t)p * n + cs, b12);
                    if (qv) __stcg(nxt + (size_t)q * n + cr, b21);
                    if (qv && sv) __stcg(nxt + (size_t)q * n + cs, b22);
                }
                if (v_on) {
                    const cd ey = make_double2(vy.x * jv.cph + vy.y * jv.sph, vy.y * jv.cph - vy.x * jv.sph);   // e^{-i phi} y
                    __stcg(v + (size_t)vrow * n + vp, make_double2(jv.c * vx.x - jv.s * ey.x, jv.c * vx.y - jv.s * ey.y));
                    __stcg(v + (size_t)vrow * n + vq, make_double2(jv.s * vx.x + jv.c * ey.x, jv.s * vx.y + jv.c * ey.y));
                }
            }
            grid_barrier();
            cd* t = cur; cur = nxt; nxt = t;
        }
        // ---- end of the sweep: every CTA holds the same maximum (each computed every rotation)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tmax = fmax(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
        if ((tid & 31) == 0) red[tid >> 5] = tmax;
        __syncthreads();
        double big = 0.0;
        for (int w = 0; w < JACOBI_T / 32; ++w) big = fmax(big, red[w]);
        __syncthreads();
        converged = big <= thr;                              // no element above the threshold was met in this sweep
    }
    // the eigenvalues are read from the diagonal of `a`
    if (cur != a) {
        for (size_t i = gtid; i < (size_t)n; i += gsize) a[i * n + i] = __ldcg(cur + i * n + i);
    }
    if (gtid == 0) { ctl[4] = (unsigned)sweep; ctl[5] = converged ? 0u : 1u; }
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
