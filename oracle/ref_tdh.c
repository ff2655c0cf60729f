/*
 * ref_tdh.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, literal implementation of what the hot path computes, written from the paper
 * (arXiv:2106.03872, /root/reference/PAPER.md) and the readings listed in DESIGN.md.  It shares no
 * code, header, table or helper with the CUDA path (paper_2106_03872_b200/csrc) and neither side
 * includes or imports the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.
 *
 * What is computed (complex128 throughout; long double only for twiddle tables):
 *
 *   H psi = T psi + V psi + V_nl psi                                  Eq. 2
 *     T psi    = DFT^-1( [t <= E_cut] * t * DFT(psi) ),  t = 1/2 |G + k|^2   PAPER.md:480 ("calculated in
 *                Fourier space, where it is diagonal"); readings R1, R6, R7, R8
 *     V psi    = V(r) psi(r)                                           PAPER.md:480,488 (diagonal in real space)
 *     V_nl psi = sum_I sum_c beta_Ic(r-R_I) D_Ic dV sum_{r' in sphere} beta_Ic(r'-R_I) psi(r')
 *                                                                      Eq. 9; readings R2-R5
 *   exp(-i dt H) psi ~= sum_{k=0..4} (-i dt)^k / k!  H^k psi           Eq. 8
 *   ETRS step (Eq. 6-7) from two such sums sharing H^k psi, V(t+dt) supplied
 *   n(r) = sum_s f_s |psi_s(r)|^2  (Eq. 1);  v_H from the periodic Poisson equation in Fourier space
 *
 * Two DFT back-ends: backend 0 = direct O(N^2)-per-pencil sum (the definition), backend 1 = a separately
 * written recursive radix-2/3 decimation-in-time FFT (only to make the large configs affordable; it is
 * accepted in tests by matching backend 0).  Everything else is literal loops in the paper's order.
 *
 * Pins (tests/test_oracle_pins.py): P1 brute-force 3-D DFT / round trip / Parseval, P2 plane waves are
 * kinetic eigenvectors incl. Nyquist and mask, P3 constant potential = shift, P4 rank / closed form of one
 * projector, P5 Hermiticity and dense-matrix spectrum, P6 Bloch-phase identity and translation covariance,
 * P7 closed-form Taylor propagation of kinetic-only H, P8 independence of batching, P9 ETRS against dense
 * matrix polynomials and the kinetic-only closed form, P10 density / Poisson closed forms, P11 overlap matrix.  The paper prints no
 * worked H.psi example, so beyond P1-P8 parity is unpinned by the paper (stated in DESIGN.md).
 *
 * Build: gcc -O2 -std=c99 -fopenmp -shared -fPIC ref_tdh.c -o libref_tdh.so -lm   (oracle/build.py)
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define REF_OK 0
#define REF_EINVAL (-1)
#define REF_ENOMEM (-3)

/* ------------------------------------------------------------------------------------------------
 * 1-D transforms along one pencil.  sign = -1 forward, +1 inverse (unnormalised here).  Reading R8.
 * w[m] = exp(sign * 2 pi i m / N), m = 0..N-1, built in long double.
 * ------------------------------------------------------------------------------------------------ */
static cplx *make_twiddles(int n, int sign)
{
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!w) return NULL;
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int m = 0; m < n; ++m) {
        long double a = two_pi * (long double)m / (long double)n;
        w[m] = (double)cosl(a) + I * (double)(sign * sinl(a));
    }
    return w;
}

/* Direct DFT: out[q] = sum_j in[j] * w[(q*j) mod n].  The definition. */
static void dft_direct(int n, const cplx *in, cplx *out, const cplx *w)
{
    for (int q = 0; q < n; ++q) {
        cplx acc = 0.0;
        for (int j = 0; j < n; ++j) acc += in[j] * w[(int)(((long long)q * j) % n)];
        out[q] = acc;
    }
}

/* Recursive decimation-in-time FFT for n = 2^a 3^b (other factors fall through to the direct sum).
 * in has stride `is`; out is contiguous; w is the top-level table of length ntop, ws = ntop / n. */
static void fft_rec(int n, const cplx *in, int is, cplx *out, const cplx *w, int ntop)
{
    const int ws = ntop / n;
    if (n == 1) { out[0] = in[0]; return; }
    if (n % 2 == 0) {
        const int m = n / 2;
        fft_rec(m, in, 2 * is, out, w, ntop);           /* even samples */
        fft_rec(m, in + is, 2 * is, out + m, w, ntop);  /* odd samples  */
        for (int q = 0; q < m; ++q) {
            cplx e = out[q], o = w[q * ws] * out[m + q];
            out[q] = e + o;
            out[m + q] = e - o;                          /* w^(q+m) = -w^q */
        }
        return;
    }
    if (n % 3 == 0) {
        const int m = n / 3;
        fft_rec(m, in, 3 * is, out, w, ntop);
        fft_rec(m, in + is, 3 * is, out + m, w, ntop);
        fft_rec(m, in + 2 * is, 3 * is, out + 2 * m, w, ntop);
        const cplx c1 = w[m * ws], c2 = w[2 * m * ws];   /* primitive cube roots exp(sign 2 pi i /3), ^2 */
        for (int q = 0; q < m; ++q) {
            cplx a = out[q];
            cplx b = w[q * ws] * out[m + q];
            cplx c = w[(2 * q) * ws] * out[2 * m + q];
            out[q] = a + b + c;
            out[m + q] = a + c1 * b + c2 * c;
            out[2 * m + q] = a + c2 * b + c1 * c;        /* (c1^2 = c2, c2^2 = c1) */
        }
        return;
    }
    /* generic prime factor: direct sum with the strided input */
    for (int q = 0; q < n; ++q) {
        cplx acc = 0.0;
        for (int j = 0; j < n; ++j) acc += in[(size_t)j * is] * w[(int)((((long long)q * j) % n) * ws)];
        out[q] = acc;
    }
}

/* In-place 3-D DFT of one state: three sets of 1-D transforms, axis z, then y, then x (PAPER.md:450:
 * "A 3D FFT is calculated as a sequence of 1D FFTs in each direction").  Inverse scaled by 1/N per axis. */
static int dft3d_one(const int n[3], cplx *a, int sign, int backend)
{
    const size_t stride[3] = {(size_t)n[1] * n[2], (size_t)n[2], 1};
    int nmax = n[0] > n[1] ? n[0] : n[1];
    if (n[2] > nmax) nmax = n[2];
    cplx *tin = (cplx *)malloc(sizeof(cplx) * (size_t)nmax);
    cplx *tout = (cplx *)malloc(sizeof(cplx) * (size_t)nmax);
    if (!tin || !tout) { free(tin); free(tout); return REF_ENOMEM; }
    for (int ax = 2; ax >= 0; --ax) {
        const int len = n[ax];
        cplx *w = make_twiddles(len, sign);
        if (!w) { free(tin); free(tout); return REF_ENOMEM; }
        const int a1 = (ax + 1) % 3, a2 = (ax + 2) % 3;
        const double scale = sign > 0 ? 1.0 / (double)len : 1.0;
        for (int i1 = 0; i1 < n[a1]; ++i1)
            for (int i2 = 0; i2 < n[a2]; ++i2) {
                cplx *base = a + i1 * stride[a1] + i2 * stride[a2];
                for (int j = 0; j < len; ++j) tin[j] = base[j * stride[ax]];
                if (backend == 0) dft_direct(len, tin, tout, w);
                else fft_rec(len, tin, 1, tout, w, len);
                for (int j = 0; j < len; ++j) base[j * stride[ax]] = tout[j] * scale;
            }
        free(w);
    }
    free(tin);
    free(tout);
    return REF_OK;
}

/* Frequency index of array index a on an axis of n points: numpy fftfreq convention (reading R7). */
static int freq_index(int a, int n)
{
    if (n % 2 == 0) return a < n / 2 ? a : a - n;
    return a <= (n - 1) / 2 ? a : a - n;
}

static size_t npoints(const int n[3]) { return (size_t)n[0] * n[1] * n[2]; }

/* ------------------------------------------------------------------------------------------------
 * exported: 3-D DFT of a block of states, in place.
 * ------------------------------------------------------------------------------------------------ */
int ref_dft3d(const int n[3], int nst, cplx *a, int sign, int backend)
{
    if (!n || !a || nst < 0 || (sign != 1 && sign != -1)) return REF_EINVAL;
    const size_t np_ = npoints(n);
    int err = REF_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        int e = dft3d_one(n, a + (size_t)s * np_, sign, backend);
        if (e != REF_OK) {
#pragma omp critical
            err = e;
        }
    }
    return err;
}

/* ------------------------------------------------------------------------------------------------
 * Kinetic term of one state, added into out:  out += DFT^-1( mask * t * DFT(psi) ).
 *   t[n] = 1/2 sum_a (G_a[n_a] + k_a)^2,  G_a = 2 pi m(a) / L_a;  mask = [t <= ecut] (ecut <= 0: none).
 * Eq. 2 first term.
 * ------------------------------------------------------------------------------------------------ */
static int kinetic_one(const int n[3], const double len[3], const double kpt[3], double ecut,
                       const cplx *psi, cplx *out, int backend)
{
    const size_t np_ = npoints(n);
    const double two_pi = 6.283185307179586476925286766559;
    cplx *f = (cplx *)malloc(sizeof(cplx) * np_);
    if (!f) return REF_ENOMEM;
    memcpy(f, psi, sizeof(cplx) * np_);
    int e = dft3d_one(n, f, -1, backend);
    if (e != REF_OK) { free(f); return e; }
    const int use_mask = (ecut > 0.0) && isfinite(ecut);
    for (int ix = 0; ix < n[0]; ++ix) {
        const double gx = two_pi * freq_index(ix, n[0]) / len[0] + kpt[0];
        for (int iy = 0; iy < n[1]; ++iy) {
            const double gy = two_pi * freq_index(iy, n[1]) / len[1] + kpt[1];
            for (int iz = 0; iz < n[2]; ++iz) {
                const double gz = two_pi * freq_index(iz, n[2]) / len[2] + kpt[2];
                const double t = 0.5 * (gx * gx + gy * gy + gz * gz);
                const size_t p = ((size_t)ix * n[1] + iy) * n[2] + iz;
                if (use_mask && !(t <= ecut)) f[p] = 0.0;
                else f[p] *= t;
            }
        }
    }
    e = dft3d_one(n, f, +1, backend);
    if (e == REF_OK)
        for (size_t p = 0; p < np_; ++p) out[p] += f[p];
    free(f);
    return e;
}

/* Local term of one state, added into out: out[p] += V[p] psi[p].  PAPER.md:480,488. */
static void local_one(size_t np_, const double *v, const cplx *psi, cplx *out)
{
    if (!v) return;
    for (size_t p = 0; p < np_; ++p) out[p] += v[p] * psi[p];
}

/* Non-local term of one state, added into out.  Eq. 9 as the Riemann sum of row a5:
 *   pi_{I,c}  = dV sum_q beta_{I,c}[q] e^{+i k.d_I[q]} psi[S_I[q]]
 *   out[S_I[q]] += e^{-i k.d_I[q]} sum_c beta_{I,c}[q] D_{I,c} pi_{I,c}
 * loops atoms -> channels -> sphere points, projection accumulated in a scalar, then a second loop. */
static void nonlocal_one(double dv, const double kpt[3], int natoms, const int64_t *sph_off, const int32_t *sph_idx,
                         const double *sph_disp, const int32_t *chan_off, const double *beta, const double *dcoef,
                         const cplx *psi, cplx *out)
{
    const int have_k = sph_disp && (kpt[0] != 0.0 || kpt[1] != 0.0 || kpt[2] != 0.0);
    size_t boff = 0; /* start of atom I's [C_I][P_I] block in beta */
    for (int ia = 0; ia < natoms; ++ia) {
        const int64_t q0 = sph_off[ia], q1 = sph_off[ia + 1];
        const int64_t pn = q1 - q0;
        const int c0 = chan_off[ia], c1 = chan_off[ia + 1];
        for (int c = c0; c < c1; ++c) {
            const double *b = beta + boff + (size_t)(c - c0) * (size_t)pn;
            cplx proj = 0.0;
            for (int64_t q = 0; q < pn; ++q) {
                cplx ph = 1.0;
                if (have_k) {
                    const double *d = sph_disp + 3 * (q0 + q);
                    const double arg = kpt[0] * d[0] + kpt[1] * d[1] + kpt[2] * d[2];
                    ph = cos(arg) + I * sin(arg);
                }
                proj += b[q] * ph * psi[sph_idx[q0 + q]];
            }
            proj *= dv;
            const cplx coef = dcoef[c] * proj;
            for (int64_t q = 0; q < pn; ++q) {
                cplx ph = 1.0;
                if (have_k) {
                    const double *d = sph_disp + 3 * (q0 + q);
                    const double arg = kpt[0] * d[0] + kpt[1] * d[1] + kpt[2] * d[2];
                    ph = cos(arg) - I * sin(arg);
                }
                out[sph_idx[q0 + q]] += ph * (b[q] * coef);
            }
        }
        boff += (size_t)(c1 - c0) * (size_t)pn;
    }
}

static int check_geometry(const int n[3], const double len[3])
{
    if (!n || !len) return REF_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (n[a] < 1 || !(len[a] > 0.0)) return REF_EINVAL;
    return REF_OK;
}

/* ------------------------------------------------------------------------------------------------
 * exported: the three terms separately (for the pins) -- each OVERWRITES out.
 * ------------------------------------------------------------------------------------------------ */
int ref_kinetic(const int n[3], const double len[3], const double kpt[3], double ecut, int nst, const cplx *psi,
                cplx *out, int backend)
{
    if (check_geometry(n, len) || !kpt || !psi || !out || nst < 0) return REF_EINVAL;
    const size_t np_ = npoints(n);
    int err = REF_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        memset(out + (size_t)s * np_, 0, sizeof(cplx) * np_);
        int e = kinetic_one(n, len, kpt, ecut, psi + (size_t)s * np_, out + (size_t)s * np_, backend);
        if (e != REF_OK) {
#pragma omp critical
            err = e;
        }
    }
    return err;
}

int ref_local(const int n[3], const double *v, int nst, const cplx *psi, cplx *out)
{
    if (!n || !psi || !out || nst < 0) return REF_EINVAL;
    const size_t np_ = npoints(n);
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        memset(out + (size_t)s * np_, 0, sizeof(cplx) * np_);
        local_one(np_, v, psi + (size_t)s * np_, out + (size_t)s * np_);
    }
    return REF_OK;
}

static int check_projectors(const int n[3], int natoms, const int64_t *sph_off, const int32_t *sph_idx,
                            const int32_t *chan_off, const double *beta, const double *dcoef)
{
    if (natoms < 0) return REF_EINVAL;
    if (natoms == 0) return REF_OK;
    if (!sph_off || !sph_idx || !chan_off || !beta || !dcoef) return REF_EINVAL;
    const size_t np_ = npoints(n);
    for (int64_t q = sph_off[0]; q < sph_off[natoms]; ++q)
        if (sph_idx[q] < 0 || (size_t)sph_idx[q] >= np_) return REF_EINVAL;
    return REF_OK;
}

int ref_nonlocal(const int n[3], const double len[3], const double kpt[3], int natoms, const int64_t *sph_off,
                 const int32_t *sph_idx, const double *sph_disp, const int32_t *chan_off, const double *beta,
                 const double *dcoef, int nst, const cplx *psi, cplx *out)
{
    if (check_geometry(n, len) || !kpt || !psi || !out || nst < 0) return REF_EINVAL;
    if (check_projectors(n, natoms, sph_off, sph_idx, chan_off, beta, dcoef)) return REF_EINVAL;
    const size_t np_ = npoints(n);
    const double dv = (len[0] / n[0]) * (len[1] / n[1]) * (len[2] / n[2]);
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        memset(out + (size_t)s * np_, 0, sizeof(cplx) * np_);
        nonlocal_one(dv, kpt, natoms, sph_off, sph_idx, sph_disp, chan_off, beta, dcoef, psi + (size_t)s * np_,
                     out + (size_t)s * np_);
    }
    return REF_OK;
}

/* H applied to one state: every term is computed from the INPUT psi. */
static int hamiltonian_one(const int n[3], const double len[3], const double kpt[3], double ecut, const double *v,
                           int natoms, const int64_t *sph_off, const int32_t *sph_idx, const double *sph_disp,
                           const int32_t *chan_off, const double *beta, const double *dcoef, const cplx *psi,
                           cplx *hpsi, int backend)
{
    const size_t np_ = npoints(n);
    const double dv = (len[0] / n[0]) * (len[1] / n[1]) * (len[2] / n[2]);
    memset(hpsi, 0, sizeof(cplx) * np_);
    int e = kinetic_one(n, len, kpt, ecut, psi, hpsi, backend);
    if (e != REF_OK) return e;
    local_one(np_, v, psi, hpsi);
    nonlocal_one(dv, kpt, natoms, sph_off, sph_idx, sph_disp, chan_off, beta, dcoef, psi, hpsi);
    return REF_OK;
}

/* ------------------------------------------------------------------------------------------------
 * exported: H psi for a block (Eq. 2; "a routine that applies the Hamiltonian over a field set",
 * PAPER.md:478).  v may be NULL (V = 0); natoms may be 0.
 * ------------------------------------------------------------------------------------------------ */
int ref_apply_hamiltonian(const int n[3], const double len[3], const double kpt[3], double ecut, const double *v,
                          int natoms, const int64_t *sph_off, const int32_t *sph_idx, const double *sph_disp,
                          const int32_t *chan_off, const double *beta, const double *dcoef, int nst, const cplx *psi,
                          cplx *hpsi, int backend)
{
    if (check_geometry(n, len) || !kpt || !psi || !hpsi || nst < 0) return REF_EINVAL;
    if (check_projectors(n, natoms, sph_off, sph_idx, chan_off, beta, dcoef)) return REF_EINVAL;
    const size_t np_ = npoints(n);
    int err = REF_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        int e = hamiltonian_one(n, len, kpt, ecut, v, natoms, sph_off, sph_idx, sph_disp, chan_off, beta, dcoef,
                                psi + (size_t)s * np_, hpsi + (size_t)s * np_, backend);
        if (e != REF_OK) {
#pragma omp critical
            err = e;
        }
    }
    return err;
}

/* ------------------------------------------------------------------------------------------------
 * exported: nsteps Taylor steps, psi in place, H fixed (reading R10, R16).  Eq. 8 with lambda = -i dt:
 *   acc = psi; phi_0 = psi; for k = 1..order: phi_k = H phi_{k-1}; acc += (-i dt)^k / k! phi_k; psi <- acc.
 * order 4: c1 = -i dt, c2 = -dt^2/2, c3 = +i dt^3/6, c4 = +dt^4/24.
 * ------------------------------------------------------------------------------------------------ */
int ref_propagate(const int n[3], const double len[3], const double kpt[3], double ecut, const double *v, int natoms,
                  const int64_t *sph_off, const int32_t *sph_idx, const double *sph_disp, const int32_t *chan_off,
                  const double *beta, const double *dcoef, int nst, cplx *psi, double dt, int nsteps, int order,
                  int backend)
{
    if (check_geometry(n, len) || !kpt || !psi || nst < 0 || nsteps < 0 || order < 1 || order > 16) return REF_EINVAL;
    if (check_projectors(n, natoms, sph_off, sph_idx, chan_off, beta, dcoef)) return REF_EINVAL;
    const size_t np_ = npoints(n);
    int err = REF_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        cplx *x = psi + (size_t)s * np_;
        cplx *phi = (cplx *)malloc(sizeof(cplx) * np_);
        cplx *hphi = (cplx *)malloc(sizeof(cplx) * np_);
        int e = (phi && hphi) ? REF_OK : REF_ENOMEM;
        for (int step = 0; step < nsteps && e == REF_OK; ++step) {
            memcpy(phi, x, sizeof(cplx) * np_); /* phi_0 = psi; x plays the role of acc (= psi initially) */
            cplx coef = 1.0;
            for (int k = 1; k <= order && e == REF_OK; ++k) {
                e = hamiltonian_one(n, len, kpt, ecut, v, natoms, sph_off, sph_idx, sph_disp, chan_off, beta, dcoef,
                                    phi, hphi, backend);
                coef *= (-I * dt) / (double)k; /* (-i dt)^k / k! */
                for (size_t p = 0; p < np_; ++p) x[p] += coef * hphi[p];
                cplx *t = phi; phi = hphi; hphi = t;
            }
        }
        free(phi);
        free(hphi);
        if (e != REF_OK) {
#pragma omp critical
            err = e;
        }
    }
    return err;
}

/* ------------------------------------------------------------------------------------------------
 * exported (NEXT-1): the two exponentials of one ETRS step that share their powers H^k psi.
 * "we can evaluate this expression for several values of lambda for almost the same cost
 * of a single value, since lambda only appears as a multiplicative coefficient".  Eq. 8 for
 * lambda_1 = -i dt/2 and lambda_2 = -i dt, literally:
 *   half = full = psi;  phi_0 = psi;  for k = 1..order:  phi_k = H phi_{k-1};
 *       half += (-i dt/2)^k / k! phi_k;   full += (-i dt)^k / k! phi_k.
 * psi is not modified.
 * ------------------------------------------------------------------------------------------------ */
int ref_taylor_pair(const int n[3], const double len[3], const double kpt[3], double ecut, const double *v, int natoms,
                    const int64_t *sph_off, const int32_t *sph_idx, const double *sph_disp, const int32_t *chan_off,
                    const double *beta, const double *dcoef, int nst, const cplx *psi, cplx *half, cplx *full, double dt,
                    int order, int backend)
{
    if (check_geometry(n, len) || !kpt || !psi || !half || !full || nst < 0 || order < 1 || order > 16) return REF_EINVAL;
    if (check_projectors(n, natoms, sph_off, sph_idx, chan_off, beta, dcoef)) return REF_EINVAL;
    const size_t np_ = npoints(n);
    int err = REF_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        const cplx *x = psi + (size_t)s * np_;
        cplx *h = half + (size_t)s * np_, *f = full + (size_t)s * np_;
        cplx *phi = (cplx *)malloc(sizeof(cplx) * np_);
        cplx *hphi = (cplx *)malloc(sizeof(cplx) * np_);
        int e = (phi && hphi) ? REF_OK : REF_ENOMEM;
        if (e == REF_OK) {
            memcpy(phi, x, sizeof(cplx) * np_);
            memcpy(h, x, sizeof(cplx) * np_);
            memcpy(f, x, sizeof(cplx) * np_);
        }
        cplx ch = 1.0, cf = 1.0;
        for (int k = 1; k <= order && e == REF_OK; ++k) {
            e = hamiltonian_one(n, len, kpt, ecut, v, natoms, sph_off, sph_idx, sph_disp, chan_off, beta, dcoef, phi, hphi,
                                backend);
            ch *= (-I * (0.5 * dt)) / (double)k; /* (-i dt/2)^k / k! */
            cf *= (-I * dt) / (double)k;         /* (-i dt)^k / k!   */
            for (size_t p = 0; p < np_; ++p) {
                h[p] += ch * hphi[p];
                f[p] += cf * hphi[p];
            }
            cplx *t = phi; phi = hphi; hphi = t;
        }
        free(phi);
        free(hphi);
        if (e != REF_OK) {
#pragma omp critical
            err = e;
        }
    }
    return err;
}

/* ------------------------------------------------------------------------------------------------
 * exported (NEXT-1): one ETRS step, Eq. 6-7, with the potential at t+dt supplied by the
 * caller (the density -> potential map needs the XC functional, which is outside this path):
 *   approx = exp(-i dt H(t)) psi          Eq. 7  (returned; the caller derives V(t+dt) from it BEFORE calling
 *                                                 when V(t+dt) depends on it -- here v_next is an input)
 *   psi   <- exp(-i dt/2 H(t+dt)) exp(-i dt/2 H(t)) psi        Eq. 6
 * Every exponential is the order-4 Taylor sum of Eq. 8.  H(t) uses v, H(t+dt) uses v_next; the projectors
 * are the same in both (fixed ions).  approx may be NULL.
 * ------------------------------------------------------------------------------------------------ */
int ref_etrs_step(const int n[3], const double len[3], const double kpt[3], double ecut, const double *v,
                  const double *v_next, int natoms, const int64_t *sph_off, const int32_t *sph_idx, const double *sph_disp,
                  const int32_t *chan_off, const double *beta, const double *dcoef, int nst, cplx *psi, cplx *approx,
                  double dt, int backend)
{
    if (!psi || nst < 0) return REF_EINVAL;
    const size_t np_ = npoints(n);
    cplx *half = (cplx *)malloc(sizeof(cplx) * np_ * (size_t)(nst > 0 ? nst : 1));
    cplx *full = approx ? approx : (cplx *)malloc(sizeof(cplx) * np_ * (size_t)(nst > 0 ? nst : 1));
    int e = (half && full) ? REF_OK : REF_ENOMEM;
    if (e == REF_OK)
        e = ref_taylor_pair(n, len, kpt, ecut, v, natoms, sph_off, sph_idx, sph_disp, chan_off, beta, dcoef, nst, psi, half,
                            full, dt, 4, backend);
    if (e == REF_OK) {
        memcpy(psi, half, sizeof(cplx) * np_ * (size_t)nst);
        e = ref_propagate(n, len, kpt, ecut, v_next, natoms, sph_off, sph_idx, sph_disp, chan_off, beta, dcoef, nst, psi,
                          0.5 * dt, 1, 4, backend);
    }
    free(half);
    if (!approx) free(full);
    return e;
}

/* ------------------------------------------------------------------------------------------------
 * exported (NEXT-2): the density, Eq. 1:  n(r) = sum_k |phi_k(r)|^2, here with optional
 * occupations f_s (occ == NULL: all 1, Eq. 1 as printed).  "trivially parallelizable in RS points but requires a
 * parallel reduction over states": literal loop over points, inner loop over states in order.
 * accumulate != 0 adds to dens (partial sums of a block processed in pieces / shards).
 * ------------------------------------------------------------------------------------------------ */
int ref_density(const int n[3], int nst, const cplx *psi, const double *occ, double *dens, int accumulate)
{
    if (!n || !psi || !dens || nst < 0) return REF_EINVAL;
    const size_t np_ = npoints(n);
#pragma omp parallel for schedule(static)
    for (long long p = 0; p < (long long)np_; ++p) {
        double acc = accumulate ? dens[p] : 0.0;
        for (int s = 0; s < nst; ++s) {
            const cplx z = psi[(size_t)s * np_ + (size_t)p];
            const double a = creal(z) * creal(z) + cimag(z) * cimag(z);
            acc += (occ ? occ[s] : 1.0) * a;
        }
        dens[p] = acc;
    }
    return REF_OK;
}

/* ------------------------------------------------------------------------------------------------
 * exported (NEXT-2): Hartree potential of a periodic density, PAPER.md:504 ("We solve the equation in FS, where the
 * Poisson equation becomes a simple algebraic equation ... two FFTs are needed to go to FS and back"):
 *   nabla^2 v = -4 pi n   =>   v_hat(G) = 4 pi n_hat(G) / |G|^2  for G != 0,   v_hat(0) = 0
 * (the G = 0 component of a periodic charge is compensated by the ionic background; periodic boundary conditions
 * only -- the paper's free-boundary kernel is out of scope).  G_a = 2 pi m(a) / L_a with the frequency convention R7;
 * no Bloch vector enters: the density is periodic.  The result is the real part of the inverse transform.
 * ------------------------------------------------------------------------------------------------ */
int ref_hartree(const int n[3], const double len[3], const double *dens, double *vh, int backend)
{
    if (check_geometry(n, len) || !dens || !vh) return REF_EINVAL;
    const size_t np_ = npoints(n);
    const double two_pi = 6.283185307179586476925286766559;
    cplx *a = (cplx *)malloc(sizeof(cplx) * np_);
    if (!a) return REF_ENOMEM;
    for (size_t p = 0; p < np_; ++p) a[p] = dens[p];
    int e = dft3d_one(n, a, -1, backend);
    if (e == REF_OK) {
        for (int i = 0; i < n[0]; ++i) {
            const double gx = two_pi * freq_index(i, n[0]) / len[0];
            for (int j = 0; j < n[1]; ++j) {
                const double gy = two_pi * freq_index(j, n[1]) / len[1];
                for (int k = 0; k < n[2]; ++k) {
                    const double gz = two_pi * freq_index(k, n[2]) / len[2];
                    const double g2 = (gx * gx + gy * gy) + gz * gz;
                    const size_t p = ((size_t)i * n[1] + j) * n[2] + k;
                    a[p] = (g2 > 0.0) ? a[p] * (2.0 * two_pi / g2) : 0.0;
                }
            }
        }
        e = dft3d_one(n, a, +1, backend);
    }
    if (e == REF_OK)
        for (size_t p = 0; p < np_; ++p) vh[p] = creal(a[p]);
    free(a);
    return e;
}

/* ------------------------------------------------------------------------------------------------
 * exported (first building block of NEXT-3): overlap / subspace matrix of two state blocks,
 *   S[i][j] = <a_i | b_j> = dV sum_p conj(a_i[p]) b_j[p],   i < na, j < nb   (row-major [na][nb])
 * -- the matrix behind "orthogonalization and subspace diagonalization" ("rotations in the space of
 * eigenvectors ... dominated by linear algebra operations") and behind the statement that real-time propagation
 * "conserves orthogonality of the KS states mathematically and also numerically".  Literal loops.
 * ------------------------------------------------------------------------------------------------ */
int ref_overlap(const int n[3], double dv, int na, const cplx *a, int nb, const cplx *b, cplx *s)
{
    if (!n || !a || !b || !s || na < 0 || nb < 0) return REF_EINVAL;
    const size_t np_ = npoints(n);
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < na; ++i)
        for (int j = 0; j < nb; ++j) {
            cplx acc = 0.0;
            for (size_t p = 0; p < np_; ++p) acc += conj(a[(size_t)i * np_ + p]) * b[(size_t)j * np_ + p];
            s[(size_t)i * nb + j] = dv * acc;
        }
    return REF_OK;
}

/* ------------------------------------------------------------------------------------------------
 * exported (NEXT-3): one preconditioned steepest-descent update of every state, independently ("the
 * preconditioned steepest (SD) descent algorithm ... can work simultaneously and independently on all eigenvectors.
 * For preconditioning we use the method of Teter et al. that is applied in Fourier space").  The paper gives no
 * formulas; the reading (R19) is the textbook one:
 *   eps_s = <psi|H psi> / <psi|psi>,   T_s = <psi|T psi> / <psi|psi>       (sums over grid points, dV cancels)
 *   r = H psi - eps_s psi
 *   p_hat(G) = K(x) r_hat(G),  x = t(G) / T_s,  t = 1/2 |G+k|^2,
 *       K(x) = (27 + 18x + 12x^2 + 8x^3) / (27 + 18x + 12x^2 + 8x^3 + 16x^4)         (Teter, Payne, Allan 1989)
 *   psi <- psi - lambda p                                             (fixed step; no orthogonalisation here)
 * eig[s] receives eps_s (the Rayleigh quotient BEFORE the update).  The cutoff mask acts in T as in H.
 * ------------------------------------------------------------------------------------------------ */
static double teter(double x)
{
    const double num = 27.0 + x * (18.0 + x * (12.0 + x * 8.0));
    return num / (num + 16.0 * x * x * x * x);
}

int ref_sd_step(const int n[3], const double len[3], const double kpt[3], double ecut, const double *v, int natoms,
                const int64_t *sph_off, const int32_t *sph_idx, const double *sph_disp, const int32_t *chan_off,
                const double *beta, const double *dcoef, int nst, cplx *psi, double lambda, double *eig, int backend)
{
    if (check_geometry(n, len) || !kpt || !psi || nst < 0) return REF_EINVAL;
    if (check_projectors(n, natoms, sph_off, sph_idx, chan_off, beta, dcoef)) return REF_EINVAL;
    const size_t np_ = npoints(n);
    const double two_pi = 6.283185307179586476925286766559;
    int err = REF_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        cplx *x = psi + (size_t)s * np_;
        cplx *h = (cplx *)malloc(sizeof(cplx) * np_);
        cplx *t = (cplx *)calloc(np_, sizeof(cplx));
        int e = (h && t) ? REF_OK : REF_ENOMEM;
        if (e == REF_OK)
            e = hamiltonian_one(n, len, kpt, ecut, v, natoms, sph_off, sph_idx, sph_disp, chan_off, beta, dcoef, x, h, backend);
        if (e == REF_OK) e = kinetic_one(n, len, kpt, ecut, x, t, backend);          /* t += T psi (t was zero) */
        if (e == REF_OK) {
            double nn = 0.0, eh = 0.0, et = 0.0;
            for (size_t p = 0; p < np_; ++p) {
                nn += creal(x[p]) * creal(x[p]) + cimag(x[p]) * cimag(x[p]);
                eh += creal(conj(x[p]) * h[p]);
                et += creal(conj(x[p]) * t[p]);
            }
            const double eps = eh / nn, ts = et / nn;
            if (eig) eig[s] = eps;
            for (size_t p = 0; p < np_; ++p) h[p] -= eps * x[p];                    /* residual */
            e = dft3d_one(n, h, -1, backend);
            if (e == REF_OK) {
                for (int i = 0; i < n[0]; ++i) {
                    const double gx = two_pi * freq_index(i, n[0]) / len[0] + kpt[0];
                    for (int j = 0; j < n[1]; ++j) {
                        const double gy = two_pi * freq_index(j, n[1]) / len[1] + kpt[1];
                        for (int k = 0; k < n[2]; ++k) {
                            const double gz = two_pi * freq_index(k, n[2]) / len[2] + kpt[2];
                            const double tk = 0.5 * ((gx * gx + gy * gy) + gz * gz);
                            /* T_s <= 0 (a constant state at Gamma, up to rounding): x = t / T_s is undefined; reading
                             * R19 takes the limit x -> infinity: K = 1 at t = 0, K = 0 elsewhere */
                            h[((size_t)i * n[1] + j) * n[2] + k] *= ts > 0.0 ? teter(tk / ts) : (tk == 0.0 ? 1.0 : 0.0);
                        }
                    }
                }
                e = dft3d_one(n, h, +1, backend);
            }
            if (e == REF_OK)
                for (size_t p = 0; p < np_; ++p) x[p] -= lambda * h[p];
        }
        free(h);
        free(t);
        if (e != REF_OK) {
#pragma omp critical
            err = e;
        }
    }
    return err;
}

/* ------------------------------------------------------------------------------------------------
 * exported (NEXT-4): gradient of a block, "just like the Laplacian, a local operation in Fourier space":
 *   (d_a psi)[p] = DFT^-1( i (G_a + k_a) DFT(psi) ),  a = axis (0, 1, 2);  frequencies as in the kinetic term (R7), no mask.
 * ------------------------------------------------------------------------------------------------ */
static int gradient_one(const int n[3], const double len[3], const double kpt[3], int axis, const cplx *psi, cplx *out,
                        int backend)
{
    const size_t np_ = npoints(n);
    const double two_pi = 6.283185307179586476925286766559;
    memcpy(out, psi, sizeof(cplx) * np_);
    int e = dft3d_one(n, out, -1, backend);
    if (e != REF_OK) return e;
    for (int i = 0; i < n[0]; ++i)
        for (int j = 0; j < n[1]; ++j)
            for (int k = 0; k < n[2]; ++k) {
                const int idx[3] = {i, j, k};
                const double ga = two_pi * freq_index(idx[axis], n[axis]) / len[axis] + kpt[axis];
                out[((size_t)i * n[1] + j) * n[2] + k] *= I * ga;
            }
    return dft3d_one(n, out, +1, backend);
}

int ref_gradient(const int n[3], const double len[3], const double kpt[3], int axis, int nst, const cplx *psi, cplx *out,
                 int backend)
{
    if (check_geometry(n, len) || !kpt || !psi || !out || nst < 0 || axis < 0 || axis > 2) return REF_EINVAL;
    const size_t np_ = npoints(n);
    int err = REF_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nst; ++s) {
        int e = gradient_one(n, len, kpt, axis, psi + (size_t)s * np_, out + (size_t)s * np_, backend);
        if (e != REF_OK) {
#pragma omp critical
            err = e;
        }
    }
    return err;
}

/* ------------------------------------------------------------------------------------------------
 * exported (NEXT-4): Eq. 11 literally, per atom I and axis a:
 *   F[I][a] = sum_s f_s ( <d_a psi_s | v_I | psi_s> + c.c. ) = sum_s f_s 2 Re( dV sum_p conj(d_a psi_s[p]) (v_I psi_s)[p] )
 * v_I = the Kleinman-Bylander projectors of atom I (Eq. 9 restricted to that atom) plus, when vloc_atoms != NULL, the
 * atom's own local potential vloc_atoms[I][p].  occ == NULL: all f_s = 1.  forces: [natoms][3].
 * ------------------------------------------------------------------------------------------------ */
int ref_forces(const int n[3], const double len[3], const double kpt[3], int natoms, const int64_t *sph_off,
               const int32_t *sph_idx, const double *sph_disp, const int32_t *chan_off, const double *beta,
               const double *dcoef, const double *vloc_atoms, int nst, const cplx *psi, const double *occ, double *forces,
               int backend)
{
    if (check_geometry(n, len) || !kpt || !psi || !forces || nst < 0 || natoms < 0) return REF_EINVAL;
    if (check_projectors(n, natoms, sph_off, sph_idx, chan_off, beta, dcoef)) return REF_EINVAL;
    const size_t np_ = npoints(n);
    const double dv = (len[0] / n[0]) * (len[1] / n[1]) * (len[2] / n[2]);
    for (int i = 0; i < 3 * natoms; ++i) forces[i] = 0.0;
    cplx *grad = (cplx *)malloc(sizeof(cplx) * np_);
    cplx *w = (cplx *)malloc(sizeof(cplx) * np_);
    int e = (grad && w) ? REF_OK : REF_ENOMEM;
    for (int s = 0; s < nst && e == REF_OK; ++s) {
        const cplx *x = psi + (size_t)s * np_;
        const double f = occ ? occ[s] : 1.0;
        for (int a = 0; a < 3 && e == REF_OK; ++a) {
            e = gradient_one(n, len, kpt, a, x, grad, backend);
            size_t boff = 0;
            for (int ia = 0; ia < natoms && e == REF_OK; ++ia) {
                const int64_t pn = sph_off[ia + 1] - sph_off[ia];
                const int nc = chan_off[ia + 1] - chan_off[ia];
                /* w = v_I psi: this atom's projectors (nonlocal_one on a one-atom table), plus its local potential */
                memset(w, 0, sizeof(cplx) * np_);
                const int64_t so[2] = {sph_off[ia], sph_off[ia + 1]};
                const int32_t co[2] = {chan_off[ia], chan_off[ia + 1]};
                nonlocal_one(dv, kpt, 1, so, sph_idx, sph_disp, co, beta + boff, dcoef, x, w);
                if (vloc_atoms)
                    for (size_t p = 0; p < np_; ++p) w[p] += vloc_atoms[(size_t)ia * np_ + p] * x[p];
                cplx acc = 0.0;
                for (size_t p = 0; p < np_; ++p) acc += conj(grad[p]) * w[p];
                forces[3 * ia + a] += f * 2.0 * creal(dv * acc);
                boff += (size_t)nc * (size_t)pn;
            }
        }
    }
    free(grad);
    free(w);
    return e;
}

/* number of OpenMP threads the block loops will use (reported by bench.py's cpu_baseline) */
int ref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
