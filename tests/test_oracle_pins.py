"""Pins P1-P8: the CPU oracle checked against what the mathematics fixes.

Nothing here calls the CUDA path.  Each pin compares the oracle with something it does not itself compute:
a brute-force triple sum, a closed form, an invariant, a library routine used as a third cross-check.
"""
import math

import numpy as np
from dataclasses import replace as dataclasses_replace
import pytest

from paper_2106_03872_b200 import workloads as W

TWO_PI = 2.0 * math.pi


def rand_c(rng, shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def small_cfg(cid=101, n=(6, 5, 4), length=(6.0, 5.5, 4.8), natoms=2, lmax=1, rc=1.9, **kw):
    kw.setdefault("dl", (1.5, -0.7, 0.4)[: lmax + 1])
    return W.test_config(cid, n, length, nst=3, natoms=natoms, lmax=lmax, rc=rc, proj_sigma=0.6,
                         well_z=2.0, well_sigma=0.8, noise=0.01, **kw)


def dense_matrix(oracle, cfg, wl, backend=0):
    """Columns H e_p, built by applying the oracle's H to unit vectors (PAPER.md:229 'dense Hermitian matrix')."""
    npts = cfg.npts
    eye = np.eye(npts, dtype=np.complex128).reshape((npts,) + tuple(cfg.n))
    cols = oracle.apply_hamiltonian(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, eye, backend)
    return cols.reshape(npts, npts).T.copy()   # H[:, p] = H e_p


# --------------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("n", [(4, 4, 4), (6, 6, 6), (8, 8, 8), (4, 6, 9), (5, 3, 2)])
@pytest.mark.parametrize("backend", [0, 1])
def test_p1_dft_bruteforce(oracle, n, backend):
    """3-D DFT = brute-force triple sum over all points (the textbook definition); round trip; Parseval."""
    rng = np.random.default_rng(11)
    a = rand_c(rng, (2,) + n)
    # brute force: out[q] = sum_p a[p] exp(-2 pi i (qx px/Nx + qy py/Ny + qz pz/Nz)), one 6-index phase tensor
    ph = [np.exp(-2j * np.pi * np.outer(np.arange(m), np.arange(m)) / m) for m in n]
    brute = np.einsum("sxyz,ax,by,cz->sabc", a, ph[0], ph[1], ph[2])
    f = oracle.dft3d(a, -1, backend)
    assert rel(f, brute) < 1e-13
    assert rel(f, np.fft.fftn(a, axes=(1, 2, 3))) < 1e-13            # library, third cross-check
    assert rel(oracle.dft3d(f, +1, backend), a) < 1e-13               # inverse carries 1/N_p
    npts = n[0] * n[1] * n[2]
    assert abs(np.sum(np.abs(f) ** 2) - npts * np.sum(np.abs(a) ** 2)) < 1e-11 * npts * np.sum(np.abs(a) ** 2)


@pytest.mark.parametrize("N", [16, 32, 48, 64, 96])
def test_p1_naive_fft_equals_direct_on_config_grids(oracle, N):
    """The naive radix-2/3 FFT back-end is accepted only because it equals the direct DFT on every grid size used."""
    rng = np.random.default_rng(N)
    a = rand_c(rng, (1, N, N, N))
    d = oracle.dft3d(a, -1, 0)
    f = oracle.dft3d(a, -1, 1)
    assert rel(f, d) < 1e-13
    assert rel(oracle.dft3d(a, +1, 1), oracle.dft3d(a, +1, 0)) < 1e-13


@pytest.mark.parametrize("L", [4, 6, 8, 9, 12, 18, 24, 27, 36, 54, 72, 81, 108, 128, 144, 162, 192, 243, 256])
def test_p1_naive_fft_equals_direct_on_every_axis_length_used_as_reference(oracle, L):
    """the naive FFT back-end is "accepted once it matches the direct DFT ... on every grid size used".
    The GPU tests use it as the reference on general grids too (tests/test_gpu_sizes.py, test_gpu_fullsize.py, smoke():
    lengths 9, 12, 24, 27, 36, 54, 72, 81, 128 and the thin grids with 4, 6, 8, 18, 108, 144, 162, 192, 243, 256), so
    every such length is checked here on each of the three axes of a thin grid, both directions."""
    rng = np.random.default_rng(1000 + L)
    for axis in range(3):
        n = [4, 6, 4]
        n[axis] = L
        a = rand_c(rng, (2,) + tuple(n))
        assert rel(oracle.dft3d(a, -1, 1), oracle.dft3d(a, -1, 0)) < 1e-13, (L, axis)
        assert rel(oracle.dft3d(a, +1, 1), oracle.dft3d(a, +1, 0)) < 1e-13, (L, axis)


@pytest.mark.parametrize("n", [(24, 36, 54), (72, 12, 9), (81, 27, 9), (128, 24, 16), (27, 27, 27), (54, 54, 54)])
def test_p1_naive_fft_equals_direct_on_mixed_general_grids(oracle, n):
    """The mixed general grids of the GPU parity tests, whole."""
    rng = np.random.default_rng(sum(n))
    a = rand_c(rng, (1,) + n)
    assert rel(oracle.dft3d(a, -1, 1), oracle.dft3d(a, -1, 0)) < 1e-13
    assert rel(oracle.dft3d(a, +1, 1), oracle.dft3d(a, +1, 0)) < 1e-13


def test_p1_delta_and_shift_theorem(oracle):
    """A unit impulse at r0 transforms to the plane wave exp(-i G.r0): fixes the sign and index convention."""
    n = (6, 4, 8)
    a = np.zeros(n, dtype=np.complex128)
    r0 = (2, 3, 5)
    a[r0] = 1.0
    f = oracle.dft3d(a, -1, 0)
    q = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
    expect = np.exp(-2j * np.pi * sum(q[i] * r0[i] / n[i] for i in range(3)))
    assert rel(f, expect) < 1e-14


# --------------------------------------------------------------------------------------------- P2
@pytest.mark.parametrize("n,kfrac,ecut", [((6, 4, 8), (0, 0, 0), None), ((6, 4, 8), (0.25, -0.4, 0.1), None),
                                          ((5, 6, 3), (0.3, 0.0, 0.2), 4.0), ((4, 4, 4), (0.25, 0.0, 0.0), 3.0)])
def test_p2_plane_waves_are_kinetic_eigenvectors(oracle, n, kfrac, ecut):
    """psi = exp(i G.r) for EVERY G of the grid (incl. Nyquist): T psi = 1/2 |G+k|^2 psi inside the mask, 0 outside."""
    length = (5.0, 4.0, 6.5)
    kpt = [TWO_PI * kfrac[a] / length[a] for a in range(3)]
    ii = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
    # signed frequency range written out independently of the oracle: even N -> -N/2 .. N/2-1, odd N -> -(N-1)/2 .. (N-1)/2
    ranges = [range(-(m // 2), m - m // 2) for m in n]
    psis, eig = [], []
    for mx in ranges[0]:
        for my in ranges[1]:
            for mz in ranges[2]:
                m = (mx, my, mz)
                psis.append(np.exp(2j * np.pi * sum(m[a] * ii[a] / n[a] for a in range(3))))
                eig.append(0.5 * sum((TWO_PI * m[a] / length[a] + kpt[a]) ** 2 for a in range(3)))
    psis = np.array(psis)
    eig = np.array(eig)
    if ecut is not None:
        assert (eig > ecut).any() and (eig <= ecut).any()
        eig = np.where(eig <= ecut, eig, 0.0)
    for backend in (0, 1):
        out = oracle.kinetic(n, length, kpt, -1.0 if ecut is None else ecut, psis, backend)
        err = np.abs(out - eig[:, None, None, None] * psis).max()
        assert err < 1e-12 * max(1.0, eig.max())


# --------------------------------------------------------------------------------------------- P3
def test_p3_constant_potential_is_a_shift(oracle):
    cfg = small_cfg(102)
    wl = W.make(cfg)
    psi = W.states(cfg)
    c = -0.37
    h0 = oracle.apply_hamiltonian(cfg.n, cfg.length, cfg.kpt, -1.0, None, wl.proj, psi, 0)
    hc = oracle.apply_hamiltonian(cfg.n, cfg.length, cfg.kpt, -1.0, np.full(cfg.n, c), wl.proj, psi, 0)
    assert rel(hc - h0, c * psi) < 1e-13
    # local term alone is the pointwise product with the real array V
    assert rel(oracle.local(cfg.n, wl.v, psi), wl.v[None] * psi) == 0.0
    # spectrum of the dense matrix shifts by c
    wl_c = W.Workload(cfg=cfg, pos=wl.pos, v=wl.v + c, proj=wl.proj)
    e0 = np.linalg.eigvalsh(dense_matrix(oracle, cfg, wl))
    ec = np.linalg.eigvalsh(dense_matrix(oracle, cfg, wl_c))
    assert np.abs(ec - e0 - c).max() < 1e-12


# --------------------------------------------------------------------------------------------- P4
def test_p4_single_projector_closed_form(oracle):
    """One atom, one channel: V_nl = D dV |beta><beta|.  psi = 1 -> beta[q] D dV sum(beta) on the sphere, 0 elsewhere."""
    cfg = W.test_config(103, (8, 7, 6), (7.0, 6.0, 5.5), nst=1, natoms=1, lmax=0, rc=2.1, dl=(1.5,))
    wl = W.make(cfg)
    pr = wl.proj
    assert pr.natoms == 1 and 10 < len(pr.sph_idx) < cfg.npts
    beta = pr.beta_of(0)[0]
    one = np.ones(cfg.n, dtype=np.complex128)
    out = oracle.nonlocal_(cfg.n, cfg.length, (0, 0, 0), pr, one)
    expect = np.zeros(cfg.npts, dtype=np.complex128)
    expect[pr.sph_idx] = beta * 1.5 * cfg.dv * beta.sum()
    assert rel(out.ravel(), expect) < 1e-14
    # dense matrix: rank one, single non-zero eigenvalue D dV sum(beta^2)
    eye = np.eye(cfg.npts, dtype=np.complex128).reshape((cfg.npts,) + cfg.n)
    m = oracle.nonlocal_(cfg.n, cfg.length, (0, 0, 0), pr, eye).reshape(cfg.npts, cfg.npts).T
    ev = np.linalg.eigvalsh(0.5 * (m + m.conj().T))
    assert abs(ev[-1] - 1.5 * cfg.dv * np.sum(beta ** 2)) < 1e-12
    assert np.abs(ev[:-1]).max() < 1e-12
    assert np.linalg.matrix_rank(m, tol=1e-10) == 1


def test_p4_rank_and_overlap_additivity(oracle):
    """Several atoms / channels: rank <= sum C; the operator is the sum of the per-atom operators (overlapping spheres add)."""
    cfg = small_cfg(104, n=(6, 6, 5), length=(5.0, 5.0, 4.5), natoms=3, lmax=1, rc=2.2)
    wl = W.make(cfg)
    pr = wl.proj
    counts = np.bincount(pr.sph_idx, minlength=cfg.npts)
    assert counts.max() >= 2, "test geometry must have overlapping spheres"
    eye = np.eye(cfg.npts, dtype=np.complex128).reshape((cfg.npts,) + cfg.n)
    m = oracle.nonlocal_(cfg.n, cfg.length, (0, 0, 0), pr, eye).reshape(cfg.npts, cfg.npts).T
    assert np.linalg.matrix_rank(m, tol=1e-10) <= int(pr.chan_off[-1])
    # explicit sum of outer products, channel by channel
    expect = np.zeros((cfg.npts, cfg.npts))
    for a in range(pr.natoms):
        idx = pr.sph_idx[pr.sph_off[a]:pr.sph_off[a + 1]]
        for c, b in enumerate(pr.beta_of(a)):
            full = np.zeros(cfg.npts)
            full[idx] = b
            expect += pr.dcoef[pr.chan_off[a] + c] * cfg.dv * np.outer(full, full)
    assert np.abs(m - expect).max() < 1e-13


def test_p4_ylm_orthonormal_on_a_fine_sphere():
    """Input-generator check: the real Y_lm of R11 are orthonormal (Lebedev-free check by dense quadrature)."""
    th = (np.arange(400) + 0.5) * math.pi / 400
    ph = (np.arange(800) + 0.5) * TWO_PI / 800
    T, P = np.meshgrid(th, ph, indexing="ij")
    d = np.stack([np.sin(T) * np.cos(P), np.sin(T) * np.sin(P), np.cos(T)], axis=-1).reshape(-1, 3)
    wgt = (np.sin(T) * (math.pi / 400) * (TWO_PI / 800)).ravel()
    ys = [W.real_ylm(l, m, d) for l in range(3) for m in range(-l, l + 1)]
    gram = np.array([[np.sum(wgt * a * b) for b in ys] for a in ys])
    assert np.abs(gram - np.eye(9)).max() < 1e-4


# --------------------------------------------------------------------------------------------- P5
@pytest.mark.parametrize("kfrac,ecut", [((0, 0, 0), None), ((0.25, 0.1, -0.3), 6.0)])
def test_p5_hermiticity(oracle, kfrac, ecut):
    cfg = small_cfg(105, n=(8, 6, 9), length=(6.0, 5.0, 7.0), natoms=3, lmax=2, rc=2.2, kfrac=kfrac, ecut=ecut)
    wl = W.make(cfg)
    rng = np.random.default_rng(5)
    phi, psi = rand_c(rng, cfg.n), rand_c(rng, cfg.n)
    for backend in (0, 1):
        hpsi = oracle.apply_workload(wl, psi, backend)
        hphi = oracle.apply_workload(wl, phi, backend)
        lhs = np.vdot(phi, hpsi)
        rhs = np.conj(np.vdot(psi, hphi))      # <H phi|psi> = <psi|H phi>^*
        assert abs(lhs - rhs) < 1e-12 * abs(lhs)


@pytest.mark.parametrize("kfrac,ecut", [((0, 0, 0), None), ((0.25, 0.0, 0.0), 5.0)])
def test_p5_dense_matrix_is_hermitian(oracle, kfrac, ecut):
    cfg = small_cfg(106, n=(4, 6, 5), length=(4.4, 5.5, 5.0), natoms=2, lmax=1, rc=1.9, kfrac=kfrac, ecut=ecut)
    wl = W.make(cfg)
    h = dense_matrix(oracle, cfg, wl)
    assert np.abs(h - h.conj().T).max() < 1e-13 * np.abs(h).max()
    ev = np.linalg.eigvals(h)
    assert np.abs(ev.imag).max() < 1e-12
    # term by term: T + V + Vnl assembled from the separate exports equals H
    eye = np.eye(cfg.npts, dtype=np.complex128).reshape((cfg.npts,) + cfg.n)
    parts = (oracle.kinetic(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, eye, 0) + oracle.local(cfg.n, wl.v, eye)
             + oracle.nonlocal_(cfg.n, cfg.length, cfg.kpt, wl.proj, eye))
    assert np.abs(parts.reshape(cfg.npts, cfg.npts).T - h).max() < 1e-13


# --------------------------------------------------------------------------------------------- P6
@pytest.mark.parametrize("units", [(1, 0, 0), (1, 1, 0), (1, 1, 1)])
def test_p6_bloch_phase_identity(oracle, units):
    """k a reciprocal-lattice vector, no mask: H_k u = e^{-ik.r} H_Gamma (e^{ik.r} u)   (reading R2).

    Holds for +1 unit on axes with EVEN N only: the shifted frequency N/2 folds to -N/2 (R7) with the same square;
    for odd N, (N+1)/2 folds to -(N-1)/2 and the kinetic eigenvalue changes.  So every axis here is even."""
    geo = dict(n=(6, 8, 10), length=(5.0, 6.0, 6.5), natoms=3, lmax=2, rc=2.2)
    base = small_cfg(107, **geo)
    cfg_k = small_cfg(107, kfrac=tuple(float(u) for u in units), **geo)
    wl0, wlk = W.make(base), W.make(cfg_k)
    assert np.array_equal(wl0.proj.sph_idx, wlk.proj.sph_idx)
    rng = np.random.default_rng(6)
    u = rand_c(rng, base.n)
    ii = np.meshgrid(*[np.arange(m) for m in base.n], indexing="ij")
    eikr = np.exp(2j * np.pi * sum(units[a] * ii[a] / base.n[a] for a in range(3)))   # k.r with r = i h, k = 2 pi units / L
    lhs = oracle.apply_workload(wlk, u, 0)
    rhs = np.conj(eikr) * oracle.apply_workload(wl0, eikr * u, 0)
    assert rel(lhs, rhs) < 1e-13
    # the projector part alone must satisfy it too (this is what fixes the phase in the gather AND the scatter)
    nl_k = oracle.nonlocal_(base.n, base.length, cfg_k.kpt, wlk.proj, u)
    nl_0 = np.conj(eikr) * oracle.nonlocal_(base.n, base.length, (0, 0, 0), wl0.proj, eikr * u)
    assert rel(nl_k, nl_0) < 1e-13
    assert np.linalg.norm(nl_k) > 1e-3


def test_p6_translation_covariance(oracle):
    """Shift V, atoms and psi by whole grid points -> H psi shifts identically (spheres crossing the cell boundary)."""
    cfg = small_cfg(108, n=(8, 6, 10), length=(6.0, 4.8, 7.0), natoms=2, lmax=1, rc=2.0, kfrac=(0.2, 0.0, -0.1))
    pos = W.atom_positions(cfg)
    shift = (3, 5, 7)
    h = cfg.spacing
    pos2 = np.mod(pos + np.array([shift[a] * h[a] for a in range(3)]), np.array(cfg.length))
    rng = np.random.default_rng(8)
    v = rng.standard_normal(cfg.n)
    psi = rand_c(rng, cfg.n)
    wl1 = W.Workload(cfg=cfg, pos=pos, v=v, proj=W.projectors(cfg, pos))
    wl2 = W.Workload(cfg=cfg, pos=pos2, v=np.roll(v, shift, axis=(0, 1, 2)), proj=W.projectors(cfg, pos2))
    def wraps(pr, a):   # a sphere crosses the boundary on an axis if it holds index 0 and N-1 but not every index
        ijk = np.unravel_index(pr.sph_idx[pr.sph_off[a]:pr.sph_off[a + 1]], cfg.n)
        return any(0 in x and cfg.n[ax] - 1 in x and len(set(x.tolist())) < cfg.n[ax] for ax, x in enumerate(ijk))
    wrapped = [wraps(wl2.proj, a) for a in range(2)]
    assert any(wrapped), "geometry must have a sphere that crosses the cell boundary"
    h1 = oracle.apply_workload(wl1, psi, 0)
    h2 = oracle.apply_workload(wl2, np.roll(psi, shift, axis=(0, 1, 2)), 0)
    assert rel(h2, np.roll(h1, shift, axis=(0, 1, 2))) < 1e-12


# --------------------------------------------------------------------------------------------- P7
def taylor4(x):
    return 1.0 - 1j * x - x ** 2 / 2.0 + 1j * x ** 3 / 6.0 + x ** 4 / 24.0


def test_p7_taylor_modulus_polynomial():
    """|P(x)|^2 = 1 - x^6/72 + x^8/576 (R15), by exact polynomial multiplication of the Eq. 8 coefficients."""
    from fractions import Fraction as F
    re = [F(1), F(0), F(-1, 2), F(0), F(1, 24)]     # real part coefficients of P
    im = [F(0), F(-1), F(0), F(1, 6), F(0)]
    sq = [F(0)] * 9
    for i in range(5):
        for j in range(5):
            sq[i + j] += re[i] * re[j] + im[i] * im[j]
    assert sq == [F(1), 0, 0, 0, 0, 0, F(-1, 72), 0, F(1, 576)]


def test_p7_kinetic_only_propagation_closed_form(oracle):
    """V = 0, no atoms: psi_hat(n, j dt) = P(t[n] dt)^j psi_hat(n, 0); norm follows |P|^{2j}.  FFTs by numpy here."""
    n, length = (8, 6, 12), (5.0, 4.0, 7.0)
    kfrac = (0.25, 0.0, 0.0)
    kpt = [TWO_PI * kfrac[a] / length[a] for a in range(3)]
    rng = np.random.default_rng(7)
    psi0 = rand_c(rng, (2,) + n)
    dt, nsteps = 0.05, 7
    g = [TWO_PI * np.fft.fftfreq(n[a], d=1.0 / n[a]) / length[a] + kpt[a] for a in range(3)]
    t = 0.5 * (g[0][:, None, None] ** 2 + g[1][None, :, None] ** 2 + g[2][None, None, :] ** 2)
    assert t.max() * dt > 0.5                                  # a regime where |P| visibly differs from 1
    for backend in (0, 1):
        out = oracle.propagate(n, length, kpt, -1.0, None, None, psi0, dt, nsteps, 4, backend)
        expect = np.fft.ifftn(taylor4(t * dt) ** nsteps * np.fft.fftn(psi0, axes=(1, 2, 3)), axes=(1, 2, 3))
        assert rel(out, expect) < 1e-12
        x = t * dt
        norm2 = np.sum(np.abs(np.fft.fftn(psi0, axes=(1, 2, 3))) ** 2 * (1 - x ** 6 / 72 + x ** 8 / 576) ** nsteps,
                       axis=(1, 2, 3)) / (n[0] * n[1] * n[2])
        assert np.allclose(np.sum(np.abs(out) ** 2, axis=(1, 2, 3)), norm2, rtol=1e-12)


def test_p7_eigenvector_of_full_h(oracle):
    """An eigenvector of the dense small-grid H is multiplied by P(eps dt) per step; one-step error vs exp ~ x^5/120."""
    cfg = small_cfg(109, n=(4, 5, 6), length=(4.4, 5.0, 5.5), natoms=2, lmax=1, rc=1.9, kfrac=(0.1, 0.2, 0.0))
    wl = W.make(cfg)
    h = dense_matrix(oracle, cfg, wl)
    ev, vec = np.linalg.eigh(0.5 * (h + h.conj().T))
    for j in (0, len(ev) // 2, len(ev) - 1):
        eps = ev[j]
        v0 = vec[:, j].reshape(cfg.n)
        dt, nsteps = 0.03, 5
        out = oracle.propagate_workload(wl, v0, dt=dt, nsteps=nsteps, backend=0)
        assert rel(out, taylor4(eps * dt) ** nsteps * v0) < 1e-11
        one = oracle.propagate_workload(wl, v0, dt=dt, nsteps=1, backend=0)
        x = eps * dt
        err = np.linalg.norm(one - np.exp(-1j * x) * v0) / np.linalg.norm(v0)
        assert err <= abs(x) ** 5 / 120 * 1.5 + 1e-13
        if abs(x) > 0.05:
            assert err >= abs(x) ** 5 / 120 * 0.5


def test_p7_propagate_is_literal_eq8(oracle):
    """One step = psi + c1 H psi + c2 H^2 psi + c3 H^3 psi + c4 H^4 psi with the Eq. 8 coefficients, via repeated apply."""
    cfg = small_cfg(110)
    wl = W.make(cfg)
    psi = W.states(cfg)
    dt = 0.04
    acc, phi = psi.copy(), psi
    for k, c in enumerate([-1j * dt, -dt ** 2 / 2, 1j * dt ** 3 / 6, dt ** 4 / 24], start=1):
        phi = oracle.apply_workload(wl, phi, 0)
        acc = acc + c * phi
    assert rel(oracle.propagate_workload(wl, psi, dt=dt, nsteps=1, backend=0), acc) < 1e-14
    # and nsteps composes
    two = oracle.propagate_workload(wl, psi, dt=dt, nsteps=2, backend=0)
    assert rel(two, oracle.propagate_workload(wl, acc, dt=dt, nsteps=1, backend=0)) < 1e-13


def test_golden_eq8_coefficients(oracle):
    """tests/golden/eq8_taylor_coefficients.txt (Eq. 8): one oracle step on a 1-point 'grid-free' problem --
    an eigenvector of a constant potential with eigenvalue eps -- is multiplied by sum_k (1/k!) (-i)^k (eps dt)^k."""
    import os
    from fractions import Fraction as F
    rows, mod2 = [], None
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "eq8_taylor_coefficients.txt")):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        if tok[0] == "modulus2":
            mod2 = [F(t) for t in tok[1:]]
        else:
            rows.append((int(tok[0]), F(tok[1]), int(tok[2]), int(tok[3])))
    assert [r[0] for r in rows] == [0, 1, 2, 3, 4] and len(mod2) == 9
    # constant potential c on a 4^3 grid, psi = const: H psi = c psi (kinetic term of the G = 0 wave is 0 at Gamma)
    n, length, c, dt = (4, 4, 4), (3.0, 3.0, 3.0), -0.7, 0.9
    psi = np.ones(n, dtype=np.complex128)
    for lam_scale, nsteps in ((1.0, 1), (0.5, 1)):
        out = oracle.propagate(n, length, (0.0, 0.0, 0.0), -1.0, np.full(n, c), None, psi, dt * lam_scale, nsteps, 4, 0)
        x = c * dt * lam_scale
        expect = sum(float(f) * complex(re, im) * x ** k for k, f, re, im in rows)
        assert np.abs(out - expect).max() < 1e-14
        m2 = sum(float(cf) * x ** m for m, cf in enumerate(mod2))
        assert abs(abs(expect) ** 2 - m2) < 1e-14


# --------------------------------------------------------------------------------------------- P9 (NEXT-1: ETRS)
def poly4(m, lam):
    """sum_{k=0..4} (lam m)^k / k! of a dense matrix m, by explicit matrix powers (numpy, independent of the oracle's loop)."""
    a = lam * m
    a2 = a @ a
    return np.eye(m.shape[0], dtype=np.complex128) + a + a2 / 2.0 + (a2 @ a) / 6.0 + (a2 @ a2) / 24.0


def test_p9_taylor_pair_against_dense_matrix_polynomials(oracle):
    """both exponentials from one chain.  half = P4(-i dt/2 H) psi, full = P4(-i dt H) psi, with H the
    dense small-grid matrix (pinned by P1-P6) and the polynomials formed by matrix products."""
    cfg = small_cfg(111, n=(4, 5, 6), length=(4.4, 5.0, 5.5), natoms=2, lmax=1, rc=1.9, kfrac=(0.0, 0.2, -0.1))
    wl = W.make(cfg)
    h = dense_matrix(oracle, cfg, wl)
    psi = W.states(cfg)
    dt = 0.06
    half, full = oracle.taylor_pair(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, psi, dt, 4, 0)
    flat = psi.reshape(psi.shape[0], -1).T
    assert rel(half.reshape(psi.shape[0], -1).T, poly4(h, -0.5j * dt) @ flat) < 1e-13
    assert rel(full.reshape(psi.shape[0], -1).T, poly4(h, -1j * dt) @ flat) < 1e-13
    # and the two agree with the single-lambda routine pinned by P7
    assert rel(half, oracle.propagate_workload(wl, psi, dt=0.5 * dt, nsteps=1, backend=0)) < 1e-14
    assert rel(full, oracle.propagate_workload(wl, psi, dt=dt, nsteps=1, backend=0)) < 1e-14


def test_p9_etrs_step_against_dense_matrices_with_two_potentials(oracle):
    """Eq. 6-7: psi(t+dt) = P4(-i dt/2 H(t+dt)) P4(-i dt/2 H(t)) psi, approx = P4(-i dt H(t)) psi, H(t+dt) from a second V."""
    cfg = small_cfg(112, n=(5, 4, 6), length=(5.0, 4.2, 5.6), natoms=2, lmax=1, rc=1.9)
    wl = W.make(cfg)
    rng = np.random.default_rng(112)
    v2 = wl.v + rng.uniform(-0.3, 0.3, wl.v.shape)
    wl2 = W.Workload(cfg=cfg, pos=wl.pos, v=v2, proj=wl.proj)
    h1, h2 = dense_matrix(oracle, cfg, wl), dense_matrix(oracle, cfg, wl2)
    psi = W.states(cfg)
    dt = 0.05
    out, approx = oracle.etrs_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, v2, wl.proj, psi, dt, 0)
    flat = psi.reshape(psi.shape[0], -1).T
    expect = poly4(h2, -0.5j * dt) @ (poly4(h1, -0.5j * dt) @ flat)
    assert rel(out.reshape(psi.shape[0], -1).T, expect) < 1e-13
    assert rel(approx.reshape(psi.shape[0], -1).T, poly4(h1, -1j * dt) @ flat) < 1e-13
    # the order of the two half steps matters when the potentials differ (a transposed operand would pass otherwise)
    swapped = poly4(h1, -0.5j * dt) @ (poly4(h2, -0.5j * dt) @ flat)
    assert rel(swapped, expect) > 1e-8


def test_p9_etrs_kinetic_only_closed_form(oracle):
    """V = 0, no atoms, fixed H: every plane wave is multiplied by P(t dt/2)^2 per ETRS step and approx by P(t dt)."""
    n, length = (6, 8, 4), (4.0, 5.0, 3.0)
    kpt = [TWO_PI * 0.2 / length[0], 0.0, 0.0]
    rng = np.random.default_rng(9)
    psi0 = rand_c(rng, (2,) + n)
    dt = 0.08
    g = [TWO_PI * np.fft.fftfreq(n[a], d=1.0 / n[a]) / length[a] + kpt[a] for a in range(3)]
    t = 0.5 * (g[0][:, None, None] ** 2 + g[1][None, :, None] ** 2 + g[2][None, None, :] ** 2)
    for backend in (0, 1):
        out, approx = oracle.etrs_step(n, length, kpt, -1.0, None, None, None, psi0, dt, backend)
        f0 = np.fft.fftn(psi0, axes=(1, 2, 3))
        assert rel(out, np.fft.ifftn(taylor4(0.5 * t * dt) ** 2 * f0, axes=(1, 2, 3))) < 1e-12
        assert rel(approx, np.fft.ifftn(taylor4(t * dt) * f0, axes=(1, 2, 3))) < 1e-12


# --------------------------------------------------------------------------------------------- P10 (NEXT-2)
def test_p10_density_definition_and_integral(oracle):
    """Eq. 1 by hand on a tiny grid; integral = sum of occupations for normalised states; accumulation in two pieces."""
    cfg = small_cfg(113, n=(4, 3, 5), length=(4.0, 3.3, 5.5), natoms=0, lmax=0)
    psi = W.states(cfg)                                    # 3 normalised states
    occ = np.array([2.0, 1.0, 0.25])
    d = oracle.density(cfg.n, psi, occ)
    assert np.abs(d - np.einsum("s,sxyz->xyz", occ, np.abs(psi) ** 2)).max() < 1e-15 * d.max()
    assert abs(cfg.dv * d.sum() - occ.sum()) < 1e-13
    assert np.abs(oracle.density(cfg.n, psi) - np.sum(np.abs(psi) ** 2, axis=0)).max() < 1e-15 * d.max()
    part = oracle.density(cfg.n, psi[:2], occ[:2])
    both = oracle.density(cfg.n, psi[2:], occ[2:], accumulate_into=part)
    assert np.abs(both - d).max() < 1e-15 * d.max()


@pytest.mark.parametrize("n,length", [((8, 6, 4), (5.0, 4.0, 3.0)), ((6, 6, 9), (4.0, 4.5, 7.0))])
def test_p10_hartree_plane_wave_closed_form(oracle, n, length):
    """n = cos(G0.r) is an eigenfunction of the periodic Poisson operator: v = 4 pi / |G0|^2 cos(G0.r); a constant gives 0
    (G = 0 dropped); the Nyquist wave of an even axis; linearity."""
    ii = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
    for backend in (0, 1):
        total, expect = np.zeros(n), np.zeros(n)
        for w, m in [(1.0, (1, 0, 0)), (-0.5, (0, 2, 1)), (0.3, (-1, 1, -2)), (0.7, (n[0] // 2, 0, 0))]:
            phase = TWO_PI * sum(m[a] * ii[a] / n[a] for a in range(3))
            g2 = sum((TWO_PI * m[a] / length[a]) ** 2 for a in range(3))
            dens = np.cos(phase)
            v = oracle.hartree(n, length, dens, backend)
            assert rel(v, 4 * np.pi / g2 * dens) < 1e-13
            total += w * dens
            expect += w * 4 * np.pi / g2 * dens
        assert rel(oracle.hartree(n, length, total + 3.7, backend), expect) < 1e-13
        assert np.abs(oracle.hartree(n, length, np.full(n, 2.5), backend)).max() < 1e-13


def test_p10_hartree_satisfies_the_poisson_equation(oracle):
    """Spectral Laplacian of v_H (numpy FFT, independent of the oracle's DFT) equals -4 pi (n - mean n); v_H has zero mean."""
    n, length = (6, 8, 5), (5.0, 6.0, 4.5)
    rng = np.random.default_rng(10)
    dens = rng.uniform(0.0, 1.0, n)
    v = oracle.hartree(n, length, dens, 0)
    g = [TWO_PI * np.fft.fftfreq(n[a], d=1.0 / n[a]) / length[a] for a in range(3)]
    g2 = g[0][:, None, None] ** 2 + g[1][None, :, None] ** 2 + g[2][None, None, :] ** 2
    lap = np.real(np.fft.ifftn(-g2 * np.fft.fftn(v)))
    assert rel(lap, -4 * np.pi * (dens - dens.mean())) < 1e-12
    assert abs(v.mean()) < 1e-13
    assert rel(oracle.hartree(n, length, dens, 1), v) < 1e-13


# --------------------------------------------------------------------------------------------- P11 (overlap matrix)
def test_p11_overlap_plane_waves_and_hand_values(oracle):
    """Distinct plane waves are orthogonal with norm^2 = cell volume; a 2-point hand example; conjugation on the left."""
    n, length = (4, 6, 5), (3.0, 4.0, 5.0)
    dv = np.prod([length[a] / n[a] for a in range(3)])
    ii = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
    ms = [(0, 0, 0), (1, 0, 0), (0, 2, 1), (-1, 1, 2), (1, 2, -2)]
    pw = np.array([np.exp(2j * np.pi * sum(m[a] * ii[a] / n[a] for a in range(3))) for m in ms])
    s = oracle.overlap(n, dv, pw, pw)
    assert np.abs(s - np.prod(length) * np.eye(len(ms))).max() < 1e-12
    a = np.zeros((1,) + n, dtype=np.complex128)
    b = np.zeros((2,) + n, dtype=np.complex128)
    a[0, 0, 0, 0], a[0, 1, 2, 3] = 1 + 2j, -1j
    b[0, 0, 0, 0], b[1, 1, 2, 3], b[1, 0, 0, 0] = 3 - 1j, 2.0, 1j
    s = oracle.overlap(n, 0.5, a, b)
    assert s.shape == (1, 2)
    assert abs(s[0, 0] - 0.5 * (1 - 2j) * (3 - 1j)) < 1e-15 and abs(s[0, 1] - 0.5 * ((1 - 2j) * 1j + 1j * 2.0)) < 1e-15


def test_p11_overlap_is_sesquilinear_and_hermitian(oracle):
    cfg = small_cfg(114, n=(5, 4, 6), length=(5.0, 4.4, 6.0), natoms=0, lmax=0)
    rng = np.random.default_rng(114)
    a, b = rand_c(rng, (3,) + cfg.n), rand_c(rng, (4,) + cfg.n)
    s = oracle.overlap(cfg.n, cfg.dv, a, b)
    assert np.abs(s - cfg.dv * np.einsum("ixyz,jxyz->ij", a.conj(), b)).max() < 1e-13 * np.abs(s).max()
    assert np.abs(oracle.overlap(cfg.n, cfg.dv, b, a) - s.conj().T).max() < 1e-13 * np.abs(s).max()
    saa = oracle.overlap(cfg.n, cfg.dv, a, a)
    assert np.abs(saa - saa.conj().T).max() < 1e-14 * np.abs(saa).max() and np.all(np.linalg.eigvalsh(saa) > 0)
    # normalised states of the generator have unit diagonal
    psi = W.states(cfg)
    assert np.abs(np.diag(oracle.overlap(cfg.n, cfg.dv, psi, psi)) - 1).max() < 1e-13
    # Hermiticity of H as a statement about overlaps: <a|Hb> = <Ha|b> (P5 in matrix form)
    cfgp = small_cfg(115, n=(4, 5, 6), length=(4.4, 5.0, 5.5), natoms=2, lmax=1, rc=1.9)
    wl = W.make(cfgp)
    x = W.states(cfgp)
    hx = oracle.apply_workload(wl, x, 0)
    m = oracle.overlap(cfgp.n, cfgp.dv, x, hx)
    assert np.abs(m - m.conj().T).max() < 1e-12 * np.abs(m).max()


def test_p11_orthonormalize_equals_gram_schmidt(oracle):
    """Cholesky orthonormalisation = modified Gram-Schmidt with positive normalisation (explicit loops here): unit overlap,
    psi'_j in span(psi_0..psi_j), and the same vectors; a rotation by a unitary keeps the overlap (rotate pin)."""
    cfg = small_cfg(116, n=(5, 6, 4), length=(5.0, 6.0, 4.0), natoms=0, lmax=0)
    rng = np.random.default_rng(116)
    psi = rand_c(rng, (5,) + cfg.n)
    psi[3] = 0.7 * psi[1] + 0.3 * psi[3]                       # some correlation between the inputs
    out = oracle.orthonormalize(cfg.n, cfg.dv, psi)
    s = oracle.overlap(cfg.n, cfg.dv, out, out)
    assert np.abs(s - np.eye(5)).max() < 1e-12
    q = []
    for j in range(5):                                         # modified Gram-Schmidt
        v = psi[j].copy()
        for u in q:
            v -= u * (cfg.dv * np.vdot(u, v))
        q.append(v / np.sqrt(cfg.dv * np.vdot(v, v).real))
    assert rel(out, np.array(q)) < 1e-11
    # triangular structure: <psi_i | out_j> dV is upper triangular ... equivalently out_j has no component outside span(psi_0..j)
    c = np.linalg.lstsq(psi.reshape(5, -1).T, out.reshape(5, -1).T, rcond=None)[0]     # out = psi c
    assert np.abs(np.tril(c, -1)).max() < 1e-10
    # rotate: a unitary rotation of an orthonormal block stays orthonormal; a single-column rotation is a linear combination
    u, _ = np.linalg.qr(rand_c(rng, (5, 5)))
    r = oracle.rotate(out, u)
    assert np.abs(oracle.overlap(cfg.n, cfg.dv, r, r) - np.eye(5)).max() < 1e-12
    col = rand_c(rng, (5, 1))
    assert rel(oracle.rotate(psi, col)[0], np.tensordot(col[:, 0], psi, axes=(0, 0))) < 1e-14


# --------------------------------------------------------------------------------------------- P12 (NEXT-3: SD step)
def teter_k(x):
    num = 27 + 18 * x + 12 * x ** 2 + 8 * x ** 3
    return num / (num + 16 * x ** 4)


def test_p12_sd_step_two_plane_waves_closed_form(oracle):
    """Kinetic-only H, psi = a e^{iG1.r} + b e^{iG2.r}: eps = T = (|a|^2 t1 + |b|^2 t2)/(|a|^2 + |b|^2) and the update
    multiplies coefficient c_m by 1 - lambda K(t_m / T)(t_m - eps).  Also K(0) = 1, K(x) -> 1/(2x)."""
    assert teter_k(0.0) == 1.0 and abs(teter_k(1e6) * 2e6 - 1.0) < 1e-5
    n, length = (6, 4, 8), (5.0, 3.0, 7.0)
    kpt = [0.0, TWO_PI * 0.1 / length[1], 0.0]
    ii = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
    m1, m2 = (1, 0, -2), (-2, 1, 3)
    w = [np.exp(2j * np.pi * sum(m[a] * ii[a] / n[a] for a in range(3))) for m in (m1, m2)]
    t = [0.5 * sum((TWO_PI * m[a] / length[a] + kpt[a]) ** 2 for a in range(3)) for m in (m1, m2)]
    a, b, lam = 0.8 - 0.3j, 0.5j, 0.21
    psi = (a * w[0] + b * w[1])[None]
    for backend in (0, 1):
        out, eig = oracle.sd_step(n, length, kpt, -1.0, None, None, psi, lam, backend)
        eps = (abs(a) ** 2 * t[0] + abs(b) ** 2 * t[1]) / (abs(a) ** 2 + abs(b) ** 2)
        assert abs(eig[0] - eps) < 1e-12 * eps
        expect = sum(c * (1 - lam * teter_k(tm / eps) * (tm - eps)) * wm for c, tm, wm in ((a, t[0], w[0]), (b, t[1], w[1])))
        assert rel(out[0], expect) < 1e-12


def test_p12_sd_step_fixed_points_and_descent(oracle):
    """An eigenvector of the dense small-grid H is a fixed point (zero residual) with eig = its eigenvalue; for a random
    state a small step lowers the Rayleigh quotient; the update equals the explicit formula built from H, T and numpy FFTs."""
    cfg = small_cfg(117, n=(4, 5, 6), length=(4.4, 5.0, 5.5), natoms=2, lmax=1, rc=1.9)
    wl = W.make(cfg)
    h = dense_matrix(oracle, cfg, wl)
    ev, vec = np.linalg.eigh(0.5 * (h + h.conj().T))
    v0 = vec[:, 3].reshape((1,) + cfg.n)
    out, eig = oracle.sd_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, v0, 0.3, 0)
    assert abs(eig[0] - ev[3]) < 1e-12 and rel(out, v0) < 1e-11
    psi = W.states(cfg)
    lam = 0.05
    out, eig = oracle.sd_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, psi, lam, 0)
    hpsi = oracle.apply_workload(wl, psi, 0)
    tpsi = oracle.kinetic(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, psi, 0)
    g = [TWO_PI * np.fft.fftfreq(cfg.n[a], d=1.0 / cfg.n[a]) / cfg.length[a] + cfg.kpt[a] for a in range(3)]
    tg = 0.5 * (g[0][:, None, None] ** 2 + g[1][None, :, None] ** 2 + g[2][None, None, :] ** 2)
    for s in range(psi.shape[0]):
        nn = np.vdot(psi[s], psi[s]).real
        eps, ts = np.vdot(psi[s], hpsi[s]).real / nn, np.vdot(psi[s], tpsi[s]).real / nn
        assert abs(eig[s] - eps) < 1e-12 * abs(eps)
        r = hpsi[s] - eps * psi[s]
        p = np.fft.ifftn(teter_k(tg / ts) * np.fft.fftn(r))
        assert rel(out[s], psi[s] - lam * p) < 1e-12
        hn = oracle.apply_workload(wl, out[s:s + 1], 0)[0]
        assert np.vdot(out[s], hn).real / np.vdot(out[s], out[s]).real < eps


def test_p12_sd_step_state_without_kinetic_energy(oracle):
    """Reading R19, T_s <= 0: a constant state at Gamma has <psi|T psi> = 0 up to rounding, x = t / T_s is undefined and
    the limit x -> infinity is taken (K = 1 at t = 0, K = 0 elsewhere) -- the same as a tiny positive T_s gives, so the
    result cannot hang on the sign of the rounding noise: only the mean of the residual is stepped along, and the result
    is finite.  With a constant potential and no atoms the constant state is an eigenvector and stays put."""
    cfg = small_cfg(121, n=(4, 6, 5), length=(4.0, 5.5, 5.0), natoms=2, lmax=1, rc=1.9)
    wl = W.make(cfg)
    psi = np.full((1,) + cfg.n, 0.3 - 0.2j)
    lam = 0.17
    for backend in (0, 1):
        out, eig = oracle.sd_step(cfg.n, cfg.length, (0.0, 0.0, 0.0), -1.0, wl.v, wl.proj, psi, lam, backend)
        h = oracle.apply_hamiltonian(cfg.n, cfg.length, (0.0, 0.0, 0.0), -1.0, wl.v, wl.proj, psi, backend)
        eps = np.vdot(psi[0], h[0]).real / np.vdot(psi[0], psi[0]).real
        r = h[0] - eps * psi[0]
        assert np.isfinite(out).all() and abs(eig[0] - eps) < 1e-12 * abs(eps)
        assert np.abs(out[0] - (psi[0] - lam * r.mean())).max() < 1e-13
    vc = np.full(cfg.n, -0.4)
    out, eig = oracle.sd_step(cfg.n, cfg.length, (0.0, 0.0, 0.0), -1.0, vc, None, psi, lam, 0)
    assert abs(eig[0] + 0.4) < 1e-13 and rel(out[0], psi[0]) < 1e-13


# --------------------------------------------------------------------------------------------- P13 (NEXT-3: subspace diagonalisation)
def test_p13_subspace_diag_recovers_mixed_eigenvectors_and_cauchy_bounds(oracle):
    """A block spanned by exact eigenvectors of the dense small-grid H, mixed by a random unitary: the Ritz values are those
    eigenvalues and the Ritz vectors the eigenvectors up to a phase.  For a random orthonormal block: the Ritz vectors are
    orthonormal, psi'^H H psi' is diagonal with the Ritz values, the trace is kept, and Cauchy interlacing holds."""
    cfg = small_cfg(118, n=(4, 5, 6), length=(4.4, 5.0, 5.5), natoms=2, lmax=1, rc=1.9)
    wl = W.make(cfg)
    h = dense_matrix(oracle, cfg, wl)
    ev, vec = np.linalg.eigh(0.5 * (h + h.conj().T))
    pick = [0, 2, 5, 9]
    basis = vec[:, pick].T.reshape((4,) + cfg.n) / np.sqrt(cfg.dv)             # dV-orthonormal eigenvectors
    rng = np.random.default_rng(118)
    u, _ = np.linalg.qr(rand_c(rng, (4, 4)))
    psi = oracle.rotate(basis, u)
    w, out, _ = oracle.subspace_diag(cfg.n, cfg.dv, psi, oracle.apply_workload(wl, psi, 0))
    assert np.abs(w - ev[pick]).max() < 1e-12
    s = oracle.overlap(cfg.n, cfg.dv, basis, out)
    assert np.abs(np.abs(s) - np.eye(4)).max() < 1e-10                          # same vectors up to a phase
    psi = oracle.orthonormalize(cfg.n, cfg.dv, W.states(cfg))
    hp = oracle.apply_workload(wl, psi, 0)
    w, out, v = oracle.subspace_diag(cfg.n, cfg.dv, psi, hp)
    assert np.abs(oracle.overlap(cfg.n, cfg.dv, out, out) - np.eye(3)).max() < 1e-12
    m2 = oracle.overlap(cfg.n, cfg.dv, out, oracle.apply_workload(wl, out, 0))
    assert np.abs(m2 - np.diag(w)).max() < 1e-12
    assert abs(w.sum() - np.trace(oracle.overlap(cfg.n, cfg.dv, psi, hp)).real) < 1e-12
    assert all(w[i] >= ev[i] - 1e-12 for i in range(3)) and all(w[2 - i] <= ev[-1 - i] + 1e-12 for i in range(3))


# --------------------------------------------------------------------------------------------- P14 (NEXT-4: gradient, forces)
def test_p14_gradient_of_plane_waves(oracle):
    """d_a e^{iG.r} = i (G_a + k_a) e^{iG.r} (psi is the periodic part u_k, so the Bloch vector enters as in the kinetic term)."""
    n, length = (6, 8, 5), (5.0, 7.0, 4.0)
    kpt = [TWO_PI * 0.2 / length[0], 0.0, -TWO_PI * 0.1 / length[2]]
    ii = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
    ms = [(0, 0, 0), (1, -2, 2), (-2, 3, -1), (2, 1, 0)]
    psi = np.array([np.exp(2j * np.pi * sum(m[a] * ii[a] / n[a] for a in range(3))) for m in ms])
    for backend in (0, 1):
        for a in range(3):
            g = oracle.gradient(n, length, kpt, a, psi, backend)
            for s, m in enumerate(ms):
                assert rel(g[s], 1j * (TWO_PI * m[a] / length[a] + kpt[a]) * psi[s]) < 1e-12 or np.abs(g[s]).max() < 1e-12


def smooth_l1(proj):
    """Test-only projector table: the l = 1 channels of workloads.projectors multiplied by |d|, i.e.
    |d| exp(-d^2/2 sigma^2) Y_1m(d/|d|) = c exp(-d^2/2 sigma^2) (y, z, x): smooth at the atom, unlike the generator's."""
    out = W.Projectors(**{**proj.__dict__})
    out.beta = proj.beta.copy()
    off = 0
    for a in range(proj.natoms):
        p0, p1 = int(proj.sph_off[a]), int(proj.sph_off[a + 1])
        nc, npt = int(proj.chan_off[a + 1] - proj.chan_off[a]), p1 - p0
        r = np.sqrt(np.sum(proj.sph_disp[p0:p1] ** 2, axis=1))
        for c in range(1, nc):                                            # channel 0 is l = 0
            out.beta[off + c * npt: off + (c + 1) * npt] *= r
        off += nc * npt
    return out


@pytest.mark.parametrize("lmax,tol,smooth", [(0, 2e-4, False), (1, 3e-2, False), (1, 1e-5, True)])
def test_p14_forces_are_the_derivative_of_the_ionic_energy_at_fixed_orbitals(oracle, lmax, tol, smooth):
    """Eq. 11 equals d/dR_I of E_I(R) = sum_s f_s <psi_s| v_I(r - R_I) |psi_s> at fixed orbitals (translate the atom, rebuild
    its projector table and its local well, central differences).  The third case pins the l = 1 path tightly with a
    projector that is smooth at the atom (smooth_l1, sigma = 0.7 on a 24^3 grid): 1e-5 (measured 2e-6).  Equality holds in the band-limited limit: smooth
    orbitals, projectors negligible at the cutoff sphere; the l = 0 Gaussian is smooth (tight tolerance), the generator's
    l = 1 projectors exp(-d^2/2 sigma^2) Y_1m(d/|d|) jump at the atom, so aliasing leaves about 1e-2 there -- a dropped
    term, a wrong sign or a missing factor 2 is an O(1) error in both.  Checks the factor 2 Re, occupations, the per-atom
    split and both terms of v_I."""
    if smooth:      # wider cell, so that sigma = 0.7 is negligible both at the grid's Nyquist frequency and at the sphere edge
        cfg = W.test_config(122, (24, 24, 24), (9.0, 9.0, 9.0), nst=3, natoms=2, lmax=1, rc=4.0, dl=(1.5, -0.7),
                            proj_sigma=0.7, well_z=1.2, well_sigma=0.7)
    else:
        cfg = W.test_config(119 + lmax, (16, 16, 16), (6.0, 6.0, 6.0), nst=3, natoms=2, lmax=lmax, rc=2.9,
                            dl=(1.5, -0.7)[: lmax + 1], proj_sigma=0.5, well_z=1.2, well_sigma=0.7)
    table = (lambda c, p: smooth_l1(W.projectors(c, p))) if smooth else W.projectors
    pos = np.array([[2.1, 3.3, 2.7], [4.0, 1.6, 3.9]])
    ii = np.meshgrid(*[np.arange(m) for m in cfg.n], indexing="ij")
    rng = np.random.default_rng(119)
    ms = [(a, b, c) for a in (0, 1, -1) for b in (0, 1, -1) for c in (0, 1, -1)]
    pw = np.array([np.exp(2j * np.pi * sum(m[k] * ii[k] / cfg.n[k] for k in range(3))) for m in ms])
    psi = np.tensordot(rand_c(rng, (3, len(ms))), pw, axes=(1, 0))                    # band-limited, not normalised
    occ = np.array([2.0, 1.0, 0.5])
    one_atom = dataclasses_replace(cfg, natoms=1)

    def well(center):
        return W.local_potential(one_atom, np.array([center]))

    def energy(center):
        one = table(one_atom, np.array([center]))
        v = well(center)
        e = 0.0
        for s in range(3):
            nl = oracle.nonlocal_(cfg.n, cfg.length, cfg.kpt, one, psi[s])
            e += occ[s] * cfg.dv * (np.vdot(psi[s], nl).real + np.sum(v * np.abs(psi[s]) ** 2))
        return e

    proj = table(cfg, pos)
    vloc = np.array([well(pos[0]), well(pos[1])])
    f = oracle.forces(cfg.n, cfg.length, cfg.kpt, proj, psi, occ, vloc, 1)
    f_nl = oracle.forces(cfg.n, cfg.length, cfg.kpt, proj, psi, occ, None, 1)
    assert np.abs(f - f_nl).max() > 1e-3 * np.abs(f).max()                            # the local term is visible
    delta = 1e-3
    for atom in range(2):
        for a in range(3):
            d = np.zeros(3)
            d[a] = delta
            fd = (energy(pos[atom] + d) - energy(pos[atom] - d)) / (2 * delta)
            assert abs(f[atom, a] - fd) < tol * np.abs(f).max(), (atom, a, f[atom, a], fd)
    # occupations enter linearly; a constant orbital at Gamma has no gradient, hence no force; both DFT back-ends agree
    assert np.abs(oracle.forces(cfg.n, cfg.length, cfg.kpt, proj, psi, 2 * occ, vloc, 1) - 2 * f).max() < 1e-12 * np.abs(f).max()
    const = np.ones((1,) + cfg.n, dtype=np.complex128)
    assert np.abs(oracle.forces(cfg.n, cfg.length, cfg.kpt, proj, const, None, vloc, 1)).max() < 1e-10
    assert np.abs(oracle.forces(cfg.n, cfg.length, cfg.kpt, proj, psi[:1], None, None, 0) -
                  oracle.forces(cfg.n, cfg.length, cfg.kpt, proj, psi[:1], None, None, 1)).max() < 1e-10 * np.abs(f).max()


# --------------------------------------------------------------------------------------------- P8
def test_p8_independent_of_batching(oracle):
    cfg = W.CONFIGS["tiny"]
    wl = W.make(cfg)
    psi = W.states(cfg)
    full = oracle.apply_workload(wl, psi, 1)
    for s in (0, 3, 7):
        assert np.array_equal(oracle.apply_workload(wl, psi[s], 1), full[s])
    part = oracle.apply_workload(wl, psi[2:5], 1)
    assert np.array_equal(part, full[2:5])
    # the generator is per-state seeded too
    assert np.array_equal(W.states(cfg, 2, 5), psi[2:5])


# --------------------------------------------------------------------------------------------- argument checks
def test_oracle_rejects_bad_index(oracle):
    cfg = small_cfg(111)
    wl = W.make(cfg)
    bad = W.Projectors(**{**wl.proj.__dict__})
    bad.sph_idx = wl.proj.sph_idx.copy()
    bad.sph_idx[3] = cfg.npts
    with pytest.raises(RuntimeError):
        oracle.apply_hamiltonian(cfg.n, cfg.length, cfg.kpt, -1.0, wl.v, bad, W.states(cfg), 0)
