"""Axis lengths beyond the tuned set: include/tdh.h accepts every N = 2^a 3^b with 4 <= N <= 256 on every axis (the
cutoff-derived grids of PAPER.md:106) and refuses everything else with TDH_EUNSUPPORTED.  Parity of the general path
(generic_fft.cuh) against the oracle's direct O(N^2) DFT and its literal loops."""
import numpy as np
import pytest

from paper_2106_03872_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device: the product has no CPU fallback")
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2106_03872_b200 import binding
    binding.lib()
    return binding


def per_state_rel(a, b):
    a = a.reshape(a.shape[0], -1)
    b = b.reshape(b.shape[0], -1)
    return np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)


@pytest.mark.parametrize("n", [(24, 24, 24), (36, 36, 36), (54, 54, 54), (72, 72, 72), (81, 81, 81), (108, 108, 108),
                               (128, 128, 128), (4, 6, 9), (8, 12, 18), (27, 64, 24), (144, 16, 32), (256, 8, 4),
                               (96, 96, 24), (4, 4, 4), (243, 4, 6), (162, 192, 8)])
def test_fft3d_general_sizes_match_the_direct_dft(torch_cuda, B, oracle, n):
    torch = torch_cuda
    rng = np.random.default_rng(sum(n))
    nst = 1 if n[0] * n[1] * n[2] > 10 ** 6 else 3
    a = rng.standard_normal((nst,) + n) + 1j * rng.standard_normal((nst,) + n)
    with B.Grid(n, (1.0, 1.0, 1.0), max_states=nst) as g:
        d = torch.from_numpy(a).cuda()
        g.fft3d(d, -1)
        assert per_state_rel(d.cpu().numpy(), oracle.dft3d(a, -1, oracle.DIRECT)).max() < 1e-13
        g.fft3d(d, +1)
        assert per_state_rel(d.cpu().numpy(), a).max() < 1e-13
        d2 = torch.from_numpy(a).cuda()
        g.fft3d(d2, +1)
        assert per_state_rel(d2.cpu().numpy(), oracle.dft3d(a, +1, oracle.DIRECT)).max() < 1e-13


@pytest.mark.parametrize("n,nst,natoms,lmax,kfrac,ecut", [
    ((24, 36, 54), 5, 4, 1, (0.0, 0.0, 0.0), None), ((72, 72, 72), 3, 6, 2, (0.25, 0.0, -0.1), 30.0),
    ((81, 27, 9), 4, 2, 0, (0.0, 0.2, 0.0), None), ((128, 24, 16), 3, 3, 1, (0.0, 0.0, 0.0), 12.0),
    ((12, 12, 12), 9, 1, 2, (0.1, 0.1, 0.1), None), ((96, 96, 24), 2, 5, 1, (0.0, 0.0, 0.0), None)])
def test_apply_and_propagate_general_sizes(torch_cuda, B, oracle, n, nst, natoms, lmax, kfrac, ecut):
    """H psi and two Taylor-4 steps on grids outside the tuned set (incl. one with two tuned axes), chunked and not."""
    torch = torch_cuda
    length = tuple(0.42 * m for m in n)
    cfg = W.test_config(600 + n[0], n, length, nst=nst, natoms=natoms, lmax=lmax, rc=float(min(2.6, 0.45 * min(length))),
                        dl=(2.0, -0.8, 0.3)[: lmax + 1], kfrac=kfrac, ecut=ecut)
    wl = W.make(cfg)
    psi = W.states(cfg)
    backend = oracle.NAIVE_FFT
    ref_h = oracle.apply_workload(wl, psi, backend)
    ref_p = oracle.propagate_workload(wl, psi, dt=0.01, nsteps=2, backend=backend)
    nl = oracle.nonlocal_(cfg.n, cfg.length, cfg.kpt, wl.proj, psi)
    with B.grid_for(wl) as g:
        for chunk in (None, 2):
            if chunk:
                g.set_chunk_states(chunk)
            d = torch.from_numpy(psi).cuda()
            out = g.apply_hamiltonian(d)
            assert per_state_rel(out.cpu().numpy(), ref_h).max() < TOL
            g.propagate(d, 0.01, 2)
            assert per_state_rel(d.cpu().numpy(), ref_p).max() < TOL
        g.set_projectors(None)
        out0 = g.apply_hamiltonian(torch.from_numpy(psi).cuda())
        assert per_state_rel((out - out0).cpu().numpy(), nl).max() < 1e-8      # the non-local part on its own


def test_other_entry_points_on_a_general_grid(torch_cuda, B, oracle):
    """Density, Hartree, gradient, forces, SD step, Taylor pair on a (24, 36, 54) grid against the oracle, and the GEMM-based
    rotations (ragged point counts: test_rotations_on_grids_whose_point_count_is_ragged)."""
    torch = torch_cuda
    n = (24, 36, 54)
    cfg = W.test_config(650, n, (10.0, 15.0, 22.0), nst=6, natoms=3, lmax=1, rc=2.6, dl=(2.0, -0.8), kfrac=(0.0, 0.1, 0.0))
    wl = W.make(cfg)
    psi = W.states(cfg)
    rng = np.random.default_rng(650)
    occ = rng.uniform(0.5, 2.0, cfg.nst)
    with B.grid_for(wl) as g:
        d = torch.from_numpy(psi).cuda()
        dens = g.density(d, occ)
        ref_n = oracle.density(cfg.n, psi, occ)
        assert np.abs(dens.cpu().numpy() - ref_n).max() <= 1e-13 * ref_n.max()
        vh = g.hartree(dens).cpu().numpy()
        ref_vh = oracle.hartree(cfg.n, cfg.length, ref_n, oracle.NAIVE_FFT)
        assert np.linalg.norm(vh - ref_vh) <= TOL * np.linalg.norm(ref_vh)
        for a in range(3):
            assert per_state_rel(g.gradient(d, a).cpu().numpy(), oracle.gradient(cfg.n, cfg.length, cfg.kpt, a, psi)).max() < TOL
        f = g.forces(d, occ=occ)
        ref_f = oracle.forces(cfg.n, cfg.length, cfg.kpt, wl.proj, psi, occ, None)
        assert np.abs(f - ref_f).max() < 1e-10 * np.abs(ref_f).max()
        ref_sd, eig_ref = oracle.sd_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, psi, 0.1, oracle.NAIVE_FFT)
        d2 = torch.from_numpy(psi).cuda()
        eig = g.sd_step(d2, 0.1)
        assert np.abs(eig - eig_ref).max() < 1e-11 * np.abs(eig_ref).max()
        assert per_state_rel(d2.cpu().numpy(), ref_sd).max() < TOL
        half_ref, full_ref = oracle.taylor_pair(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, psi, 0.02, 4, oracle.NAIVE_FFT)
        d3 = torch.from_numpy(psi).cuda()
        full = g.taylor_pair(d3, 0.02)
        assert per_state_rel(d3.cpu().numpy(), half_ref).max() < TOL and per_state_rel(full.cpu().numpy(), full_ref).max() < TOL
        # 24 * 36 * 54 = 46656 = 64 * 729: the GEMM kernels apply
        s = g.overlap(d).cpu().numpy()
        assert np.abs(s - oracle.overlap(cfg.n, cfg.dv, psi, psi)).max() < 1e-12
        q = g.orthonormalize(d)
        assert np.abs(g.overlap(q).cpu().numpy() - np.eye(cfg.nst)).max() < 1e-12


@pytest.mark.parametrize("n,nst", [((27, 27, 27), 8), ((9, 9, 9), 3), ((54, 54, 54), 5), ((81, 4, 6), 70)])
def test_rotations_on_grids_whose_point_count_is_ragged(torch_cuda, B, oracle, n, nst):
    """Overlap, rotation, orthonormalisation and subspace diagonalisation on grids whose point count is no multiple of 64
    or even of 16 (27^3 = 19683, 9^3 = 729, 54^3 = 64 x 2460.4, 81 x 4 x 6 = 1944): the last chunk of K of the overlap GEMM
    and the last tile of points of the rotation GEMM are predicated.  Against the oracle's literal sums."""
    torch = torch_cuda
    cfg = W.test_config(660 + n[0], n, tuple(max(0.45 * m, 4.4) for m in n), nst=nst, natoms=2, lmax=1, rc=1.9, dl=(2.0, -0.8))
    wl = W.make(cfg)
    psi = W.states(cfg)
    rng = np.random.default_rng([W.BASE_SEED, 660, n[0], nst])
    m = rng.standard_normal((nst, nst + 3)) + 1j * rng.standard_normal((nst, nst + 3))
    with B.grid_for(wl) as g:
        d = torch.from_numpy(psi).cuda()
        other = torch.from_numpy(psi[::-1].copy()).cuda()
        s = g.overlap(d, other).cpu().numpy()
        ref_s = oracle.overlap(cfg.n, cfg.dv, psi, psi[::-1].copy())
        assert np.abs(s - ref_s).max() <= 1e-13 * np.abs(np.diag(oracle.overlap(cfg.n, cfg.dv, psi, psi))).max()
        r = g.rotate(d, torch.from_numpy(m).cuda()).cpu().numpy()
        assert per_state_rel(r, oracle.rotate(psi, m)).max() < 1e-13
        q = g.orthonormalize(d)
        q_ref = oracle.orthonormalize(cfg.n, cfg.dv, psi)
        assert per_state_rel(q.cpu().numpy(), q_ref).max() < 1e-11
        assert np.abs(g.overlap(q).cpu().numpy() - np.eye(nst)).max() < 1e-12
        w_ref, _, _ = oracle.subspace_diag(cfg.n, cfg.dv, q_ref, oracle.apply_workload(wl, q_ref, oracle.NAIVE_FFT))
        w, out = g.subspace_diag(q, g.apply_hamiltonian(q))
        assert np.abs(w - w_ref).max() < 1e-11 * max(1.0, np.abs(w_ref).max())
        assert np.abs(g.overlap(out).cpu().numpy() - np.eye(nst)).max() < 1e-11


def test_size_contract(torch_cuda, B):
    """TDH_EUNSUPPORTED exactly for a prime factor other than 2 or 3, for N < 4 and for N > 256."""
    for n in ((20, 16, 16), (16, 7, 16), (16, 16, 2), (3, 16, 16), (288, 16, 16), (16, 16, 512), (16, 250, 16)):
        with pytest.raises(B.TdhError) as e:
            B.Grid(n, (1.0, 1.0, 1.0))
        assert e.value.code == B.TDH_EUNSUPPORTED, n
    for n in ((4, 4, 4), (256, 4, 4), (6, 243, 8), (192, 216, 4)):
        B.Grid(n, (1.0, 1.0, 1.0)).close()
