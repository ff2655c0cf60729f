"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, same seeded inputs.

Bar (BASELINE.json north_star): relative L2 error per state <= 1e-11 in complex128.
"""
import math

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


def gpu_apply(torch, B, wl, psi, chunk=None, max_states=None):
    with B.grid_for(wl, max_states=max_states or psi.shape[0]) as g:
        if chunk is not None:
            g.set_chunk_states(chunk)
        out = g.apply_hamiltonian(torch.from_numpy(psi).cuda())
        torch.cuda.synchronize()
        return out.cpu().numpy(), g.last_launch_count()


# ------------------------------------------------------------------------------------------------ FFT alone (rows a1, a3)
@pytest.mark.parametrize("n", [(16, 16, 16), (32, 32, 32), (48, 48, 48), (64, 64, 64), (96, 96, 96),
                               (16, 32, 48), (48, 16, 32), (96, 64, 16), (32, 96, 64), (64, 48, 96)])
def test_fft3d_matches_oracle(torch_cuda, B, oracle, n):
    torch = torch_cuda
    rng = np.random.default_rng(sum(n))
    nst = 3
    a = rng.standard_normal((nst,) + n) + 1j * rng.standard_normal((nst,) + n)
    with B.Grid(n, (1.0, 1.0, 1.0), max_states=nst) as g:
        d = torch.from_numpy(a).cuda()
        g.fft3d(d, -1)
        torch.cuda.synchronize()
        f = d.cpu().numpy()
        ref = oracle.dft3d(a, -1, 1)
        assert per_state_rel(f, ref).max() < 1e-13
        g.fft3d(d, +1)
        torch.cuda.synchronize()
        assert per_state_rel(d.cpu().numpy(), a).max() < 1e-13
        # inverse alone against the oracle's inverse
        d2 = torch.from_numpy(a).cuda()
        g.fft3d(d2, +1)
        torch.cuda.synchronize()
        assert per_state_rel(d2.cpu().numpy(), oracle.dft3d(a, +1, 1)).max() < 1e-13


def test_fft3d_single_axis_impulses(torch_cuda, B):
    """Unit impulses: each axis' sign, order and stride, against the closed form exp(-i G.r0)."""
    torch = torch_cuda
    n = (16, 32, 48)
    r0s = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (5, 17, 29)]
    a = np.zeros((len(r0s),) + n, dtype=np.complex128)
    for s, r0 in enumerate(r0s):
        a[(s,) + r0] = 1.0
    with B.Grid(n, (1.0, 1.0, 1.0), max_states=len(r0s)) as g:
        d = torch.from_numpy(a).cuda()
        g.fft3d(d, -1)
        torch.cuda.synchronize()
        f = d.cpu().numpy()
    q = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
    for s, r0 in enumerate(r0s):
        expect = np.exp(-2j * np.pi * sum(q[i] * r0[i] / n[i] for i in range(3)))
        assert np.abs(f[s] - expect).max() < 1e-13


# ------------------------------------------------------------------------------------------------ H psi on the configs
@pytest.mark.parametrize("name,nst,backend", [("tiny", 8, 0), ("small", 64, 1), ("medium", 24, 1)])
def test_apply_matches_oracle_on_configs(torch_cuda, B, oracle, name, nst, backend):
    cfg = W.CONFIGS[name]
    wl = W.make(cfg)
    psi = W.states(cfg, 0, nst)
    out, launches = gpu_apply(torch_cuda, B, wl, psi)
    ref = oracle.apply_workload(wl, psi, backend)
    err = per_state_rel(out, ref)
    assert err.max() < TOL, err
    assert launches >= (1 if cfg.n[0] <= 32 else 4)      # 16^3 and 32^3: the whole application is one launch


def test_apply_terms_separately(torch_cuda, B, oracle):
    """Kinetic only, local only (as H - T), non-local only: isolates each epilogue term."""
    torch = torch_cuda
    cfg = W.test_config(201, (16, 32, 48), (6.0, 11.0, 15.0), nst=5, natoms=6, lmax=2, rc=2.4, dl=(2.0, -0.8, 0.3),
                        kfrac=(0.25, -0.1, 0.3), ecut=20.0)
    wl = W.make(cfg)
    psi = W.states(cfg)
    d = torch.from_numpy(psi).cuda()
    with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, cfg.nst) as g:
        t_only = g.apply_hamiltonian(d).cpu().numpy()
        assert per_state_rel(t_only, oracle.kinetic(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, psi, 1)).max() < TOL
        g.set_potential(torch.from_numpy(wl.v).cuda())
        tv = g.apply_hamiltonian(d).cpu().numpy()
        assert per_state_rel(tv - t_only, oracle.local(cfg.n, wl.v, psi)).max() < TOL
        g.set_potential(None)
        g.set_projectors(wl.proj)
        tn = g.apply_hamiltonian(d).cpu().numpy()
        nl_ref = oracle.nonlocal_(cfg.n, cfg.length, cfg.kpt, wl.proj, psi)
        assert np.linalg.norm(nl_ref) > 1e-3
        assert per_state_rel(tn - t_only, nl_ref).max() < 1e-10     # difference of two O(10) numbers
        g.set_projectors(None)
        assert np.array_equal(g.apply_hamiltonian(d).cpu().numpy(), t_only)


@pytest.mark.parametrize("n,nst,natoms,lmax", [((16, 16, 16), 1, 1, 0), ((32, 16, 48), 7, 3, 1), ((48, 48, 16), 13, 5, 2),
                                               ((64, 32, 32), 9, 4, 1), ((16, 96, 32), 3, 2, 2)])
def test_apply_ragged_blocks_and_mixed_grids(torch_cuda, B, oracle, n, nst, natoms, lmax):
    """State counts that are not multiples of the 8-state MMA tile or of the chunk; non-cubic grids; overlapping spheres."""
    cfg = W.test_config(202 + nst, n, tuple(0.45 * m for m in n), nst=nst, natoms=natoms, lmax=lmax, rc=2.6,
                        dl=(2.0, -0.8, 0.3)[: lmax + 1], kfrac=(0.0, 0.2, 0.0))
    wl = W.make(cfg)
    psi = W.states(cfg)
    ref = oracle.apply_workload(wl, psi, 1)
    for chunk in (None, 1, 2, 5):
        out, _ = gpu_apply(torch_cuda, B, wl, psi, chunk=chunk)
        assert per_state_rel(out, ref).max() < TOL


def test_apply_independent_of_batching(torch_cuda, B):
    """P8 on the GPU: H psi_s does not depend on the block or chunk it is submitted in (bitwise)."""
    cfg = W.CONFIGS["small"]
    wl = W.make(cfg)
    psi = W.states(cfg, 0, 20)
    full, _ = gpu_apply(torch_cuda, B, wl, psi)
    part, _ = gpu_apply(torch_cuda, B, wl, psi[5:12], chunk=3)
    assert np.array_equal(part, full[5:12])
    one, _ = gpu_apply(torch_cuda, B, wl, psi[19:20])
    assert np.array_equal(one, full[19:20])


def test_plane_waves_and_constant_potential_on_gpu(torch_cuda, B):
    """Closed forms straight on the GPU path: T e^{iG.r} = 1/2|G+k|^2 e^{iG.r} incl. Nyquist and mask; V = c shifts."""
    torch = torch_cuda
    n, length = (16, 32, 16), (5.0, 9.0, 6.0)
    kfrac = (0.25, 0.0, -0.5)
    kpt = [2 * math.pi * kfrac[a] / length[a] for a in range(3)]
    ms = [(0, 0, 0), (1, 0, 0), (-8, 0, 0), (0, -16, 3), (7, 15, -8), (-3, 5, 7), (2, -1, 1)]
    ii = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
    psi = np.array([np.exp(2j * np.pi * sum(m[a] * ii[a] / n[a] for a in range(3))) for m in ms])
    eig = np.array([0.5 * sum((2 * math.pi * m[a] / length[a] + kpt[a]) ** 2 for a in range(3)) for m in ms])
    ecut = float(np.sort(eig)[3] + 1e-9)
    d = torch.from_numpy(psi).cuda()
    with B.Grid(n, length, kpt, -1.0, len(ms)) as g:
        out = g.apply_hamiltonian(d).cpu().numpy()
        assert np.abs(out - eig[:, None, None, None] * psi).max() < 1e-12 * eig.max()
        g.set_potential(torch.full(n, -0.37, dtype=torch.float64, device="cuda"))
        out_c = g.apply_hamiltonian(d).cpu().numpy()
        assert np.abs(out_c - out + 0.37 * psi).max() < 1e-12 * eig.max()
    with B.Grid(n, length, kpt, ecut, len(ms)) as g:
        out = g.apply_hamiltonian(d).cpu().numpy()
        keep = np.where(eig <= ecut, eig, 0.0)
        assert (keep == 0).sum() >= 3
        assert np.abs(out - keep[:, None, None, None] * psi).max() < 1e-12 * eig.max()


# ------------------------------------------------------------------------------------------------ propagate (row a7)
def test_propagate_matches_oracle_tiny_and_small(torch_cuda, B, oracle):
    torch = torch_cuda
    for name, nst, nsteps, dt in (("tiny", 8, 6, 0.02), ("small", 6, 3, 0.02)):
        cfg = W.CONFIGS[name]
        wl = W.make(cfg)
        psi = W.states(cfg, 0, nst)
        with B.grid_for(wl, max_states=nst) as g:
            d = torch.from_numpy(psi).cuda()
            g.propagate(d, dt, nsteps)
            torch.cuda.synchronize()
            out = d.cpu().numpy()
            assert g.last_launch_count() == nsteps * 4              # 4 applications per step, one launch each (on-chip path)
        ref = oracle.propagate_workload(wl, psi, dt=dt, nsteps=nsteps, backend=1)
        assert per_state_rel(out, ref).max() < TOL
        # norms agree with the oracle's (R15: not with 1)
        n_gpu = np.sum(np.abs(out) ** 2, axis=(1, 2, 3))
        n_ref = np.sum(np.abs(ref) ** 2, axis=(1, 2, 3))
        assert np.abs(n_gpu / n_ref - 1).max() < 1e-11


def test_propagate_kinetic_only_closed_form(torch_cuda, B):
    """P7 on the GPU: psi_hat(j dt) = P(t dt)^j psi_hat(0) with k != 0; transforms by numpy here."""
    torch = torch_cuda
    n, length = (32, 16, 48), (7.0, 4.0, 9.0)
    kfrac = (0.25, 0.0, 0.0)
    kpt = [2 * math.pi * kfrac[a] / length[a] for a in range(3)]
    rng = np.random.default_rng(3)
    psi0 = rng.standard_normal((3,) + n) + 1j * rng.standard_normal((3,) + n)
    dt, nsteps = 0.01, 9
    g_ax = [2 * math.pi * np.fft.fftfreq(n[a], d=1.0 / n[a]) / length[a] + kpt[a] for a in range(3)]
    t = 0.5 * (g_ax[0][:, None, None] ** 2 + g_ax[1][None, :, None] ** 2 + g_ax[2][None, None, :] ** 2)
    x = t * dt
    P = 1 - 1j * x - x ** 2 / 2 + 1j * x ** 3 / 6 + x ** 4 / 24
    expect = np.fft.ifftn(P ** nsteps * np.fft.fftn(psi0, axes=(1, 2, 3)), axes=(1, 2, 3))
    with B.Grid(n, length, kpt, -1.0, 3) as g:
        d = torch.from_numpy(psi0).cuda()
        g.propagate(d, dt, nsteps)
        torch.cuda.synchronize()
        out = d.cpu().numpy()
    assert per_state_rel(out, expect).max() < 1e-12


def test_propagate_zero_steps_and_chunking(torch_cuda, B, oracle):
    torch = torch_cuda
    cfg = W.CONFIGS["tiny"]
    wl = W.make(cfg)
    psi = W.states(cfg)
    with B.grid_for(wl) as g:
        d = torch.from_numpy(psi).cuda()
        g.propagate(d, 0.02, 0)
        assert np.array_equal(d.cpu().numpy(), psi)
        outs = []
        for chunk in (0, 1, 3):
            g.set_chunk_states(chunk)
            d = torch.from_numpy(psi).cuda()
            g.propagate(d, 0.02, 2)
            outs.append(d.cpu().numpy())
        assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


# ------------------------------------------------------------------------------------------------ host-buffer path
def test_host_entry_points_equal_device_path(torch_cuda, B):
    torch = torch_cuda
    cfg = W.CONFIGS["small"]
    wl = W.make(cfg)
    psi = W.states(cfg, 0, 24)
    with B.grid_for(wl, max_states=24) as g:
        dev = g.apply_hamiltonian(torch.from_numpy(psi).cuda()).cpu().numpy()
        pin_in = torch.from_numpy(psi).pin_memory()
        pin_out = torch.empty_like(pin_in).pin_memory()
        g.apply_hamiltonian_host(pin_in, pin_out)
        assert np.array_equal(pin_out.numpy(), dev)
        out_np = np.empty_like(psi)                      # pageable memory works too
        g.apply_hamiltonian_host(psi, out_np)
        assert np.array_equal(out_np, dev)
        d = torch.from_numpy(psi).cuda()
        g.propagate(d, 0.02, 2)
        h = psi.copy()
        g.propagate_host(h, 0.02, 2)
        assert np.array_equal(h, d.cpu().numpy())


# ------------------------------------------------------------------------------------------------ errors
def test_error_codes(torch_cuda, B):
    torch = torch_cuda
    with pytest.raises(B.TdhError) as e:
        B.Grid((20, 16, 16), (1, 1, 1))
    assert e.value.code == B.TDH_EUNSUPPORTED
    with pytest.raises(B.TdhError) as e:
        B.Grid((16, 16, 16), (1, -1, 1))
    assert e.value.code == B.TDH_EINVAL
    cfg = W.CONFIGS["tiny"]
    wl = W.make(cfg)
    with B.grid_for(wl, max_states=4) as g:
        psi = torch.zeros((5,) + cfg.n, dtype=torch.complex128, device="cuda")
        with pytest.raises(B.TdhError) as e:
            g.apply_hamiltonian(psi)
        assert e.value.code == B.TDH_EINVAL
        with pytest.raises(B.TdhError) as e:
            g.apply_hamiltonian(psi[:2], out=psi[1:3])
        assert e.value.code == B.TDH_EINVAL
        with pytest.raises(B.TdhError) as e:
            g.propagate(psi[:2], 0.02, 1, order=3)
        assert e.value.code == B.TDH_EINVAL
        bad = W.Projectors(**{**wl.proj.__dict__})
        bad.sph_idx = wl.proj.sph_idx.copy()
        bad.sph_idx[0] = cfg.npts
        with pytest.raises(B.TdhError) as e:
            g.set_projectors(bad)
        assert e.value.code == B.TDH_EINDEX
        bad.sph_idx[0] = bad.sph_idx[1]
        with pytest.raises(B.TdhError) as e:
            g.set_projectors(bad)
        assert e.value.code == B.TDH_EINDEX


def test_reserve_preallocates_the_on_demand_scratch(torch_cuda, B, oracle):
    """tdh_reserve allocates what the rotations, the SD step, the forces' local term and the host entry points would
    allocate at first use: after it those calls leave the device's free memory unchanged, and their results are the usual
    ones."""
    torch = torch_cuda
    cfg = W.CONFIGS["tiny"]
    wl = W.make(cfg)
    psi = W.states(cfg)
    with B.grid_for(wl) as g:
        with pytest.raises(B.TdhError):
            g.reserve(rotation_states=cfg.nst + 1)
        g.reserve(rotation_states=cfg.nst, forces_local_term=True, host_buffers=True)
        d = torch.from_numpy(psi).cuda()
        out = torch.empty_like(d)
        host_out = np.empty_like(psi)
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        q = g.orthonormalize(d, out=out)
        g.apply_hamiltonian_host(psi, host_out)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0
        assert per_state_rel(q.cpu().numpy(), oracle.orthonormalize(cfg.n, cfg.dv, psi)).max() < 1e-11
        assert per_state_rel(host_out, oracle.apply_workload(wl, psi, oracle.DIRECT)).max() < 1e-11
