"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (whole block in one call, default
chunking), on sampled states the oracle can compute one by one; and the projector shapes the configs do not reach
(more than 9 channels per atom, three spheres on one grid point).

The blocks are filled on the device with seeded noise; the sampled states are the configs' own seeded states
(workloads.state), placed at the first, a middle and the last position of the block.
"""
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


@pytest.fixture(scope="module")
def oracle():
    from oracle import build, ref
    build.build()
    return ref


def per_state_rel(a, b):
    a = a.reshape(a.shape[0], -1)
    b = b.reshape(b.shape[0], -1)
    return np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)


def device_block(torch, cfg, nst, sample):
    """(nst, n) complex128 block of seeded device noise scaled like the config's states; states `sample` are W.state."""
    gen = torch.Generator(device="cuda")
    gen.manual_seed(W.BASE_SEED + cfg.cid)
    psi = torch.empty((nst,) + tuple(cfg.n), dtype=torch.complex128, device="cuda")
    scale = 1.0 / np.sqrt(2.0 * cfg.npts * cfg.dv)
    for s0 in range(0, nst, 64):
        s1 = min(nst, s0 + 64)
        v = torch.view_as_real(psi[s0:s1])
        v.copy_(torch.randn(v.shape, dtype=torch.float64, device="cuda", generator=gen))
        v.mul_(scale)
    host = np.stack([W.state(cfg, s) for s in sample])
    for j, s in enumerate(sample):
        psi[s].copy_(torch.from_numpy(host[j]))
    return psi, host


def default_chunks(cfg, nst):
    """State ranges of the launches tdh_apply_hamiltonian makes by default (as many states as a
    4 GiB work buffer holds, a multiple of 8 when the block is split)."""
    cap = min(nst, (4 << 30) // (cfg.npts * 16))
    c = cap // 8 * 8 if (cap < nst and cap >= 8) else cap
    return [(s0, min(nst, s0 + c)) for s0 in range(0, nst, c)]


def test_large_full_block_every_chunk_and_sub_blocks(torch_cuda, B, oracle):
    """Config 4 (96^3, 1024 states, 128 atoms): one tdh_apply_hamiltonian call on the whole block, as bench.py times it.
    The first and the last state of EVERY default chunk (296 + 296 + 296 + 136 states) are compared with the oracle, the
    whole output is finite, and the sub-blocks of bench.py's 32 / 128 / 512 sweep give bitwise the whole-block result."""
    torch = torch_cuda
    cfg = W.CONFIGS["large"]
    free, _ = torch.cuda.mem_get_info()
    nst = cfg.nst if free > 48 * 2 ** 30 else 320           # smaller boxes: same launch configuration, fewer states
    chunks = default_chunks(cfg, nst)
    assert len(chunks) >= 2
    sample = sorted({s for a, b in chunks for s in (a, b - 1)})
    wl = W.make(cfg)
    psi, host = device_block(torch, cfg, nst, sample)
    with B.grid_for(wl, max_states=nst) as g:
        out = g.apply_hamiltonian(psi)
        torch.cuda.synchronize()
        assert g.last_launch_count() == len(chunks) * (4 + 2)        # nl_project, 3 FFT kernels, nl_scatter x 2 colours
        got = np.stack([out[s].cpu().numpy() for s in sample])
        for a in range(0, nst, 64):                                     # no state is left unwritten or non-finite
            assert bool(torch.isfinite(torch.view_as_real(out[a:a + 64])).all())
        ref = oracle.apply_workload(wl, host, oracle.NAIVE_FFT)
        err = per_state_rel(got, ref)
        assert err.max() < TOL, err
        # bench.py's block-size sweep: a sub-block call gives bitwise the states of the whole-block call
        sub = torch.empty_like(psi[:min(512, nst // 2)])
        for b, s0 in ((32, nst // 2 + 96), (128, nst // 2), (min(512, nst // 2), nst // 2)):
            g.apply_hamiltonian(psi[s0:s0 + b], out=sub[:b])
            torch.cuda.synchronize()
            assert torch.equal(sub[:b], out[s0:s0 + b]), (b, s0)
    del psi, out, sub
    torch.cuda.empty_cache()


def test_large_propagate_default_chunking_sampled(torch_cuda, B, oracle):
    """north_star: propagate on config 4.  Two Taylor-4 steps of the whole 1024-state block in place with the default
    chunking (split tiles, coloured nl_scatter inside the Horner chain, the addend aliasing the output in the last
    application); one state of every chunk against ref_propagate."""
    torch = torch_cuda
    cfg = W.CONFIGS["large"]
    free, _ = torch.cuda.mem_get_info()
    nst = cfg.nst if free > 48 * 2 ** 30 else 320
    chunks = default_chunks(cfg, nst)
    sample = sorted({(a + b) // 2 for a, b in chunks} | {0, nst - 1})
    wl = W.make(cfg)
    psi, host = device_block(torch, cfg, nst, sample)
    nsteps, dt = 2, cfg.dt
    with B.grid_for(wl, max_states=nst) as g:
        g.propagate(psi, dt, nsteps)
        torch.cuda.synchronize()
        assert g.last_launch_count() == len(chunks) * nsteps * 4 * 6
        got = np.stack([psi[s].cpu().numpy() for s in sample])
    ref = oracle.propagate_workload(wl, host, dt=dt, nsteps=nsteps, backend=oracle.NAIVE_FFT)
    err = per_state_rel(got, ref)
    assert err.max() < TOL, err
    del psi
    torch.cuda.empty_cache()


def test_medium_full_block_apply_and_propagate(torch_cuda, B, oracle):
    """north_star: config 3 (48^3, 256 states, k = (0.25,0,0) 2pi/L, 30 Ha mask, 9 channels per atom) on its FULL block:
    apply compared for all 256 states, then three Taylor-4 steps of the resident block against ref_propagate on sampled
    states."""
    torch = torch_cuda
    cfg = W.CONFIGS["medium"]
    wl = W.make(cfg)
    psi = W.states(cfg)
    assert psi.shape[0] == 256
    ref = oracle.apply_workload(wl, psi, oracle.NAIVE_FFT)
    sample = [0, 1, 100, 254, 255]
    ref_p = oracle.propagate_workload(wl, psi[sample], dt=cfg.dt, nsteps=3, backend=oracle.NAIVE_FFT)
    with B.grid_for(wl) as g:
        d = torch.from_numpy(psi).cuda()
        out = g.apply_hamiltonian(d)
        err = per_state_rel(out.cpu().numpy(), ref)
        assert err.max() < TOL, err
        g.propagate(d, cfg.dt, 3)
        got = d.cpu().numpy()[sample]
    err = per_state_rel(got, ref_p)
    assert err.max() < TOL, err


def test_tddft_full_block_sampled_states(torch_cuda, B, oracle):
    """Config 5 (64^3, 512 states, 64 atoms, 20 Taylor-4 steps of dt = 0.02): propagate the whole block in place."""
    torch = torch_cuda
    cfg = W.CONFIGS["tddft"]
    nst = cfg.nst
    sample = [0, 255, nst - 1]
    wl = W.make(cfg)
    psi, host = device_block(torch, cfg, nst, sample)
    with B.grid_for(wl, max_states=nst) as g:
        g.propagate(psi, cfg.dt, cfg.nsteps)
        torch.cuda.synchronize()
        got = np.stack([psi[s].cpu().numpy() for s in sample])
    ref = oracle.propagate_workload(wl, host, backend=oracle.NAIVE_FFT)
    err = per_state_rel(got, ref)
    assert err.max() < TOL, err
    # norm after 20 steps equals the oracle's (reading R15: Taylor-4 is not unitary for white-noise states)
    n_got = cfg.dv * np.sum(np.abs(got.reshape(len(sample), -1)) ** 2, axis=1)
    n_ref = cfg.dv * np.sum(np.abs(ref.reshape(len(sample), -1)) ** 2, axis=1)
    assert np.abs(n_got - n_ref).max() < 1e-11
    del psi
    torch.cuda.empty_cache()


def synthetic_projectors(cfg, centers, nchan, rng):
    """Random real projector tables with `nchan` channels on spheres around `centers` (any channel count, any overlap)."""
    sph_off, chan_off = [0], [0]
    idx_all, disp_all, beta_all, d_all = [], [], [], []
    for c in centers:
        idx, disp = W.sphere_points(cfg, np.asarray(c, dtype=np.float64))
        idx_all.append(idx)
        disp_all.append(disp)
        beta_all.append(rng.standard_normal((nchan, len(idx))).ravel())
        d_all.append(rng.uniform(-1.0, 2.0, nchan))
        sph_off.append(sph_off[-1] + len(idx))
        chan_off.append(chan_off[-1] + nchan)
    return W.Projectors(natoms=len(centers), sph_off=np.asarray(sph_off, dtype=np.int64),
                        sph_idx=np.concatenate(idx_all).astype(np.int32), sph_disp=np.concatenate(disp_all),
                        chan_off=np.asarray(chan_off, dtype=np.int32), beta=np.concatenate(beta_all),
                        dcoef=np.concatenate(d_all))


@pytest.mark.parametrize("n,nchan,kfrac", [((48, 48, 48), 12, (0.0, 0.0, 0.0)), ((16, 32, 16), 16, (0.25, 0.0, -0.1)),
                                           ((96, 96, 16), 5, (0.0, 0.0, 0.0)), ((32, 32, 32), 1, (0.0, 0.3, 0.0))])
def test_many_channels_and_three_overlapping_spheres(torch_cuda, B, oracle, n, nchan, kfrac):
    """Channel counts that pad to 16 / 9 / 1, and grid points covered by three and four spheres (layers >= 3)."""
    torch = torch_cuda
    length = tuple(0.4 * m for m in n)
    cfg = W.test_config(230 + nchan, n, length, nst=6, natoms=1, lmax=0, rc=2.2, dl=(1.0,), kfrac=kfrac)
    rng = np.random.default_rng([W.BASE_SEED, 230, nchan])
    mid = [0.5 * l for l in length]
    centers = [mid, [mid[0] + 0.3, mid[1], mid[2]], [mid[0], mid[1] - 0.4, mid[2] + 0.2], [mid[0] + 0.1, mid[1] + 0.1, mid[2]],
               [0.1, 0.2, length[2] - 0.1]]                  # the last sphere wraps around the cell corner
    proj = synthetic_projectors(cfg, centers, nchan, rng)
    v = rng.uniform(-1.0, 1.0, n)
    psi = W.states(cfg)
    ref = oracle.apply_hamiltonian(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, v, proj, psi, oracle.NAIVE_FFT)
    nl = oracle.nonlocal_(cfg.n, cfg.length, cfg.kpt, proj, psi)
    assert np.linalg.norm(nl) > 1e-2 * np.linalg.norm(ref)   # the non-local term is a visible part of the result
    with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, cfg.nst) as g:
        g.set_potential(torch.from_numpy(v).cuda())
        g.set_projectors(proj)
        out = g.apply_hamiltonian(torch.from_numpy(psi).cuda()).cpu().numpy()
        assert per_state_rel(out, ref).max() < TOL
        d = torch.from_numpy(psi).cuda()
        g.propagate(d, 0.01, 2)
        ref_p = oracle.propagate(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, v, proj, psi, 0.01, 2, 4, oracle.NAIVE_FFT)
        assert per_state_rel(d.cpu().numpy(), ref_p).max() < TOL


@pytest.mark.parametrize("mode", ["0", "1"])
def test_both_back_projection_paths(torch_cuda, B, oracle, monkeypatch, mode):
    """The back-projection exists as records fused into plane_inv (TDH_NL_MODE=0) and as the coloured nl_scatter kernel
    (TDH_NL_MODE=1); the library picks one per grid.  Both must match the oracle on split and whole-plane tiles."""
    torch = torch_cuda
    monkeypatch.setenv("TDH_NL_MODE", mode)
    for cid, n, natoms, lmax in [(260, (32, 96, 96), 6, 1), (261, (48, 48, 32), 7, 2), (262, (16, 16, 16), 3, 0)]:
        cfg = W.test_config(cid, n, tuple(0.42 * m for m in n), nst=11, natoms=natoms, lmax=lmax, rc=2.9,
                            dl=(2.0, -0.8, 0.3)[: lmax + 1], kfrac=(0.1, 0.0, -0.2) if cid == 261 else (0.0, 0.0, 0.0))
        wl = W.make(cfg)
        psi = W.states(cfg)
        ref = oracle.apply_workload(wl, psi, oracle.NAIVE_FFT)
        with B.grid_for(wl) as g:
            d = torch.from_numpy(psi).cuda()
            out = g.apply_hamiltonian(d)
            n_launch = g.last_launch_count()
            assert per_state_rel(out.cpu().numpy(), ref).max() < TOL
            if cid != 262:                                           # 16^3 runs the one-launch on-chip path
                assert (n_launch > 4) == (mode == "1")
            g.propagate(d, 0.01, 1)
            ref_p = oracle.propagate_workload(wl, psi, dt=0.01, nsteps=1, backend=oracle.NAIVE_FFT)
            assert per_state_rel(d.cpu().numpy(), ref_p).max() < TOL



def test_scatter_by_bulk_reduce_add_equals_read_modify_write(torch_cuda, B, oracle, monkeypatch):
    """The separate back-projection kernel exists as a read-modify-write kernel (TDH_SCATTER_BULK=0) and with the addition
    done by the L2 (cp.reduce.async.bulk add.f64 per z-run and state; the library picks by the spheres' mean run length).  Both match the oracle; one IEEE
    addition per point either way, so the two results are bitwise equal.  Overlapping spheres (two colours), runs that wrap
    around the cell, a ragged state group, k != 0 with phases, 9 channels, a general (non-tuned) grid."""
    torch = torch_cuda
    monkeypatch.setenv("TDH_NL_MODE", "1")
    cases = [(280, (32, 96, 96), 9, 1, (0.0, 0.0, 0.0)), (281, (48, 48, 32), 7, 2, (0.1, 0.0, -0.2)),
             (282, (24, 36, 54), 5, 1, (0.0, 0.25, 0.0)), (283, (16, 27, 9), 4, 1, (0.0, 0.0, 0.0))]
    for cid, n, natoms, lmax, kfrac in cases:
        # (16, 27, 9): odd row length 9 with spheres wider than the cell in z -- runs of consecutive flat indices that
        # continue from the end of one row into the next
        cfg = W.test_config(cid, n, tuple(0.42 * m for m in n), nst=11, natoms=natoms, lmax=lmax,
                            rc=3.4 if cid != 283 else 1.8,
                            dl=(2.0, -0.8, 0.3)[: lmax + 1], kfrac=kfrac)
        wl = W.make(cfg)
        psi = W.states(cfg)
        ref = oracle.apply_workload(wl, psi, oracle.NAIVE_FFT)
        ref_p = oracle.propagate_workload(wl, psi, dt=0.01, nsteps=1, backend=oracle.NAIVE_FFT)
        got = {}
        for bulk in ("1", "0"):
            monkeypatch.setenv("TDH_SCATTER_BULK", bulk)
            with B.grid_for(wl) as g:
                d = torch.from_numpy(psi).cuda()
                h = g.apply_hamiltonian(d).cpu().numpy()
                assert g.last_launch_count() > 4                     # the separate kernel ran
                assert per_state_rel(h, ref).max() < TOL, (cid, bulk)
                g.propagate(d, 0.01, 1)
                p = d.cpu().numpy()
                assert per_state_rel(p, ref_p).max() < TOL, (cid, bulk)
                got[bulk] = (h, p)
        assert np.array_equal(got["1"][0], got["0"][0]) and np.array_equal(got["1"][1], got["0"][1]), cid

# ------------------------------------------------------------------------------------------------ NEXT-1: ETRS
@pytest.mark.parametrize("name,nst,backend", [("tiny", 8, 0), ("small", 24, 1), ("medium", 10, 1)])
def test_taylor_pair_and_etrs_match_oracle(torch_cuda, B, oracle, name, nst, backend):
    """tdh_taylor_pair and tdh_etrs_step (Eq. 6-7, V(t+dt) supplied) against the oracle."""
    torch = torch_cuda
    cfg = W.CONFIGS[name]
    wl = W.make(cfg)
    psi = W.states(cfg, 0, nst)
    rng = np.random.default_rng([W.BASE_SEED + cfg.cid, 7])
    v_next = wl.v + rng.uniform(-0.2, 0.2, wl.v.shape)
    dt = 0.02
    half_ref, full_ref = oracle.taylor_pair(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, psi, dt, 4, backend)
    out_ref, approx_ref = oracle.etrs_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, v_next, wl.proj, psi, dt, backend)
    with B.grid_for(wl, max_states=nst) as g:
        for chunk in (None, 3):
            if chunk:
                g.set_chunk_states(chunk)
            g.set_potential(torch.from_numpy(wl.v).cuda())
            d = torch.from_numpy(psi).cuda()
            full = g.taylor_pair(d, dt)
            assert per_state_rel(d.cpu().numpy(), half_ref).max() < TOL
            assert per_state_rel(full.cpu().numpy(), full_ref).max() < TOL
            d = torch.from_numpy(psi).cuda()
            approx = g.etrs_step(d, dt, torch.from_numpy(v_next).cuda())
            assert per_state_rel(d.cpu().numpy(), out_ref).max() < TOL
            assert per_state_rel(approx.cpu().numpy(), approx_ref).max() < TOL
        # the handle now holds V(t+dt): a plain application uses it
        wl2 = W.Workload(cfg=cfg, pos=wl.pos, v=v_next, proj=wl.proj)
        h = g.apply_hamiltonian(torch.from_numpy(psi).cuda()).cpu().numpy()
        assert per_state_rel(h, oracle.apply_workload(wl2, psi, backend)).max() < TOL


def test_etrs_single_state_handle_and_errors(torch_cuda, B, oracle):
    """max_states = 1 (workspace of one state) still has room for the four powers; overlapping buffers are refused."""
    torch = torch_cuda
    cfg = W.CONFIGS["tiny"]
    wl = W.make(cfg)
    psi = W.states(cfg, 0, 1)
    out_ref, _ = oracle.etrs_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, None, wl.proj, psi, 0.03, 0)
    with B.grid_for(wl, max_states=1) as g:
        d = torch.from_numpy(psi).cuda()
        g.etrs_step(d, 0.03, None)
        assert per_state_rel(d.cpu().numpy(), out_ref).max() < TOL
        with pytest.raises(B.TdhError) as e:
            g.taylor_pair(d, 0.03, full=d)
        assert e.value.code == B.TDH_EINVAL
        with pytest.raises(B.TdhError):
            g.taylor_pair(d, 0.03, order=2)


@pytest.mark.parametrize("mode", ["0", "1"])
def test_degenerate_projectors(torch_cuda, B, oracle, monkeypatch, mode):
    """An atom whose sphere holds no grid point, an atom with no channel, a one-point sphere, all in one table."""
    torch = torch_cuda
    monkeypatch.setenv("TDH_NL_MODE", mode)
    n, length = (16, 16, 32), (6.0, 6.0, 12.0)
    cfg = W.test_config(270, n, length, nst=5, natoms=1, lmax=1, rc=2.0, dl=(1.3, -0.6))
    full = W.projectors(cfg, np.array([[3.0, 3.0, 6.0]]))
    P = int(full.sph_off[1])
    beta_full = full.beta.reshape(4, P)
    # atoms: 0 = regular (4 channels), 1 = empty sphere (2 channels, 0 points), 2 = no channels (P points),
    #        3 = a single point with one channel
    sph_off = np.array([0, P, P, 2 * P, 2 * P + 1], dtype=np.int64)
    one_pt = np.array([123], dtype=np.int32)
    sph_idx = np.concatenate([full.sph_idx, full.sph_idx, one_pt]).astype(np.int32)
    sph_disp = np.concatenate([full.sph_disp, full.sph_disp, np.zeros((1, 3))])
    chan_off = np.array([0, 4, 6, 6, 7], dtype=np.int32)
    beta = np.concatenate([beta_full.ravel(), np.zeros(0), np.zeros(0), np.array([0.8])])
    dcoef = np.array([1.3, -0.6, -0.6, -0.6, 9.0, 9.0, 2.5])
    proj = W.Projectors(natoms=4, sph_off=sph_off, sph_idx=sph_idx, sph_disp=sph_disp, chan_off=chan_off, beta=beta,
                        dcoef=dcoef)
    psi = W.states(cfg)
    v = W.local_potential(cfg, np.array([[3.0, 3.0, 6.0]]))
    ref = oracle.apply_hamiltonian(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, v, proj, psi, oracle.NAIVE_FFT)
    with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, cfg.nst) as g:
        g.set_potential(torch.from_numpy(v).cuda())
        g.set_projectors(proj)
        out = g.apply_hamiltonian(torch.from_numpy(psi).cuda()).cpu().numpy()
        assert per_state_rel(out, ref).max() < TOL
        # the single-point projector is visible at its point and nowhere else
        g.set_projectors(None)
        base = g.apply_hamiltonian(torch.from_numpy(psi).cuda()).cpu().numpy()
        diff = (out - base).reshape(cfg.nst, -1)
        assert np.abs(diff[:, 123]).min() > 1e-6


# ------------------------------------------------------------------------------------------------ NEXT-2: density, Hartree
@pytest.mark.parametrize("name,nst", [("tiny", 8), ("small", 37), ("medium", 19)])
def test_density_matches_oracle(torch_cuda, B, oracle, name, nst):
    """tdh_density (Eq. 1) with and without occupations, in one piece and accumulated over two pieces (the sharded form)."""
    torch = torch_cuda
    cfg = W.CONFIGS[name]
    psi = W.states(cfg, 0, nst)
    rng = np.random.default_rng([W.BASE_SEED + cfg.cid, 8])
    occ = rng.uniform(0.0, 2.0, nst)
    with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, nst) as g:
        d = torch.from_numpy(psi).cuda()
        for o in (None, occ):
            ref = oracle.density(cfg.n, psi, o)
            got = g.density(d, o).cpu().numpy()
            assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
        cut = nst // 3 + 1
        part = g.density(d[:cut], occ[:cut])
        g.density(d[cut:], occ[cut:], out=part, accumulate=True)
        assert np.abs(part.cpu().numpy() - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("n,length", [((16, 16, 16), (10.0, 10.0, 10.0)), ((32, 48, 16), (9.0, 14.0, 5.0)),
                                      ((96, 96, 32), (30.0, 30.0, 10.0)), ((64, 64, 64), (25.0, 25.0, 25.0))])
def test_hartree_matches_oracle_and_closed_form(torch_cuda, B, oracle, n, length):
    """tdh_hartree against the oracle on a seeded density, and against 4 pi / |G|^2 cos(G.r) directly."""
    torch = torch_cuda
    rng = np.random.default_rng([W.BASE_SEED, 9, n[0], n[1]])
    dens = rng.uniform(0.0, 1.0, n)
    ref = oracle.hartree(n, length, dens, oracle.NAIVE_FFT)
    # a Bloch vector on the handle must not enter the Poisson solve
    with B.Grid(n, length, (0.1, -0.2, 0.05), -1.0, 1) as g:
        got = g.hartree(torch.from_numpy(dens).cuda()).cpu().numpy()
        assert np.linalg.norm(got - ref) <= TOL * np.linalg.norm(ref)
        ii = np.meshgrid(*[np.arange(m) for m in n], indexing="ij")
        for m in [(1, 0, 0), (0, -2, 3), (n[0] // 2, 1, 0), (3, 5, -7)]:
            wave = np.cos(2 * np.pi * sum(m[a] * ii[a] / n[a] for a in range(3)))
            g2 = sum((2 * np.pi * m[a] / length[a]) ** 2 for a in range(3))
            v = g.hartree(torch.from_numpy(wave + 0.3).cuda()).cpu().numpy()
            assert np.abs(v - 4 * np.pi / g2 * wave).max() < 1e-11 * 4 * np.pi / g2
        d = torch.from_numpy(dens).cuda()
        g.hartree(d, out=d)                                 # in place
        assert np.linalg.norm(d.cpu().numpy() - ref) <= TOL * np.linalg.norm(ref)


def test_self_consistent_etrs_step_with_hartree(torch_cuda, B, oracle):
    """The paper's loop (Eq. 6-7) closed with the Hartree term: approx -> n(t+dt) -> v_H -> H(t+dt) -> second half step,
    composed from tdh_taylor_pair, tdh_density, tdh_hartree, tdh_set_potential, tdh_propagate; same composition of the oracle."""
    torch = torch_cuda
    cfg = W.CONFIGS["small"]
    wl = W.make(cfg)
    nst = 12
    psi = W.states(cfg, 0, nst)
    occ = np.full(nst, 2.0)
    dt = 0.02
    v0 = wl.v + oracle.hartree(cfg.n, cfg.length, oracle.density(cfg.n, psi, occ))
    half_ref, approx_ref = oracle.taylor_pair(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, v0, wl.proj, psi, dt)
    v1 = wl.v + oracle.hartree(cfg.n, cfg.length, oracle.density(cfg.n, approx_ref, occ))
    out_ref = oracle.propagate(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, v1, wl.proj, half_ref, 0.5 * dt, 1)
    with B.grid_for(wl, max_states=nst) as g:
        vext = torch.from_numpy(wl.v).cuda()
        d = torch.from_numpy(psi).cuda()
        g.set_potential(vext + g.hartree(g.density(d, occ)))
        approx = g.taylor_pair(d, dt)
        g.set_potential(vext + g.hartree(g.density(approx, occ)))
        g.propagate(d, 0.5 * dt, 1)
        assert per_state_rel(d.cpu().numpy(), out_ref).max() < TOL


# ------------------------------------------------------------------------------------------------ overlap matrix (NEXT-3, block 1)
@pytest.mark.parametrize("n,na,nb", [((16, 16, 16), 8, 8), ((32, 16, 48), 5, 70), ((48, 48, 48), 130, 33), ((16, 32, 16), 1, 1)])
def test_overlap_matches_oracle(torch_cuda, B, oracle, n, na, nb):
    """tdh_overlap (FP64 tensor-core GEMM, split-K) against the literal loops, ragged tile edges included."""
    torch = torch_cuda
    rng = np.random.default_rng([W.BASE_SEED, 11, na, nb])
    length = tuple(0.5 * m for m in n)
    a = (rng.standard_normal((na,) + n) + 1j * rng.standard_normal((na,) + n))
    b = (rng.standard_normal((nb,) + n) + 1j * rng.standard_normal((nb,) + n))
    dv = float(np.prod([length[i] / n[i] for i in range(3)]))
    ref = oracle.overlap(n, dv, a, b)
    with B.Grid(n, length, (0.0, 0.0, 0.0), -1.0, max(na, nb)) as g:
        got = g.overlap(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()).cpu().numpy()
        scale = np.sqrt(np.outer(np.sum(np.abs(a) ** 2, axis=(1, 2, 3)), np.sum(np.abs(b) ** 2, axis=(1, 2, 3)))) * dv
        assert np.abs(got - ref).max() <= 1e-13 * scale.max()
        saa = g.overlap(torch.from_numpy(a).cuda()).cpu().numpy()
        assert np.abs(saa - saa.conj().T).max() <= 1e-13 * np.abs(saa).max()


def test_propagation_keeps_orthonormality(torch_cuda, B, oracle):
    """real-time propagation conserves the orthogonality of the states -- measured with tdh_overlap on a
    band-limited orthonormal block (Taylor-4 is unitary to O(x^6), R15), and equal to the oracle's overlap of its states."""
    torch = torch_cuda
    cfg = W.CONFIGS["small"]
    wl = W.make(cfg)
    nst = 16
    # orthonormal low-frequency block: the first plane waves, mixed by a random unitary
    ii = np.meshgrid(*[np.arange(m) for m in cfg.n], indexing="ij")
    ms = [(a, b, c) for a in (0, 1, -1) for b in (0, 1, -1) for c in (0, 1)][:nst]
    pw = np.array([np.exp(2j * np.pi * sum(m[k] * ii[k] / cfg.n[k] for k in range(3))) for m in ms])
    pw /= np.sqrt(np.prod(cfg.length))
    rng = np.random.default_rng(5)
    q, _ = np.linalg.qr(rng.standard_normal((nst, nst)) + 1j * rng.standard_normal((nst, nst)))
    psi = np.tensordot(q, pw, axes=(1, 0))
    with B.grid_for(wl, max_states=nst) as g:
        d = torch.from_numpy(psi).cuda()
        s0 = g.overlap(d).cpu().numpy()
        assert np.abs(s0 - np.eye(nst)).max() < 1e-12
        g.propagate(d, 0.01, 10)
        s1 = g.overlap(d).cpu().numpy()
        ref = oracle.propagate_workload(wl, psi, dt=0.01, nsteps=10)
        assert np.abs(s1 - oracle.overlap(cfg.n, cfg.dv, ref, ref)).max() < 1e-11
        assert np.abs(s1 - np.eye(nst)).max() < 1e-6            # orthonormal up to the Taylor truncation


@pytest.mark.parametrize("n,n_in,n_out", [((16, 16, 16), 8, 8), ((32, 16, 48), 70, 5), ((48, 48, 16), 33, 130), ((16, 32, 16), 1, 1)])
def test_rotate_matches_oracle(torch_cuda, B, oracle, n, n_in, n_out):
    """tdh_rotate (FP64 tensor-core GEMM over the state index) against the literal loops, ragged edges included."""
    torch = torch_cuda
    rng = np.random.default_rng([W.BASE_SEED, 12, n_in, n_out])
    psi = rng.standard_normal((n_in,) + n) + 1j * rng.standard_normal((n_in,) + n)
    m = rng.standard_normal((n_in, n_out)) + 1j * rng.standard_normal((n_in, n_out))
    ref = oracle.rotate(psi, m)
    with B.Grid(n, tuple(0.5 * k for k in n), (0.0, 0.0, 0.0), -1.0, max(n_in, n_out)) as g:
        got = g.rotate(torch.from_numpy(psi).cuda(), torch.from_numpy(m).cuda()).cpu().numpy()
        assert per_state_rel(got, ref).max() < 1e-13


@pytest.mark.parametrize("name,nst", [("tiny", 8), ("small", 64), ("medium", 37)])
def test_orthonormalize_matches_oracle(torch_cuda, B, oracle, name, nst):
    """tdh_orthonormalize = overlap + Cholesky + triangular inverse + rotation, against the oracle's composition; the
    result has unit overlap (measured with tdh_overlap); linearly dependent input is refused."""
    torch = torch_cuda
    cfg = W.CONFIGS[name]
    psi = W.states(cfg, 0, nst)
    psi[1] = 0.6 * psi[0] + 0.8 * psi[1]                       # correlated inputs
    ref = oracle.orthonormalize(cfg.n, cfg.dv, psi)
    with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, nst) as g:
        d = torch.from_numpy(psi).cuda()
        out = g.orthonormalize(d)
        assert g.last_launch_count() == 5
        assert per_state_rel(out.cpu().numpy(), ref).max() < 1e-11
        s = g.overlap(out).cpu().numpy()
        assert np.abs(s - np.eye(nst)).max() < 1e-12
        d[2] = d[0] - 2.0 * d[1]
        with pytest.raises(B.TdhError):
            g.orthonormalize(d)


# ------------------------------------------------------------------------------------------------ NEXT-3: SD step
@pytest.mark.parametrize("name,nst,backend", [("tiny", 8, 0), ("small", 21, 1), ("medium", 9, 1)])
def test_sd_step_matches_oracle(torch_cuda, B, oracle, name, nst, backend):
    """tdh_sd_step (Teter-preconditioned steepest descent, reading R19) against the oracle, chunked and not."""
    torch = torch_cuda
    cfg = W.CONFIGS[name]
    wl = W.make(cfg)
    psi = W.states(cfg, 0, nst)
    lam = 0.1
    ref, eig_ref = oracle.sd_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, psi, lam, backend)
    with B.grid_for(wl, max_states=nst) as g:
        for chunk in (None, 4):
            if chunk:
                g.set_chunk_states(chunk)
            d = torch.from_numpy(psi).cuda()
            eig = g.sd_step(d, lam)
            assert np.abs(eig - eig_ref).max() < 1e-11 * np.abs(eig_ref).max()
            assert per_state_rel(d.cpu().numpy(), ref).max() < TOL


def test_sd_sweeps_with_orthonormalisation_lower_the_energy(torch_cuda, B, oracle):
    """A few ground-state iterations composed from the C-ABI calls (SD update + Cholesky orthonormalisation): the sum of the
    Rayleigh quotients decreases monotonically and the block stays orthonormal; the same sequence of the oracle agrees."""
    torch = torch_cuda
    cfg = W.CONFIGS["tiny"]
    wl = W.make(cfg)
    psi = oracle.orthonormalize(cfg.n, cfg.dv, W.states(cfg))
    ref = psi.copy()
    with B.grid_for(wl) as g:
        d = torch.from_numpy(psi).cuda()
        sums = []
        for it in range(4):
            eig = g.sd_step(d, 0.3)
            d = g.orthonormalize(d)
            ref, eig_ref = oracle.sd_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, ref, 0.3, 0)
            ref = oracle.orthonormalize(cfg.n, cfg.dv, ref)
            assert np.abs(eig - eig_ref).max() < 1e-10
            sums.append(eig.sum())
        assert all(b < a for a, b in zip(sums, sums[1:]))
        assert per_state_rel(d.cpu().numpy(), ref).max() < 1e-9          # four compounded iterations
        assert np.abs(g.overlap(d).cpu().numpy() - np.eye(cfg.nst)).max() < 1e-12


# ------------------------------------------------------------------------------------------------ NEXT-3: subspace diagonalisation
@pytest.mark.parametrize("name,nst", [("tiny", 8), ("small", 33), ("medium", 64)])
def test_subspace_diag_matches_oracle(torch_cuda, B, oracle, name, nst):
    """tdh_subspace_diag: Ritz values equal the oracle's (library eigensolver); the Ritz vectors are unique only up to a
    phase, so what is compared is |<gpu_i|ref_i>| = 1 for separated Ritz values plus what must hold for any valid answer:
    orthonormality and psi'^H H psi' = diag(w)."""
    torch = torch_cuda
    cfg = W.CONFIGS[name]
    wl = W.make(cfg)
    psi = oracle.orthonormalize(cfg.n, cfg.dv, W.states(cfg, 0, nst))
    hpsi = oracle.apply_workload(wl, psi, oracle.NAIVE_FFT)
    w_ref, out_ref, _ = oracle.subspace_diag(cfg.n, cfg.dv, psi, hpsi)
    with B.grid_for(wl, max_states=nst) as g:
        d = torch.from_numpy(psi).cuda()
        h = g.apply_hamiltonian(d)
        w, out = g.subspace_diag(d, h)
        assert np.abs(w - w_ref).max() < 1e-11 * max(1.0, np.abs(w_ref).max())
        assert np.all(np.diff(w) >= 0)
        s = g.overlap(out).cpu().numpy()
        assert np.abs(s - np.eye(nst)).max() < 1e-11
        m = g.overlap(out, g.apply_hamiltonian(out)).cpu().numpy()
        assert np.abs(m - np.diag(w)).max() < 1e-10 * max(1.0, np.abs(w).max())
        ov = np.abs(np.diag(oracle.overlap(cfg.n, cfg.dv, out_ref, out.cpu().numpy())))
        gap = np.minimum(np.diff(w_ref, prepend=-np.inf), np.diff(w_ref, append=np.inf))
        sep = gap > 1e-3
        assert sep.sum() >= nst // 2 and np.abs(ov[sep] - 1).max() < 1e-8


@pytest.mark.parametrize("want_eig", [True, False])
def test_subspace_diag_reports_an_unconverged_eigensolver(torch_cuda, B, oracle, want_eig):
    """A subspace matrix with a non-finite entry cannot be diagonalised: the call fails whether or not the caller asked
    for the Ritz values (without eig_host it used to return TDH_OK with an unconverged rotation); the next call works."""
    torch = torch_cuda
    cfg = W.CONFIGS["tiny"]
    wl = W.make(cfg)
    psi = oracle.orthonormalize(cfg.n, cfg.dv, W.states(cfg, 0, 8))
    with B.grid_for(wl, max_states=8) as g:
        d = torch.from_numpy(psi).cuda()
        h = g.apply_hamiltonian(d)
        bad = h.clone()
        bad[3, 1, 2, 3] = float("nan")
        with pytest.raises(B.TdhError) as err:
            g.subspace_diag(d, bad, want_eig=want_eig)
        assert err.value.code == B.TDH_ECUDA and "did not converge" in str(err.value)
        w, out = g.subspace_diag(d, h, want_eig=want_eig)
        assert (w is None) == (not want_eig)
        m = g.overlap(out, g.apply_hamiltonian(out)).cpu().numpy()
        assert np.abs(m - np.diag(np.diag(m))).max() < 1e-10 * max(1.0, np.abs(m).max())
        assert g.last_jacobi_sweeps() >= 1


def test_ground_state_iterations_converge_towards_the_lowest_eigenvalues(torch_cuda, B, oracle):
    """The eigensolver loop of PAPER.md:389-393 composed from the C-ABI calls (SD update, orthonormalisation, subspace
    diagonalisation) on a 16^3 grid: the trace over the subspace never increases, and the Ritz values stay above the lowest
    eigenvalues of the oracle's H (computed by Lanczos) and close most of the initial gap."""
    torch = torch_cuda
    cfg = W.test_config(280, (16, 16, 16), (7.0, 7.0, 7.0), nst=4, natoms=2, lmax=1, rc=2.0, dl=(1.5, -0.7))
    wl = W.make(cfg)
    with B.grid_for(wl) as g:
        d = g.orthonormalize(torch.from_numpy(W.states(cfg)).cuda())
        hist = []
        for it in range(30):
            g.sd_step(d, 0.4, want_eig=False)
            d = g.orthonormalize(d)
            w, d = g.subspace_diag(d, g.apply_hamiltonian(d))
            hist.append(w.copy())
        hist = np.array(hist)
        assert np.all(np.diff(hist.sum(axis=1)) < 1e-12)           # the trace over the subspace never increases
    # reference: the four lowest eigenvalues of the oracle's H by Lanczos (scipy) on the same 16^3 grid
    from scipy.sparse.linalg import LinearOperator, eigsh
    op = LinearOperator((cfg.npts, cfg.npts), dtype=np.complex128,
                        matvec=lambda x: oracle.apply_workload(wl, np.asarray(x, dtype=np.complex128).reshape((1,) + cfg.n),
                                                               oracle.NAIVE_FFT).ravel())
    ev = np.sort(eigsh(op, k=4, which="SA", tol=1e-10, return_eigenvectors=False))
    assert np.all(hist[-1] >= ev - 1e-8)                           # variational bound (Cauchy interlacing)
    assert hist[-1, 0] - ev[0] < 0.05 * (hist[0, 0] - ev[0])       # and the iteration has closed most of the gap


# ------------------------------------------------------------------------------------------------ NEXT-4: gradient, forces
@pytest.mark.parametrize("name,nst", [("tiny", 8), ("small", 11), ("medium", 5)])
def test_gradient_matches_oracle(torch_cuda, B, oracle, name, nst):
    """tdh_gradient (i (G_a + k_a) in Fourier space) for the three axes, whole and split planes, k != 0."""
    torch = torch_cuda
    cfg = W.CONFIGS[name]
    psi = W.states(cfg, 0, nst)
    with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, nst) as g:
        d = torch.from_numpy(psi).cuda()
        for a in range(3):
            ref = oracle.gradient(cfg.n, cfg.length, cfg.kpt, a, psi)
            assert per_state_rel(g.gradient(d, a).cpu().numpy(), ref).max() < TOL
    n = (16, 96, 96)
    cfg2 = W.test_config(290, n, (5.0, 30.0, 30.0), nst=2, natoms=0)
    psi = W.states(cfg2)
    with B.Grid(cfg2.n, cfg2.length, cfg2.kpt, -1.0, 2) as g:
        d = torch.from_numpy(psi).cuda()
        for a in range(3):
            assert per_state_rel(g.gradient(d, a).cpu().numpy(), oracle.gradient(cfg2.n, cfg2.length, cfg2.kpt, a, psi)).max() < TOL


@pytest.mark.parametrize("name,nst,chunk", [("tiny", 8, None), ("small", 13, 4), ("medium", 6, None)])
def test_forces_match_oracle(torch_cuda, B, oracle, name, nst, chunk):
    """tdh_forces (Eq. 11) against the oracle: non-local part alone and with per-atom local potentials, occupations."""
    torch = torch_cuda
    cfg = W.CONFIGS[name]
    wl = W.make(cfg)
    psi = W.states(cfg, 0, nst)
    rng = np.random.default_rng([W.BASE_SEED + cfg.cid, 14])
    occ = rng.uniform(0.2, 2.0, nst)
    import dataclasses
    one = dataclasses.replace(cfg, natoms=1)
    vloc = np.array([W.local_potential(one, wl.pos[i:i + 1]) for i in range(cfg.natoms)])
    with B.grid_for(wl, max_states=nst) as g:
        if chunk:
            g.set_chunk_states(chunk)
        d = torch.from_numpy(psi).cuda()
        for o, v in ((None, None), (occ, vloc)):
            ref = oracle.forces(cfg.n, cfg.length, cfg.kpt, wl.proj, psi, o, v)
            got = g.forces(d, cfg.natoms, o, None if v is None else torch.from_numpy(v).cuda())
            assert np.abs(got - ref).max() < 1e-10 * np.abs(ref).max(), (got, ref)


def test_new_entry_points_are_deterministic(torch_cuda, B):
    """No atomics on any data path (split-K partials, coloured scatter, ordered reductions, grid barriers): two runs of every
    NEXT entry point give bit-identical results."""
    torch = torch_cuda
    cfg = W.CONFIGS["small"]
    wl = W.make(cfg)
    nst = 24
    psi = torch.from_numpy(W.states(cfg, 0, nst)).cuda()

    def run():
        with B.grid_for(wl, max_states=nst) as g:
            q = g.orthonormalize(psi)
            h = g.apply_hamiltonian(q)
            w, r = g.subspace_diag(q, h)
            d = q.clone()
            eig = g.sd_step(d, 0.1)
            f = g.forces(q, cfg.natoms)
            n = g.density(q)
            vh = g.hartree(n)
            full = g.taylor_pair(d, 0.02)
            return [q.cpu().numpy(), g.overlap(q, h).cpu().numpy(), w, r.cpu().numpy(), eig, d.cpu().numpy(), f,
                    n.cpu().numpy(), vh.cpu().numpy(), full.cpu().numpy()]

    a, b = run(), run()
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_rotations_at_full_grid_size_sampled(torch_cuda, B, oracle):
    """Large grid (96^3), 256 states: sampled entries of the overlap matrix against the oracle's literal sums, unit overlap
    after tdh_orthonormalize, and sampled states of a rotation against the oracle."""
    torch = torch_cuda
    cfg = W.CONFIGS["large"]
    nst = 256
    sample = [0, 77, 255]
    psi, host = device_block(torch, cfg, nst, sample)
    with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, nst) as g:
        s = g.overlap(psi).cpu().numpy()
        ref = oracle.overlap(cfg.n, cfg.dv, host, host)
        assert np.abs(s[np.ix_(sample, sample)] - ref).max() < 1e-12
        q = g.orthonormalize(psi)
        assert np.abs(g.overlap(q).cpu().numpy() - np.eye(nst)).max() < 1e-12
        # a rotation that only mixes the sampled states into three output states
        rng = np.random.default_rng(31)
        m = np.zeros((nst, 3), dtype=np.complex128)
        m[sample, :] = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
        r = g.rotate(psi, torch.from_numpy(m).cuda()).cpu().numpy()
        assert per_state_rel(r, oracle.rotate(host, m[sample, :])).max() < 1e-13
    del psi, q
    torch.cuda.empty_cache()


def test_seeded_sweep_over_grid_shapes_and_options(torch_cuda, B, oracle, monkeypatch):
    """Sixteen seeded combinations of grid shape (every supported size on every axis), state count, atoms, channel set,
    Bloch vector, cutoff, chunking and back-projection path: apply and two Taylor steps against the oracle."""
    torch = torch_cuda
    rng = np.random.default_rng(20260501)
    sizes = [16, 32, 48, 64, 96]
    done = 0
    while done < 16:
        n = tuple(int(rng.choice(sizes)) for _ in range(3))
        if n[0] * n[1] * n[2] > 64 * 64 * 64:
            continue
        h = rng.uniform(0.3, 0.5)
        length = tuple(float(h * m * rng.uniform(0.9, 1.1)) for m in n)
        nst = int(rng.integers(1, 10))
        natoms = int(rng.integers(0, 5))
        lmax = int(rng.integers(0, 3))
        kw = dict(nst=nst, natoms=natoms, lmax=lmax, rc=float(min(2.6, 0.45 * min(length))), dl=(2.0, -0.8, 0.3)[: lmax + 1],
                  kfrac=tuple(float(rng.choice([0.0, 0.0, 0.25, -0.1])) for _ in range(3)))
        if rng.random() < 0.4:
            kw["ecut"] = float(rng.choice([15.0, 40.0]))
        cfg = W.test_config(500 + done, n, length, **kw)
        wl = W.make(cfg)
        psi = W.states(cfg)
        ref_h = oracle.apply_workload(wl, psi, oracle.NAIVE_FFT)
        ref_p = oracle.propagate_workload(wl, psi, dt=0.01, nsteps=2)
        monkeypatch.setenv("TDH_NL_MODE", str(done % 2))
        with B.grid_for(wl) as g:
            if rng.random() < 0.5:
                g.set_chunk_states(int(rng.integers(1, nst + 1)))
            d = torch.from_numpy(psi).cuda()
            assert per_state_rel(g.apply_hamiltonian(d).cpu().numpy(), ref_h).max() < TOL, (done, n, kw)
            g.propagate(d, 0.01, 2)
            assert per_state_rel(d.cpu().numpy(), ref_p).max() < TOL, (done, n, kw)
        done += 1


# ------------------------------------------------------------------------------------------------ rotations at the sizes bench.py times
def test_rotations_512_states_match_oracle(torch_cuda, B, oracle):
    """tdh_orthonormalize and tdh_subspace_diag at nst = 512 (the cooperative Cholesky and the eigensolver at the size
    bench.py times) against the oracle, all states, on a 32^3 grid (the oracle's literal loops stay affordable)."""
    torch = torch_cuda
    cfg = W.test_config(300, (32, 32, 32), (15.0, 15.0, 15.0), nst=512, natoms=6, lmax=1, rc=2.5, dl=(2.0, -0.8))
    wl = W.make(cfg)
    psi = W.states(cfg)
    q_ref = oracle.orthonormalize(cfg.n, cfg.dv, psi)
    h_ref = oracle.apply_workload(wl, q_ref, oracle.NAIVE_FFT)
    w_ref, out_ref, _ = oracle.subspace_diag(cfg.n, cfg.dv, q_ref, h_ref)
    with B.grid_for(wl) as g:
        q = g.orthonormalize(torch.from_numpy(psi).cuda())
        assert per_state_rel(q.cpu().numpy(), q_ref).max() < 1e-11
        assert np.abs(g.overlap(q).cpu().numpy() - np.eye(512)).max() < 1e-12
        qd = torch.from_numpy(q_ref).cuda()
        w, out = g.subspace_diag(qd, g.apply_hamiltonian(qd))
        assert np.abs(w - w_ref).max() < 1e-11 * max(1.0, np.abs(w_ref).max())
        assert np.abs(g.overlap(out).cpu().numpy() - np.eye(512)).max() < 1e-11
        ov = np.abs(np.diag(oracle.overlap(cfg.n, cfg.dv, out_ref, out.cpu().numpy())))
        gap = np.minimum(np.diff(w_ref, prepend=-np.inf), np.diff(w_ref, append=np.inf))
        sep = gap > 1e-4
        assert sep.sum() >= 256 and np.abs(ov[sep] - 1).max() < 1e-7


def test_rotations_tddft_block_properties(torch_cuda, B):
    """The TDDFT block (512 x 64^3), exactly what bench.py times: unit overlap after tdh_orthonormalize to 1e-12, and the
    Ritz values of tdh_subspace_diag equal LAPACK's eigenvalues of the same subspace matrix (read back with tdh_overlap)
    to 1e-11; psi'^H H psi' is diagonal."""
    torch = torch_cuda
    cfg = W.CONFIGS["tddft"]
    wl = W.make(cfg)
    nst = cfg.nst
    psi, _ = device_block(torch, cfg, nst, [0])
    with B.grid_for(wl, max_states=nst) as g:
        q = g.orthonormalize(psi)
        assert np.abs(g.overlap(q).cpu().numpy() - np.eye(nst)).max() < 1e-12
        h = g.apply_hamiltonian(q)
        m = g.overlap(q, h).cpu().numpy()
        w, out = g.subspace_diag(q, h, out=psi)
        w_lapack = np.linalg.eigvalsh(0.5 * (m + m.conj().T))
        assert np.abs(w - w_lapack).max() < 1e-11 * max(1.0, np.abs(w_lapack).max())
        m2 = g.overlap(out, g.apply_hamiltonian(out, out=h)).cpu().numpy()
        assert np.abs(m2 - np.diag(w)).max() < 1e-10 * max(1.0, np.abs(w).max())
    del psi, q, h
    torch.cuda.empty_cache()


def test_rotations_1024_states_smoke(torch_cuda, B, oracle):
    """The largest block the rotations accept (nst = 1024) on a 16^3 grid: orthonormalise, diagonalise, compare the Ritz
    values with the oracle and the overlap with the identity."""
    torch = torch_cuda
    cfg = W.test_config(301, (16, 16, 16), (10.0, 10.0, 10.0), nst=1024, natoms=2, lmax=0, rc=2.0, dl=(1.5,))
    wl = W.make(cfg)
    psi = W.states(cfg)
    q_ref = oracle.orthonormalize(cfg.n, cfg.dv, psi)
    w_ref, _, _ = oracle.subspace_diag(cfg.n, cfg.dv, q_ref, oracle.apply_workload(wl, q_ref, oracle.NAIVE_FFT))
    with B.grid_for(wl) as g:
        q = g.orthonormalize(torch.from_numpy(psi).cuda())
        assert np.abs(g.overlap(q).cpu().numpy() - np.eye(1024)).max() < 1e-12
        assert per_state_rel(q.cpu().numpy(), q_ref).max() < 1e-10       # 1024 compounded Gram-Schmidt columns
        w, out = g.subspace_diag(q, g.apply_hamiltonian(q))
        assert np.abs(w - w_ref).max() < 1e-10 * max(1.0, np.abs(w_ref).max())
        assert np.abs(g.overlap(out).cpu().numpy() - np.eye(1024)).max() < 1e-11
        with pytest.raises(B.TdhError) as e:
            g2 = B.Grid(cfg.n, cfg.length, max_states=1025)
            g2.orthonormalize(torch.zeros((1025,) + cfg.n, dtype=torch.complex128, device="cuda"))
        assert e.value.code == B.TDH_EUNSUPPORTED


# ------------------------------------------------------------------------------------------------ advisor findings (round 1)
def test_rejected_projector_table_keeps_the_installed_one(torch_cuda, B, oracle):
    """tdh_set_projectors validates and builds before it replaces: after a rejected table (index out of range) the handle
    still applies the previous projectors."""
    torch = torch_cuda
    cfg = W.CONFIGS["tiny"]
    wl = W.make(cfg)
    psi = W.states(cfg)
    ref = oracle.apply_workload(wl, psi, oracle.DIRECT)
    with B.grid_for(wl) as g:
        bad = W.Projectors(**{**wl.proj.__dict__})
        bad.sph_idx = wl.proj.sph_idx.copy()
        bad.sph_idx[5] = cfg.npts
        with pytest.raises(B.TdhError) as e:
            g.set_projectors(bad)
        assert e.value.code == B.TDH_EINDEX
        out = g.apply_hamiltonian(torch.from_numpy(psi).cuda()).cpu().numpy()
        assert per_state_rel(out, ref).max() < TOL
        assert g.natoms == cfg.natoms
        with pytest.raises(B.TdhError):
            g.forces(torch.from_numpy(psi).cuda(), natoms=cfg.natoms - 1)


@pytest.mark.parametrize("mode", ["0", "1"])
def test_projector_table_without_any_channel(torch_cuda, B, oracle, monkeypatch, mode):
    """Every atom has zero channels: V_nl = 0; on a split-tile grid (96 x 96 planes) the separate back-projection kernel
    has no 4-channel tile to launch."""
    torch = torch_cuda
    monkeypatch.setenv("TDH_NL_MODE", mode)
    n, length = (16, 96, 96), (5.0, 30.0, 30.0)
    cfg = W.test_config(302, n, length, nst=3, natoms=2, lmax=0, rc=2.0, dl=(1.0,))
    wl = W.make(cfg)
    pr = wl.proj
    empty = W.Projectors(natoms=2, sph_off=pr.sph_off, sph_idx=pr.sph_idx, sph_disp=pr.sph_disp,
                         chan_off=np.zeros(3, dtype=np.int32), beta=np.zeros(0), dcoef=np.zeros(0))
    psi = W.states(cfg)
    ref = oracle.apply_hamiltonian(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, None, psi, oracle.NAIVE_FFT)
    with B.grid_for(wl) as g:
        g.set_projectors(empty)
        d = torch.from_numpy(psi).cuda()
        assert per_state_rel(g.apply_hamiltonian(d).cpu().numpy(), ref).max() < TOL
        g.propagate(d, 0.01, 1)
        assert bool(torch.isfinite(torch.view_as_real(d)).all())


def test_rotate_detects_partial_overlap(torch_cuda, B):
    """out starting inside psi beyond the first min(n_in, n_out) states is an overlap too."""
    torch = torch_cuda
    n = (16, 16, 16)
    with B.Grid(n, (8.0, 8.0, 8.0), max_states=10) as g:
        psi = torch.zeros((10,) + n, dtype=torch.complex128, device="cuda")
        m = torch.zeros((10, 1), dtype=torch.complex128, device="cuda")
        with pytest.raises(B.TdhError) as e:
            g.rotate(psi, m, out=psi[5:6])
        assert e.value.code == B.TDH_EINVAL
        out = torch.empty((1,) + n, dtype=torch.complex128, device="cuda")
        g.rotate(psi, m, out=out)


def test_sd_step_state_without_kinetic_energy(torch_cuda, B, oracle):
    """Reading R19 for T_s <= 0 (a constant state at Gamma): finite, and equal to the oracle."""
    torch = torch_cuda
    cfg = W.test_config(303, (16, 32, 16), (6.0, 11.0, 6.0), nst=3, natoms=2, lmax=1, rc=2.0, dl=(1.3, -0.6))
    wl = W.make(cfg)
    psi = W.states(cfg)
    psi[1] = 0.3 - 0.2j
    ref, eig_ref = oracle.sd_step(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, wl.v, wl.proj, psi, 0.17, oracle.NAIVE_FFT)
    with B.grid_for(wl) as g:
        d = torch.from_numpy(psi).cuda()
        eig = g.sd_step(d, 0.17)
        out = d.cpu().numpy()
    assert np.isfinite(out).all() and np.abs(eig - eig_ref).max() < 1e-11 * np.abs(eig_ref).max()
    assert per_state_rel(out, ref).max() < TOL
