"""The one-launch on-chip path for 16^3 and 32^3 grids (small_kernels.cuh) against the oracle, and against the tiled
four-launch path (TDH_SMALL=0) that the same grids ran before: both must match the oracle on every case."""
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


@pytest.mark.parametrize("small", ["1", "0"])
@pytest.mark.parametrize("name", ["tiny", "small"])
def test_configs_apply_and_propagate_both_paths(torch_cuda, B, oracle, monkeypatch, name, small):
    """Configs 1 and 2 in full: apply and six Taylor-4 steps; one launch per application on the on-chip path."""
    torch = torch_cuda
    monkeypatch.setenv("TDH_SMALL", small)
    cfg = W.CONFIGS[name]
    wl = W.make(cfg)
    psi = W.states(cfg)
    ref_h = oracle.apply_workload(wl, psi, oracle.NAIVE_FFT)
    nsteps = 6 if name == "tiny" else 2
    ref_p = oracle.propagate_workload(wl, psi, dt=cfg.dt, nsteps=nsteps, backend=oracle.NAIVE_FFT)
    with B.grid_for(wl) as g:
        d = torch.from_numpy(psi).cuda()
        out = g.apply_hamiltonian(d)
        assert g.last_launch_count() == (1 if small == "1" else 4)
        assert per_state_rel(out.cpu().numpy(), ref_h).max() < TOL
        g.propagate(d, cfg.dt, nsteps)
        assert g.last_launch_count() == nsteps * 4 * (1 if small == "1" else 4)
        assert per_state_rel(d.cpu().numpy(), ref_p).max() < TOL


@pytest.mark.parametrize("n,nst,natoms,lmax,kfrac,ecut", [
    (16, 5, 3, 2, (0.25, 0.0, -0.1), 12.0), (32, 7, 6, 2, (0.1, 0.2, 0.0), 25.0), (16, 1, 0, 0, (0.0, 0.0, 0.0), None),
    (32, 3, 9, 1, (0.0, 0.0, 0.0), None), (16, 9, 4, 0, (0.0, 0.0, 0.3), None)])
def test_small_path_options(torch_cuda, B, oracle, n, nst, natoms, lmax, kfrac, ecut):
    """Bloch vector with phases in the projectors, cutoff mask, 1 / 4 / 9 channels, overlapping spheres (rc close to L/2),
    no atoms, no potential, ragged chunks; the non-local part on its own as well."""
    torch = torch_cuda
    length = (0.4 * n,) * 3
    cfg = W.test_config(700 + n + nst, (n, n, n), length, nst=nst, natoms=natoms, lmax=lmax, rc=0.45 * length[0],
                        dl=(2.0, -0.8, 0.3)[: lmax + 1], kfrac=kfrac, ecut=ecut)
    wl = W.make(cfg)
    psi = W.states(cfg)
    ref_h = oracle.apply_workload(wl, psi, oracle.NAIVE_FFT)
    ref_p = oracle.propagate_workload(wl, psi, dt=0.01, nsteps=2, backend=oracle.NAIVE_FFT)
    with B.grid_for(wl) as g:
        for chunk in (None, 2):
            if chunk:
                g.set_chunk_states(chunk)
            d = torch.from_numpy(psi).cuda()
            out = g.apply_hamiltonian(d)
            assert g.last_launch_count() == (1 if chunk is None else (nst + 1) // 2)
            assert per_state_rel(out.cpu().numpy(), ref_h).max() < TOL
            g.propagate(d, 0.01, 2)
            assert per_state_rel(d.cpu().numpy(), ref_p).max() < TOL
        if natoms:
            nl = oracle.nonlocal_(cfg.n, cfg.length, cfg.kpt, wl.proj, psi)
            g.set_projectors(None)
            out0 = g.apply_hamiltonian(torch.from_numpy(psi).cuda())
            assert per_state_rel((out - out0).cpu().numpy(), nl).max() < 1e-8
            g.set_potential(None)
            t_only = g.apply_hamiltonian(torch.from_numpy(psi).cuda()).cpu().numpy()
            assert per_state_rel(t_only, oracle.kinetic(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, psi, oracle.NAIVE_FFT)).max() < TOL


def test_small_path_many_channels_and_layers(torch_cuda, B, oracle):
    """16 channels per atom and grid points covered by four spheres (record layers), on both on-chip grids."""
    torch = torch_cuda
    from test_gpu_fullsize import synthetic_projectors
    for n in (16, 32):
        length = (0.42 * n,) * 3
        cfg = W.test_config(720 + n, (n, n, n), length, nst=4, natoms=1, lmax=0, rc=0.4 * length[0], dl=(1.0,),
                            kfrac=(0.0, 0.25, 0.0))
        rng = np.random.default_rng([W.BASE_SEED, 720, n])
        mid = [0.5 * l for l in length]
        centers = [mid, [mid[0] + 0.3, mid[1], mid[2]], [mid[0], mid[1] - 0.4, mid[2] + 0.2], [mid[0] + 0.1, mid[1] + 0.1, mid[2]],
                   [0.1, 0.2, length[2] - 0.1]]
        proj = synthetic_projectors(cfg, centers, 16, rng)
        v = rng.uniform(-1.0, 1.0, cfg.n)
        psi = W.states(cfg)
        ref = oracle.apply_hamiltonian(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, v, proj, psi, oracle.NAIVE_FFT)
        with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, cfg.nst) as g:
            g.set_potential(torch.from_numpy(v).cuda())
            g.set_projectors(proj)
            out = g.apply_hamiltonian(torch.from_numpy(psi).cuda())
            assert g.last_launch_count() == 1
            assert per_state_rel(out.cpu().numpy(), ref).max() < TOL


def test_small_path_is_deterministic_and_independent_of_batching(torch_cuda, B):
    torch = torch_cuda
    cfg = W.CONFIGS["small"]
    wl = W.make(cfg)
    psi = torch.from_numpy(W.states(cfg, 0, 20)).cuda()
    with B.grid_for(wl, max_states=20) as g:
        a = g.apply_hamiltonian(psi)
        b = g.apply_hamiltonian(psi)
        assert torch.equal(a, b)
        part = g.apply_hamiltonian(psi[5:12].contiguous())
        assert torch.equal(part, a[5:12])


@pytest.mark.parametrize("small", ["0", "1"])
def test_small_planes_many_states_stress(torch_cuda, B, oracle, monkeypatch, small):
    """32^3 with 1024 states (one launch chain over the whole 512 MB block) through both paths, forty applications with
    re-created handles and tensors, every application bitwise the first.  Regression test for the phase-parity race of
    the tile ring: before the armed flags of tile_kernels.cuh such launches failed, or returned
    wrong values, in most processes; sampled states against the oracle."""
    torch = torch_cuda
    import dataclasses
    monkeypatch.setenv("TDH_SMALL", small)
    cfg = dataclasses.replace(W.CONFIGS["small"], nst=1024)
    wl = W.make(cfg)
    sample = [0, 300, 1023]
    host = np.stack([W.state(cfg, s) for s in sample])
    ref = oracle.apply_workload(wl, host, oracle.NAIVE_FFT)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(5)
    for trial in range(5):
        psi = torch.empty((cfg.nst,) + cfg.n, dtype=torch.complex128, device="cuda")
        torch.view_as_real(psi).copy_(torch.randn((cfg.nst,) + cfg.n + (2,), dtype=torch.float64, device="cuda", generator=gen) * 0.01)
        for j, s in enumerate(sample):
            psi[s].copy_(torch.from_numpy(host[j]))
        out = torch.empty_like(psi)
        with B.grid_for(wl) as g:
            first = g.apply_hamiltonian(psi)
            for _ in range(8):
                g.apply_hamiltonian(psi, out=out)
                assert torch.equal(out, first)
            torch.cuda.synchronize()
            assert g.last_launch_count() == (4 if small == "0" else 1)          # one chunk: no bound on a launch
            del first
            got = np.stack([out[s].cpu().numpy() for s in sample])
            assert per_state_rel(got, ref).max() < TOL
        del psi, out
        torch.cuda.empty_cache()


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_propagate_graph_replay_and_invalidation(torch_cuda, B, oracle, monkeypatch, name):
    """tdh_propagate on small blocks replays a captured CUDA graph.  A replay (same buffer, same arguments) must continue the
    propagation exactly as plain launches do, another buffer or step count must not reuse the frozen arguments, and a
    new potential must invalidate the graph (the kernels' arguments are frozen at capture)."""
    torch = torch_cuda
    cfg = W.CONFIGS[name]
    wl = W.make(cfg)
    nst = cfg.nst if name == "tiny" else 6
    psi = W.states(cfg, 0, nst)
    dt = cfg.dt
    rng = np.random.default_rng([W.BASE_SEED + cfg.cid, 11])
    v2 = wl.v + rng.uniform(-0.3, 0.3, wl.v.shape)
    wl2 = W.Workload(cfg=cfg, pos=wl.pos, v=v2, proj=wl.proj)
    ref_a = oracle.propagate_workload(wl, psi, dt=dt, nsteps=2, backend=oracle.NAIVE_FFT)        # first call
    ref_b = oracle.propagate_workload(wl, ref_a, dt=dt, nsteps=2, backend=oracle.NAIVE_FFT)      # replay
    ref_c = oracle.propagate_workload(wl2, ref_b, dt=dt, nsteps=2, backend=oracle.NAIVE_FFT)     # new potential
    ref_d = oracle.propagate_workload(wl2, psi, dt=dt, nsteps=1, backend=oracle.NAIVE_FFT)       # other buffer and count
    results = {}
    for graph in ("1", "0"):
        monkeypatch.setenv("TDH_GRAPH", graph)
        with B.grid_for(wl, max_states=nst) as g:
            d = torch.from_numpy(psi).cuda()
            g.propagate(d, dt, 2)
            a = d.cpu().numpy()
            g.propagate(d, dt, 2)
            b = d.cpu().numpy()
            g.set_potential(torch.from_numpy(v2).cuda())
            g.propagate(d, dt, 2)
            c = d.cpu().numpy()
            e = torch.from_numpy(psi).cuda()
            g.set_chunk_states(3)                                    # several chunks inside one captured call
            g.propagate(e, dt, 1)
            dd = e.cpu().numpy()
            assert g.last_launch_count() == 4 * (g.last_launch_count() // 4)
        for got, ref in ((a, ref_a), (b, ref_b), (c, ref_c), (dd, ref_d)):
            assert per_state_rel(got, ref).max() < TOL
        results[graph] = (a, b, c, dd)
    for x, y in zip(results["1"], results["0"]):
        assert np.array_equal(x, y)                                  # the graph replays the same kernels: bitwise equal


@pytest.mark.parametrize("cluster", ["1", "0"])
def test_16cubed_cluster_and_single_cta_variants(torch_cuda, B, oracle, monkeypatch, cluster):
    """16^3 blocks of few states run a cluster of four CTAs per state (radix-4 local x transform, radix-4 over distributed
    shared memory), blocks of many states one CTA per state: both against the oracle, with projectors of 1 and 9 channels,
    k != 0 and a cutoff; 40 states make the library switch to one CTA per state by itself."""
    torch = torch_cuda
    monkeypatch.setenv("TDH_SMALL16_CLUSTER", cluster)
    for cid, nst, natoms, lmax, kfrac, ecut in ((910, 8, 2, 0, (0.0, 0.0, 0.0), None), (911, 5, 3, 2, (0.25, 0.0, -0.1), 12.0),
                                                (912, 40, 2, 1, (0.0, 0.0, 0.0), None)):
        kw = dict(nst=nst, natoms=natoms, lmax=lmax, rc=2.0, dl=(1.5, -0.8, 0.3)[: lmax + 1], kfrac=kfrac)
        if ecut:
            kw["ecut"] = ecut
        cfg = W.test_config(cid, (16, 16, 16), (10.0, 10.0, 10.0), **kw)
        wl = W.make(cfg)
        psi = W.states(cfg)
        ref_h = oracle.apply_workload(wl, psi, oracle.DIRECT)
        ref_p = oracle.propagate_workload(wl, psi, dt=0.02, nsteps=2, backend=oracle.DIRECT)
        with B.grid_for(wl) as g:
            d = torch.from_numpy(psi).cuda()
            out = g.apply_hamiltonian(d)
            assert g.last_launch_count() == 1
            assert per_state_rel(out.cpu().numpy(), ref_h).max() < TOL, (cid, cluster)
            g.propagate(d, 0.02, 2)
            assert per_state_rel(d.cpu().numpy(), ref_p).max() < TOL, (cid, cluster)
