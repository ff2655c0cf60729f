"""NEXT-4: slab decomposition of the grid (Fig. 6), all ranks emulated as handles on one
device and driven phase by phase (shard.SlabGroup): the reassembled H psi and the distributed transform against the
CPU oracle."""
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


CASES = [((32, 32, 32), 2, 1), ((32, 32, 32), 4, 1), ((64, 64, 64), 2, 1), ((64, 64, 64), 4, 2), ((96, 96, 96), 2, 1),
         ((96, 96, 96), 4, 1), ((32, 96, 64), 2, 2), ((48, 48, 16), 4, 0), ((16, 32, 48), 2, 1)]


@pytest.mark.parametrize("n,world,lmax", CASES)
def test_slab_apply_matches_oracle(torch_cuda, B, oracle, monkeypatch, n, world, lmax):
    """H psi (kinetic through the distributed transform, V, projectors whose spheres straddle the slab boundaries) of the
    reassembled block against the oracle; without projectors the slab path is bitwise the undivided one."""
    torch = torch_cuda
    from paper_2106_03872_b200 import shard
    big = n[0] * n[1] * n[2] > 64 ** 3
    kw = dict(kfrac=(0.25, 0.0, -0.1), ecut=25.0) if n == (64, 64, 64) and world == 4 else {}
    cfg = W.test_config(400 + world, n, tuple(0.4 * m for m in n), nst=2 if big else 5, natoms=6, lmax=lmax, rc=2.6,
                        dl=(2.0, -0.8, 0.3)[: lmax + 1], **kw)
    wl = W.make(cfg)
    psi = W.states(cfg)
    ref = oracle.apply_workload(wl, psi, oracle.NAIVE_FFT)
    nl = oracle.nonlocal_(cfg.n, cfg.length, cfg.kpt, wl.proj, psi)
    assert np.linalg.norm(nl) > 1e-5 * np.linalg.norm(ref)
    d = torch.from_numpy(psi).cuda()
    with shard.SlabGroup(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, cfg.nst, world) as sg:
        sg.set_potential(torch.from_numpy(wl.v).cuda())
        sg.set_projectors(wl.proj)
        out = sg.apply(d)
        torch.cuda.synchronize()
        err = per_state_rel(out.cpu().numpy(), ref)
        assert err.max() < TOL, err
        assert sum(g.last_launch_count() for g in sg.grids) >= 5 * world
        sg.set_projectors(None)
        out0 = sg.apply(d)
        # white-noise states make the kinetic term dominate: the non-local part is compared on its own as well
        # (a difference of two O(100) numbers: 1e-8 of its own norm is 1e-14 of theirs)
        assert per_state_rel((out - out0).cpu().numpy(), nl).max() < 1e-8
    monkeypatch.setenv("TDH_SMALL", "0")                    # the undivided TILED path (32^3 would run on chip otherwise)
    with B.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, cfg.nst) as g:
        g.set_potential(torch.from_numpy(wl.v).cuda())
        assert torch.equal(out0, g.apply_hamiltonian(d))


def test_new_projectors_disconnect_the_peers(torch_cuda, B):
    """tdh_set_projectors on a slab handle frees the partial-projection buffer the peers were given: until
    tdh_slab_set_peers has been called again every phase call of that handle is refused instead of reading freed memory."""
    torch = torch_cuda
    from paper_2106_03872_b200 import shard
    n = (32, 32, 32)
    cfg = W.test_config(431, n, tuple(0.4 * m for m in n), nst=2, natoms=3, lmax=1, rc=2.6, dl=(2.0, -0.8))
    wl = W.make(cfg)
    d = torch.from_numpy(W.states(cfg)).cuda()
    with shard.SlabGroup(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, cfg.nst, 2) as sg:
        sg.set_projectors(wl.proj)
        ref = sg.apply(d)
        parts = sg.split(d)
        g0 = sg.grids[0]
        g0.set_projectors(shard.slab_projectors(wl.proj, cfg.n, *shard.slab_planes(n[0], 0, 2)))
        for phase in range(4):
            with pytest.raises(B.TdhError) as err:
                g0.slab_apply_phase(phase, parts[0], torch.empty_like(parts[0]))
            assert err.value.code == B.TDH_EINVAL and "tdh_slab_set_peers" in str(err.value)
        sg._connect()
        assert torch.equal(sg.apply(d), ref)


@pytest.mark.parametrize("n,world", [((32, 32, 32), 2), ((64, 64, 64), 4), ((96, 96, 96), 4), ((16, 96, 32), 2)])
def test_slab_fft_matches_oracle(torch_cuda, B, oracle, n, world):
    """The distributed 3-D transform alone: the ranks' spectrum slabs, put back in natural order with the work-layout maps,
    equal the oracle's DFT; the inverse restores the block."""
    torch = torch_cuda
    from paper_2106_03872_b200 import shard
    rng = np.random.default_rng(sum(n) + world)
    nst = 2
    a = rng.standard_normal((nst,) + n) + 1j * rng.standard_normal((nst,) + n)
    ref = oracle.dft3d(a, -1, oracle.NAIVE_FFT)
    with shard.SlabGroup(n, (1.0, 1.0, 1.0), max_states=nst, world=world) as sg:
        parts = sg.fft_forward(torch.from_numpy(a).cuda())
        rowmap, colmap = sg.grids[0].work_layout()
        work = torch.cat(parts, dim=2).cpu().numpy()                       # [s][kx][Y][z'] with all rows
        spec = work[:, :, rowmap][:, :, :, colmap]                          # natural (ky, kz)
        assert per_state_rel(spec, ref).max() < 1e-13
        back = sg.fft_inverse(parts)
        assert per_state_rel(back.cpu().numpy(), a).max() < 1e-13


def test_slab_error_codes(torch_cuda, B):
    torch = torch_cuda
    for n, world in (((32, 32, 32), 3), ((16, 16, 16), 4), ((32, 32, 32), 9), ((32, 32, 32), 1)):
        with pytest.raises(B.TdhError) as e:
            B.Grid(n, (1.0, 1.0, 1.0), max_states=1, slab=(0, world))
        assert e.value.code in (B.TDH_EUNSUPPORTED, B.TDH_EINVAL)
    with B.Grid((32, 32, 32), (8.0, 8.0, 8.0), max_states=2, slab=(1, 2)) as g:
        psi = torch.zeros((2, 16, 32, 32), dtype=torch.complex128, device="cuda")
        with pytest.raises(B.TdhError) as e:                                 # peers not connected yet
            g.slab_apply_phase(0, psi, psi.clone())
        assert e.value.code == B.TDH_EINVAL
        with pytest.raises(B.TdhError) as e:                                 # whole-grid entry points refuse slab handles
            g.apply_hamiltonian(psi)
        assert e.value.code == B.TDH_EINVAL
        fs, rs, dp = g.slab_buffers()
        assert fs and rs and not dp
        with pytest.raises(B.TdhError):                                      # entry `rank` must be the handle's own buffers
            g.slab_set_peers([fs, fs], [fs, fs])


_IPC_WORKER = r"""
import sys
sys.path.insert(0, {root!r})
import numpy as np
import torch
import torch.distributed as dist
from paper_2106_03872_b200 import binding as B, shard, workloads as W
from oracle import ref
rank = int(sys.argv[1])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
torch.cuda.set_device(0)
cfg = W.test_config(410, (32, 48, 32), (12.0, 18.0, 12.0), nst=3, natoms=5, lmax=1, rc=2.6, dl=(2.0, -0.8))
wl = W.make(cfg)
psi = W.states(cfg)
try:
    sr = shard.SlabRank(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, cfg.nst)
except B.TdhError as e:
    print("IPC-UNAVAILABLE", e)
    sys.exit(0)
x0, x1 = sr.planes()
sr.set_potential(torch.from_numpy(np.ascontiguousarray(wl.v[x0:x1])).cuda())
sr.set_projectors(wl.proj)
out = sr.apply(torch.from_numpy(np.ascontiguousarray(psi[:, x0:x1])).cuda())
torch.cuda.synchronize()
expect = ref.apply_workload(wl, psi, ref.NAIVE_FFT)[:, x0:x1]
got = out.cpu().numpy()
err = np.linalg.norm((got - expect).reshape(cfg.nst, -1), axis=1) / np.linalg.norm(expect.reshape(cfg.nst, -1), axis=1)
assert err.max() < 1e-11, err
sr.close()
dist.destroy_process_group()
print("ok", rank)
"""


def test_slab_two_processes_share_buffers_through_cuda_ipc(torch_cuda, tmp_path):
    """shard.SlabRank: one process per rank (here both on the one GPU of the box), exchange buffers opened through CUDA IPC,
    the kernels of each process store into the other process's buffers, a host barrier between the phases (no kernel
    waits for another).  The rank's planes of H psi against the oracle."""
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    script = tmp_path / "ipc_worker.py"
    script.write_text(_IPC_WORKER.format(root=root, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
             for r in range(2)]
    outs = []
    for p in procs:
        try:
            outs.append(p.communicate(timeout=300)[0].decode())
        except subprocess.TimeoutExpired:
            for q in procs:
                q.kill()
            pytest.fail("slab IPC workers timed out")
    if any("IPC-UNAVAILABLE" in o for o in outs):
        pytest.skip("CUDA IPC is not available in this container: " + outs[0][-300:])
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o
