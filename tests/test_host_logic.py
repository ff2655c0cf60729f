"""CPU-only checks: the C-ABI library loads and exports every declared symbol, fails loudly without a GPU,
the generator is deterministic, and the multi-rank sharding logic works under gloo with world_size 2."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2106_03872_b200 import shard
from paper_2106_03872_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tdh_lib():
    from paper_2106_03872_b200 import build, binding
    build.build()
    return binding.lib()


def test_library_exports_every_declared_symbol(tdh_lib):
    from paper_2106_03872_b200 import binding
    header = open(os.path.join(ROOT, "include", "tdh.h")).read()
    declared = set(re.findall(r"\b(tdh_[a-z0-9_]+)\s*\(", header))
    declared -= {"tdh_grid", "tdh_c128"}
    assert declared == set(binding.SYMBOLS)
    for name in declared:
        assert hasattr(tdh_lib, name), name
    assert isinstance(tdh_lib.tdh_last_error(), bytes)
    assert tdh_lib.tdh_kernel_name(0) == b"nl_project"


def test_argument_checks_need_no_gpu(tdh_lib):
    """Invalid arguments are rejected before any CUDA call."""
    h = ctypes.c_void_p()
    n = (ctypes.c_int * 3)(20, 16, 16)
    l3 = (ctypes.c_double * 3)(1.0, 1.0, 1.0)
    k3 = (ctypes.c_double * 3)(0.0, 0.0, 0.0)
    assert tdh_lib.tdh_create_grid(n, l3, k3, -1.0, 1, None, ctypes.byref(h)) == -2
    assert b"unsupported" in tdh_lib.tdh_last_error()
    n = (ctypes.c_int * 3)(16, 16, 16)
    assert tdh_lib.tdh_create_grid(n, l3, k3, -1.0, 0, None, ctypes.byref(h)) == -1
    assert tdh_lib.tdh_create_grid(None, l3, k3, -1.0, 1, None, ctypes.byref(h)) == -1
    assert tdh_lib.tdh_apply_hamiltonian(None, 1, None, None) == -1
    assert tdh_lib.tdh_destroy_grid(None) == 0


def test_product_fails_loudly_without_gpu(tdh_lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2106_03872_b200 import binding
    with pytest.raises(binding.TdhError):
        binding.Grid((16, 16, 16), (1.0, 1.0, 1.0))
    h = ctypes.c_void_p()
    n = (ctypes.c_int * 3)(16, 16, 16)
    l3 = (ctypes.c_double * 3)(1.0, 1.0, 1.0)
    k3 = (ctypes.c_double * 3)(0.0, 0.0, 0.0)
    assert tdh_lib.tdh_create_grid(n, l3, k3, -1.0, 1, None, ctypes.byref(h)) == -4     # TDH_ECUDA, no fallback


def test_product_does_not_import_oracle():
    """The package must never reach into oracle/ (a product path through the oracle voids parity)."""
    pkg = os.path.join(ROOT, "paper_2106_03872_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "ref_tdh" not in text, f
    for f in ("ref_tdh.c", "ref.py", "build.py"):
        text = open(os.path.join(ROOT, "oracle", f)).read()
        assert "paper_2106_03872_b200" not in text.replace("paper_2106_03872_b200/csrc", ""), f


def test_generator_is_deterministic_and_shaped():
    for name in W.CONFIG_ORDER:
        cfg = W.CONFIGS[name]
        pos = W.atom_positions(cfg)
        assert pos.shape == (cfg.natoms, 3) and (pos >= 0).all() and (pos < cfg.length[0]).all()
        assert np.array_equal(pos, W.atom_positions(cfg))
    cfg = W.CONFIGS["small"]
    wl = W.make(cfg)
    assert wl.v.shape == cfg.n and wl.v.min() < -3.0
    pr = wl.proj
    assert pr.chan_off[-1] == 8 * 4 and len(pr.beta) == 4 * len(pr.sph_idx)
    per_sphere = np.diff(pr.sph_off)
    assert 600 < per_sphere.min() and per_sphere.max() < 680          # P = 636 [627-647]
    a = W.state(cfg, 5)
    assert abs(cfg.dv * np.sum(np.abs(a) ** 2) - 1.0) < 1e-12
    # sphere membership is strict |d| < rc and displacements are minimum images
    r = np.linalg.norm(pr.sph_disp, axis=1)
    assert r.max() < cfg.rc
    # large config: overlapping spheres along x (R13)
    big = W.CONFIGS["large"]
    p2 = W.atom_positions(big)
    assert len(p2) == 128


def test_state_range_partitions():
    for nst in (0, 1, 7, 64, 1024):
        for world in (1, 2, 3, 8):
            cover = []
            for r in range(world):
                s0, s1 = shard.state_range(r, world, nst)
                assert 0 <= s0 <= s1 <= nst
                cover += list(range(s0, s1))
            assert cover == list(range(nst))
            sizes = [shard.state_range(r, world, nst)[1] - shard.state_range(r, world, nst)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2106_03872_b200 import shard
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
s0, s1 = shard.state_range(rank, 2, 9)
got = [None, None]
dist.all_gather_object(got, (s0, s1))
assert got == [(0, 5), (5, 9)], got
t = shard.max_over_ranks(1.0 + rank)
assert t == 2.0, t
# NEXT-2: the density of a state block is the all-reduced sum of the shard densities (Eq. 1, PAPER.md:474)
import numpy as np
from paper_2106_03872_b200 import workloads as W
cfg = W.test_config(150, (4, 3, 5), (4.0, 3.0, 5.0), nst=9, natoms=0)
psi = W.states(cfg)
occ = np.linspace(0.5, 2.0, 9)
part = torch.from_numpy(np.einsum("s,sxyz->xyz", occ[s0:s1], np.abs(psi[s0:s1]) ** 2))
shard.allreduce_density(part)
full = np.einsum("s,sxyz->xyz", occ, np.abs(psi) ** 2)
assert np.abs(part.numpy() - full).max() < 1e-14 * full.max()
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_world_size_2_gloo(tmp_path):
    """N>1 path on CPU: two gloo ranks shard the states with no data-path collective and agree on the max time."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
             for r in range(2)]
    outs = [p.communicate(timeout=120)[0].decode() for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o


_SLAB_WORKER = r"""
import sys
sys.path.insert(0, {root!r})
import numpy as np
import torch
import torch.distributed as dist
from paper_2106_03872_b200 import shard
WORLD = 2
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=WORLD)
rank = dist.get_rank()
n, nst = (8, 12, 5), 3
nxl, nyl = n[0] // WORLD, n[1] // WORLD
# every element of the global block carries its own global index
A = torch.arange(nst * n[0] * n[1] * n[2], dtype=torch.float64).reshape(nst, *n)
x0, x1 = shard.slab_planes(n[0], rank, WORLD)
y0, y1 = shard.slab_rows(n[1], rank, WORLD)
mine = A[:, x0:x1].contiguous()


def route(src, planes, rows_of, dest_fn, dest_shape):
    # send every row of `src` to the rank and offset `dest_fn` names (grouped isend / irecv); returns the filled buffer
    rows = [[] for _ in range(WORLD)]
    offs = [[] for _ in range(WORLD)]
    for s in range(nst):
        for xi, x in enumerate(planes):
            for ri, row in enumerate(rows_of):
                q, off = dest_fn(n, WORLD, s, x, row)
                rows[q].append(src[s, xi, ri])
                offs[q].append(off)
    send_d = [torch.stack(r) for r in rows]
    send_o = [torch.tensor(o, dtype=torch.int64) for o in offs]
    recv_d = [torch.empty_like(send_d[q]) for q in range(WORLD)]      # the partition is even: equal counts both ways
    recv_o = [torch.empty_like(send_o[q]) for q in range(WORLD)]
    ops = []
    for q in range(WORLD):
        if q == rank:
            recv_d[q], recv_o[q] = send_d[q], send_o[q]
            continue
        ops += [dist.P2POp(dist.isend, send_d[q], q, tag=1), dist.P2POp(dist.irecv, recv_d[q], q, tag=1)]
        ops += [dist.P2POp(dist.isend, send_o[q], q, tag=2), dist.P2POp(dist.irecv, recv_o[q], q, tag=2)]
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    buf = torch.full((int(np.prod(dest_shape)),), -1.0, dtype=torch.float64)
    for q in range(WORLD):
        for row, off in zip(recv_d[q], recv_o[q].tolist()):
            assert (buf[off:off + n[2]] == -1.0).all(), "two rows landed on one address"
            buf[off:off + n[2]] = row
    assert (buf >= 0).all(), "a row of the slab was never written"
    return buf.reshape(dest_shape)


# forward exchange: my planes, all rows -> the owners of the rows
fs = route(mine, range(x0, x1), range(n[1]), shard.fs_destination, (nst, n[0], nyl, n[2]))
assert torch.equal(fs, A[:, :, y0:y1]), "Fourier-space slab is not rows [y0, y1) of all planes"
# way back: my rows, all planes -> the owners of the planes
rs = route(fs, range(n[0]), range(y0, y1), shard.rs_destination, (nst, nxl, n[1], n[2]))
assert torch.equal(rs, mine), "the way back does not restore the real-space slab"

# projector tables: the ranks' parts are a partition of the table, with local indices and the full channel list
from paper_2106_03872_b200 import workloads as W
cfg = W.test_config(160, (8, 12, 6), (4.0, 6.0, 3.0), nst=1, natoms=3, lmax=1, rc=1.4, dl=(1.0, -0.5))
pr = W.projectors(cfg)
part = shard.slab_projectors(pr, cfg.n, *shard.slab_planes(cfg.n[0], rank, WORLD))
assert part.natoms == pr.natoms and np.array_equal(part.chan_off, pr.chan_off) and np.array_equal(part.dcoef, pr.dcoef)
plane = cfg.n[1] * cfg.n[2]
xs0 = shard.slab_planes(cfg.n[0], rank, WORLD)[0]
counts = [int(part.sph_off[a + 1] - part.sph_off[a]) for a in range(pr.natoms)]
allc = [None] * WORLD
dist.all_gather_object(allc, counts)
assert [sum(c[a] for c in allc) for a in range(pr.natoms)] == [int(pr.sph_off[a + 1] - pr.sph_off[a]) for a in range(pr.natoms)]
boff_p = boff_f = 0
for a in range(pr.natoms):
    nc = int(pr.chan_off[a + 1] - pr.chan_off[a])
    f0, f1 = int(pr.sph_off[a]), int(pr.sph_off[a + 1])
    p0, p1 = int(part.sph_off[a]), int(part.sph_off[a + 1])
    full_idx = pr.sph_idx[f0:f1].astype(np.int64)
    keep = (full_idx // plane >= xs0) & (full_idx // plane < xs0 + cfg.n[0] // WORLD)
    assert np.array_equal(part.sph_idx[p0:p1].astype(np.int64) + xs0 * plane, full_idx[keep])
    assert np.array_equal(part.sph_disp[p0:p1], pr.sph_disp[f0:f1][keep])
    bf = pr.beta[boff_f:boff_f + nc * (f1 - f0)].reshape(nc, f1 - f0)
    bp = part.beta[boff_p:boff_p + nc * (p1 - p0)].reshape(nc, p1 - p0)
    assert np.array_equal(bp, bf[:, keep])
    boff_f += nc * (f1 - f0)
    boff_p += nc * (p1 - p0)
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_slab_index_maps_world_size_2_gloo(tmp_path):
    """NEXT-4: the two store-address maps of the slab decomposition (shard.fs_destination / rs_destination: the addresses
    the tile_fwd and x-pencil kernels store to) route a block between two gloo ranks with grouped isend / irecv: every row
    lands exactly once, the Fourier-space slab is rows [y0, y1) of all planes, the way back restores the planes; the ranks'
    projector tables partition the full one."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    script = tmp_path / "slab_worker.py"
    script.write_text(_SLAB_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
             for r in range(2)]
    outs = [p.communicate(timeout=180)[0].decode() for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o


def test_bench_reference_arm_prints_the_contract_line():
    """bench.py --impl reference runs the oracle on the host cores and prints one JSON line with the contract's keys."""
    import json
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny",
                        "--steps", "2", "--warmup", "1", "--cpu-sample-states", "2"], capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["higher_is_better"] is True and line["value"] > 0
    assert line["unit"] == "states*gridpoints/s" and line["steps"] == 2 and line["warmup"] == 1
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0


def test_bench_own_arm_refuses_to_run_without_a_gpu():
    """No CPU fallback: the product arm of bench.py exits with an error when there is no CUDA device."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)


def test_twiddle_table_of_the_fft_codelets():
    """csrc/twiddle48.h holds cos(2 pi k / 48), k = 0..12, as literals (made once with 60-digit decimal arithmetic): each
    agrees with the C library's cosine to one unit in the last place, and the exactly representable ones are exact."""
    import math
    text = open(os.path.join(ROOT, "paper_2106_03872_b200", "csrc", "twiddle48.h")).read()
    vals = [float(v) for v in re.findall(r"^\s+([0-9.eE+-]+),? /\* k=\d+ \*/", text, flags=re.M)]
    assert len(vals) == 13
    for k, v in enumerate(vals):
        assert abs(v - math.cos(2 * math.pi * k / 48)) <= 2.0 ** -52, k
    assert vals[0] == 1.0 and vals[8] == 0.5 and abs(vals[12]) < 1e-16
