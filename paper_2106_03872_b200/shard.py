"""State sharding for multi-GPU runs (Fig. 7).

Each state's H psi and each Taylor chain is independent of every other state, so a block is split into contiguous
state ranges, one per rank, with V and the projector tables replicated.  There is no collective on the path of H|psi> and
of the Taylor steps; torch.distributed supplies the barrier and the max-over-ranks timing in bench.py, and the one real
exchange step of a self-consistent propagation: the sum of the per-shard densities (Eq. 1, "requires a parallel reduction
over states") -- one all-reduce of N_p doubles per step (NCCL over NVLink on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import types
from typing import Optional, Sequence, Tuple

import numpy as np


def state_range(rank: int, world: int, nst: int) -> Tuple[int, int]:
    """Contiguous [s0, s1) of rank `rank`; sizes differ by at most one, lower ranks get the larger shards."""
    if not (0 <= rank < world) or nst < 0:
        raise ValueError("bad rank / world / nst")
    base, rem = divmod(nst, world)
    s0 = rank * base + min(rank, rem)
    return s0, s0 + base + (1 if rank < rem else 0)


def max_over_ranks(seconds: float) -> float:
    """Max over ranks of a timing (the job is as slow as its slowest rank).  No-op without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(seconds)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([seconds], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def allreduce_density(dens):
    """Sum the per-rank partial densities (tdh_density of each rank's states) in place; no-op without a process group.

    `dens` is a float64 tensor of the grid's shape, on the GPU under NCCL, on the CPU under gloo.
    """
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(dens, op=dist.ReduceOp.SUM)
    return dens


# ----------------------------------------------------------------------------------------------------------------
# Slab decomposition of the grid (Fig. 6)
#
# Rank r of `world` holds, of every state, the planes x in [r n0/world, (r+1) n0/world) in real space and the rows
# Y in [r n1/world, (r+1) n1/world) of the work layout (all k_x, all k_z) in Fourier space.  The kernels store each value
# straight into the buffer of its owner; the two maps below are those store addresses restated on the host (they are what
# the gloo test checks and what a pack / send / unpack data plane would use).
# ----------------------------------------------------------------------------------------------------------------
def slab_planes(n0: int, rank: int, world: int) -> Tuple[int, int]:
    """[x0, x1) of the rank in real space."""
    if n0 % world or not (0 <= rank < world):
        raise ValueError("world must divide n0")
    return rank * (n0 // world), (rank + 1) * (n0 // world)


def slab_rows(n1: int, rank: int, world: int) -> Tuple[int, int]:
    """[Y0, Y1) work-layout rows of the rank in Fourier space (row pairs stay together: n1 / world is even)."""
    if n1 % (2 * world) or not (0 <= rank < world):
        raise ValueError("world must divide n1 / 2")
    return rank * (n1 // world), (rank + 1) * (n1 // world)


def fs_destination(n: Sequence[int], world: int, s: int, x: int, row: int):
    """(rank, element offset) of spectrum row `row` of plane x of state s in its owner's Fourier-space slab
    [state][n0][n1/world][n2] (the address tile_fwd stores to)."""
    nyl = n[1] // world
    q = row // nyl
    return q, ((s * n[0] + x) * nyl + (row - q * nyl)) * n[2]


def rs_destination(n: Sequence[int], world: int, s: int, x: int, row: int):
    """(rank, element offset) of row `row` of plane x of state s in its owner's real-space work block
    [state][n0/world][n1][n2] (the address the x-pencil kernel stores to)."""
    nxl = n[0] // world
    p = x // nxl
    return p, ((s * nxl + (x - p * nxl)) * n[1] + row) * n[2]


def slab_projectors(proj, n: Sequence[int], x0: int, x1: int):
    """The part of a projector table that lies in planes [x0, x1), with local flat indices ((x - x0) n1 + y) n2 + z.
    Every atom and every channel is kept (an atom may be left without points), so all ranks agree on the channel list."""
    if proj is None or proj.natoms == 0:
        return None
    plane = n[1] * n[2]
    sph_off, idx_all, disp_all, beta_all = [0], [], [], []
    boff = 0
    for a in range(proj.natoms):
        p0, p1 = int(proj.sph_off[a]), int(proj.sph_off[a + 1])
        nc = int(proj.chan_off[a + 1] - proj.chan_off[a])
        idx = np.asarray(proj.sph_idx[p0:p1], dtype=np.int64)
        keep = (idx // plane >= x0) & (idx // plane < x1)
        idx_all.append((idx[keep] - x0 * plane).astype(np.int32))
        if proj.sph_disp is not None:
            disp_all.append(np.asarray(proj.sph_disp[p0:p1])[keep])
        beta = np.asarray(proj.beta[boff:boff + nc * (p1 - p0)]).reshape(nc, p1 - p0)
        beta_all.append(beta[:, keep].ravel())
        boff += nc * (p1 - p0)
        sph_off.append(sph_off[-1] + int(keep.sum()))
    return types.SimpleNamespace(
        natoms=proj.natoms, sph_off=np.asarray(sph_off, dtype=np.int64),
        sph_idx=np.concatenate(idx_all).astype(np.int32) if idx_all else np.zeros(0, np.int32),
        sph_disp=None if proj.sph_disp is None else np.ascontiguousarray(np.concatenate(disp_all).reshape(-1, 3)),
        chan_off=np.asarray(proj.chan_off, dtype=np.int32), beta=np.concatenate(beta_all) if beta_all else np.zeros(0),
        dcoef=np.asarray(proj.dcoef, dtype=np.float64))


class SlabGroup:
    """All `world` ranks of a slab decomposition as handles on ONE device, driven phase by phase on one stream: the
    stream order is the barrier between the phases.  This is how the slab path is tested on a single GPU (no kernel ever
    waits for another one); with one process per GPU use SlabRank."""

    def __init__(self, n, length, kpt=(0.0, 0.0, 0.0), ecut=-1.0, max_states=1, world=2):
        from . import binding
        self.n, self.world = tuple(int(v) for v in n), int(world)
        self.grids = [binding.Grid(n, length, kpt, ecut, max_states, slab=(r, world)) for r in range(world)]
        self._connect()

    def _connect(self):
        bufs = [g.slab_buffers() for g in self.grids]
        for g in self.grids:
            g.slab_set_peers([b[0] for b in bufs], [b[1] for b in bufs],
                             [b[2] for b in bufs] if all(b[2] for b in bufs) else None)

    def close(self):
        for g in self.grids:
            g.close()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_potential(self, v):
        for r, g in enumerate(self.grids):
            x0, x1 = slab_planes(self.n[0], r, self.world)
            g.set_potential(None if v is None else v[x0:x1].contiguous())

    def set_projectors(self, proj):
        for r, g in enumerate(self.grids):
            x0, x1 = slab_planes(self.n[0], r, self.world)
            g.set_projectors(slab_projectors(proj, self.n, x0, x1))
        self._connect()

    def split(self, psi):
        """Full block (nst, n0, n1, n2) -> the ranks' real-space slabs (contiguous copies)."""
        return [psi[:, slice(*slab_planes(self.n[0], r, self.world))].contiguous() for r in range(self.world)]

    def apply(self, psi):
        """H psi of a full block, computed by the ranks' slab handles; returns the reassembled block."""
        import torch
        parts = self.split(psi)
        outs = [torch.empty_like(p) for p in parts]
        for phase in range(4):
            for g, p, o in zip(self.grids, parts, outs):
                g.slab_apply_phase(phase, p, o)
        return torch.cat(outs, dim=1)

    def fft_forward(self, psi):
        """Distributed forward transform; returns the ranks' spectrum slabs (nst, n0, n1/world, n2) in work layout."""
        parts = self.split(psi)
        for phase in range(2):
            for g, p in zip(self.grids, parts):
                g.slab_fft_phase(-1, phase, p)
        nyl = self.n[1] // self.world
        return [p.view(p.shape[0], self.n[0], nyl, self.n[2]) for p in parts]

    def fft_inverse(self, spec_parts):
        """Inverse of fft_forward (in place on the slabs); returns the reassembled real-space block."""
        import torch
        for phase in range(2):
            for g, p in zip(self.grids, spec_parts):
                g.slab_fft_phase(+1, phase, p)
        nxl = self.n[0] // self.world
        return torch.cat([p.view(p.shape[0], nxl, self.n[1], self.n[2]) for p in spec_parts], dim=1)


class SlabRank:
    """One rank of a slab decomposition in a one-process-per-GPU job (torch.distributed initialised).  The exchange
    buffers are shared through CUDA IPC, the data moves by the kernels' own stores into peer memory (NVLink between
    GPUs), and the barrier between the phases is a stream synchronisation followed by dist.barrier()."""

    def __init__(self, n, length, kpt=(0.0, 0.0, 0.0), ecut=-1.0, max_states=1):
        import torch.distributed as dist
        from . import binding
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.n = tuple(int(v) for v in n)
        self.grid = binding.Grid(n, length, kpt, ecut, max_states, slab=(self.rank, self.world))
        self._opened = []
        self.connect()

    def connect(self):
        import torch.distributed as dist
        from . import binding
        for p in self._opened:
            binding.ipc_close(p)
        self._opened = []
        mine = self.grid.slab_buffers()
        tokens = [None if not p else binding.ipc_export(p) for p in mine]
        everyone = [None] * self.world
        dist.all_gather_object(everyone, tokens)
        ptrs = []
        for r, toks in enumerate(everyone):
            if r == self.rank:
                ptrs.append(mine)
                continue
            row = []
            for t in toks:
                row.append(binding.ipc_import(t) if t is not None else 0)
                if t is not None:
                    self._opened.append(row[-1])
            ptrs.append(tuple(row))
        self.grid.slab_set_peers([p[0] for p in ptrs], [p[1] for p in ptrs],
                                 [p[2] for p in ptrs] if all(p[2] for p in ptrs) else None)

    def planes(self) -> Tuple[int, int]:
        return slab_planes(self.n[0], self.rank, self.world)

    def set_potential(self, v_local):
        self.grid.set_potential(v_local)

    def set_projectors(self, proj_full):
        """Collective.  tdh_set_projectors frees this rank's partial-projection buffer, which the peers have mapped through
        CUDA IPC and read in their PLANES_FWD phase: first every rank finishes its phases (barrier), then every rank
        closes its imports, and only after a second barrier -- nobody maps the old buffer any more -- is it freed and
        replaced; connect() exports and imports the new ones."""
        from . import binding
        self._barrier()
        for p in self._opened:
            binding.ipc_close(p)
        self._opened = []
        self._barrier()
        x0, x1 = self.planes()
        self.grid.set_projectors(slab_projectors(proj_full, self.n, x0, x1))
        self.connect()

    def _barrier(self):
        import torch
        import torch.distributed as dist
        torch.cuda.synchronize()
        dist.barrier()

    def apply(self, psi_local, out=None):
        """H psi on this rank's planes; collective: every rank calls it with the same number of states."""
        import torch
        if out is None:
            out = torch.empty_like(psi_local)
        self._barrier()
        for phase in range(4):
            self.grid.slab_apply_phase(phase, psi_local, out)
            self._barrier()
        return out

    def close(self):
        from . import binding
        self._barrier()
        for p in self._opened:
            binding.ipc_close(p)
        self._opened = []
        self.grid.close()
