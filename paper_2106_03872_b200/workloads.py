"""Seeded synthetic workloads (BASELINE.json ``configs``).

This module only *makes inputs*: atom positions, the local potential V(r) as an array, the
Kleinman-Bylander projector tables (sphere index lists, real beta values, D coefficients) and the
orbital block psi.  It contains none of the method's arithmetic (no FFT, no Hamiltonian, no
propagator) and is the one module that both the CUDA path's tests/bench and the CPU oracle's
tests are allowed to share.  Everything is numpy on the host.

The inputs stand in for the paper's workloads (N2 / H2O in a box, 8-atom Si cell, Al supercell;
PAPER.md:104,533,541,563) whose pseudopotential files are not available here; shapes and sizes
follow BASELINE.json.  Readings R11-R14 of SURVEY.md section 8(c) are implemented here.

Seeds: config c (1..5) has base seed 210603870 + c.  ``default_rng([base, 0])`` draws atom
positions (or lattice jitter), ``default_rng([base, 1])`` the potential noise (config 1),
``default_rng([base, 2, s])`` state s (N_p real parts, then N_p imaginary parts, standard normal,
then normalised so that dV * sum |psi|^2 = 1).  Per-state seeding makes a state independent of
the block it is generated in (PAPER.md:397-399 in spirit).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence, Tuple

import numpy as np

BASE_SEED = 210603870


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    cid: int                                  # 1..5 for the BASELINE configs, >=100 for test-only configs
    n: Tuple[int, int, int]                   # grid points per axis
    length: Tuple[float, float, float]        # cell lengths (bohr)
    nst: int                                  # number of states
    natoms: int
    placement: str                            # "uniform" | "lattice"
    lattice: Tuple[int, int, int] = (1, 1, 1)  # sites per axis for "lattice" (R13)
    jitter: float = 0.2
    well_z: float = 4.0                       # V = -Z sum_I exp(-|r-R_I|^2 / (2 sigma^2))   (R12)
    well_sigma: float = 0.7
    noise: float = 0.0                        # uniform +-noise added per grid point (config 1)
    lmax: int = 0                             # projector channels l = 0..lmax, m = -l..l
    proj_sigma: float = 0.6
    rc: float = 2.0                           # projector sphere radius, strict |d| < rc   (R4)
    dl: Tuple[float, ...] = (1.5,)            # KB coefficient per l                          (R3)
    kfrac: Tuple[float, float, float] = (0.0, 0.0, 0.0)   # k in units of 2 pi / L_a
    ecut: Optional[float] = None              # Ha; None = no mask
    dt: float = 0.02
    nsteps: int = 20

    @property
    def npts(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]

    @property
    def spacing(self) -> Tuple[float, float, float]:
        return tuple(self.length[a] / self.n[a] for a in range(3))

    @property
    def dv(self) -> float:
        h = self.spacing
        return h[0] * h[1] * h[2]

    @property
    def kpt(self) -> np.ndarray:
        return np.array([2.0 * math.pi * self.kfrac[a] / self.length[a] for a in range(3)])

    @property
    def ecut_abi(self) -> float:
        """Value passed through the ABI: <= 0 means 'no mask'."""
        return -1.0 if self.ecut is None else float(self.ecut)

    @property
    def nchan_per_atom(self) -> int:
        return (self.lmax + 1) ** 2


def _cubic(name, cid, L, N, **kw) -> Config:
    return Config(name=name, cid=cid, n=(N, N, N), length=(float(L),) * 3, **kw)


#: The five BASELINE.json configs, in order (index 0 = Tiny ... 4 = TDDFT).
CONFIGS = {
    "tiny": _cubic("tiny", 1, 10.0, 16, nst=8, natoms=2, placement="uniform",
                   well_z=2.0, well_sigma=0.8, noise=0.01, lmax=0, proj_sigma=0.6, rc=2.0, dl=(1.5,)),
    "small": _cubic("small", 2, 15.0, 32, nst=64, natoms=8, placement="uniform",
                    well_z=4.0, well_sigma=0.7, lmax=1, proj_sigma=0.6, rc=2.5, dl=(2.0, -0.8)),
    "medium": _cubic("medium", 3, 20.0, 48, nst=256, natoms=32, placement="lattice", lattice=(4, 4, 2),
                     well_z=4.0, well_sigma=0.7, lmax=2, proj_sigma=0.6, rc=2.5, dl=(2.0, -0.8, 0.3),
                     kfrac=(0.25, 0.0, 0.0), ecut=30.0),
    "large": _cubic("large", 4, 30.0, 96, nst=1024, natoms=128, placement="lattice", lattice=(8, 4, 4),
                    well_z=4.0, well_sigma=0.7, lmax=1, proj_sigma=0.6, rc=3.0, dl=(2.0, -0.8)),
    "tddft": _cubic("tddft", 5, 25.0, 64, nst=512, natoms=64, placement="lattice", lattice=(4, 4, 4),
                    well_z=4.0, well_sigma=0.7, lmax=1, proj_sigma=0.6, rc=2.5, dl=(2.0, -0.8),
                    dt=0.02, nsteps=20),
}
CONFIG_ORDER = ("tiny", "small", "medium", "large", "tddft")


def test_config(cid: int, n: Sequence[int], length: Sequence[float], nst: int, natoms: int, **kw) -> Config:
    """A free-form config for parity / edge-case tests (cid >= 100 keeps seeds apart)."""
    assert cid >= 100
    kw.setdefault("placement", "uniform")
    return Config(name=f"test{cid}", cid=cid, n=tuple(int(x) for x in n),
                  length=tuple(float(x) for x in length), nst=nst, natoms=natoms, **kw)


# ----------------------------------------------------------------------------------------------
# atoms
# ----------------------------------------------------------------------------------------------
def atom_positions(cfg: Config) -> np.ndarray:
    """(natoms, 3) Cartesian positions in [0, L).  tag 0 of the config's seed."""
    rng = np.random.default_rng([BASE_SEED + cfg.cid, 0])
    L = np.asarray(cfg.length)
    if cfg.natoms == 0:
        return np.zeros((0, 3))
    if cfg.placement == "uniform":
        return rng.uniform(0.0, 1.0, size=(cfg.natoms, 3)) * L
    if cfg.placement == "lattice":
        nx, ny, nz = cfg.lattice
        assert nx * ny * nz == cfg.natoms
        a, b, c = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
        sites = np.stack([(a.ravel() + 0.5) / nx, (b.ravel() + 0.5) / ny, (c.ravel() + 0.5) / nz], axis=1) * L
        jit = rng.uniform(-cfg.jitter, cfg.jitter, size=(cfg.natoms, 3))
        return np.mod(sites + jit, L)
    raise ValueError(cfg.placement)


# ----------------------------------------------------------------------------------------------
# local potential (an input array; reading R12)
# ----------------------------------------------------------------------------------------------
def _min_image_axis(n: int, length: float, r0: float) -> np.ndarray:
    """d[i] = minimum-image (i*h - r0) along one periodic axis."""
    h = length / n
    d = np.arange(n) * h - r0
    return d - length * np.round(d / length)


def local_potential(cfg: Config, pos: Optional[np.ndarray] = None) -> np.ndarray:
    """V(r) on the grid, float64, shape n.  Sum of Gaussian wells at the atoms (+ noise for config 1)."""
    if pos is None:
        pos = atom_positions(cfg)
    n = cfg.n
    v = np.zeros(n, dtype=np.float64)
    if len(pos):
        s2 = 2.0 * cfg.well_sigma ** 2
        # the Gaussian of the min-image distance separates per axis in an orthorhombic cell
        g = [np.stack([np.exp(-_min_image_axis(n[a], cfg.length[a], p[a]) ** 2 / s2) for p in pos]) for a in range(3)]
        v -= cfg.well_z * np.einsum("ai,aj,ak->ijk", g[0], g[1], g[2], optimize=True)
    if cfg.noise > 0.0:
        rng = np.random.default_rng([BASE_SEED + cfg.cid, 1])
        v += rng.uniform(-cfg.noise, cfg.noise, size=n)
    return np.ascontiguousarray(v)


# ----------------------------------------------------------------------------------------------
# projectors (input tables; readings R4, R5, R11)
# ----------------------------------------------------------------------------------------------
def real_ylm(l: int, m: int, d: np.ndarray) -> np.ndarray:
    """Real spherical harmonics, l <= 2, orthonormal constants of R11.  d: (P,3).  Value 0 at d = 0 for l > 0."""
    x, y, z = d[:, 0], d[:, 1], d[:, 2]
    r2 = x * x + y * y + z * z
    if l == 0:
        return np.full(len(d), 0.5 * math.sqrt(1.0 / math.pi))
    r = np.sqrt(r2)
    ok = r2 > 0.0
    rs = np.where(ok, r, 1.0)
    r2s = np.where(ok, r2, 1.0)
    if l == 1:
        c = math.sqrt(3.0 / (4.0 * math.pi))
        num = {-1: y, 0: z, 1: x}[m]
        return np.where(ok, c * num / rs, 0.0)
    if l == 2:
        c15 = math.sqrt(15.0 / math.pi)
        c5 = math.sqrt(5.0 / math.pi)
        val = {
            -2: 0.5 * c15 * x * y / r2s,
            -1: 0.5 * c15 * y * z / r2s,
            0: 0.25 * c5 * (3.0 * z * z - r2) / r2s,
            1: 0.5 * c15 * x * z / r2s,
            2: 0.25 * c15 * (x * x - y * y) / r2s,
        }[m]
        return np.where(ok, val, 0.0)
    raise ValueError("l <= 2 only")


@dataclasses.dataclass
class Projectors:
    natoms: int
    sph_off: np.ndarray    # int64 [natoms+1]
    sph_idx: np.ndarray    # int32 [sum P]
    sph_disp: np.ndarray   # float64 [sum P, 3]
    chan_off: np.ndarray   # int32 [natoms+1]
    beta: np.ndarray       # float64, per atom [C_I][P_I] concatenated
    dcoef: np.ndarray      # float64 [sum C]

    def beta_of(self, atom: int) -> np.ndarray:
        """[C_I, P_I] view of one atom's projector values."""
        c0, c1 = int(self.chan_off[atom]), int(self.chan_off[atom + 1])
        p0, p1 = int(self.sph_off[atom]), int(self.sph_off[atom + 1])
        start = sum(int(self.chan_off[a + 1] - self.chan_off[a]) * int(self.sph_off[a + 1] - self.sph_off[a])
                    for a in range(atom))
        return self.beta[start:start + (c1 - c0) * (p1 - p0)].reshape(c1 - c0, p1 - p0)


def sphere_points(cfg: Config, center: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """Flat indices (int32) and min-image displacements of the grid points with |r - center| < rc (strict).

    rc < L/2 on every axis (R5), so each grid point appears at most once.
    """
    n, h = cfg.n, cfg.spacing
    assert all(cfg.rc < 0.5 * cfg.length[a] for a in range(3)), "sphere must not overlap its own image"
    ax_i, ax_d = [], []
    for a in range(3):
        lo = int(math.ceil((center[a] - cfg.rc) / h[a]))
        hi = int(math.floor((center[a] + cfg.rc) / h[a]))
        ii = np.arange(lo, hi + 1)
        ax_i.append(np.mod(ii, n[a]))
        ax_d.append(ii * h[a] - center[a])
    I, J, K = np.meshgrid(ax_i[0], ax_i[1], ax_i[2], indexing="ij")
    DX, DY, DZ = np.meshgrid(ax_d[0], ax_d[1], ax_d[2], indexing="ij")
    r2 = DX * DX + DY * DY + DZ * DZ
    keep = r2 < cfg.rc * cfg.rc
    idx = ((I * n[1] + J) * n[2] + K)[keep].astype(np.int32)
    disp = np.stack([DX[keep], DY[keep], DZ[keep]], axis=1)
    return idx, np.ascontiguousarray(disp)


def projectors(cfg: Config, pos: Optional[np.ndarray] = None) -> Projectors:
    """KB projector tables: beta_{lm}(d) = exp(-|d|^2 / (2 sigma^2)) * Y_lm(d/|d|), channels l asc, m asc."""
    if pos is None:
        pos = atom_positions(cfg)
    sph_off, chan_off = [0], [0]
    idx_all, disp_all, beta_all, d_all = [], [], [], []
    for p in pos:
        idx, disp = sphere_points(cfg, p)
        rad = np.exp(-np.sum(disp * disp, axis=1) / (2.0 * cfg.proj_sigma ** 2))
        rows, dco = [], []
        for l in range(cfg.lmax + 1):
            for m in range(-l, l + 1):
                rows.append(rad * real_ylm(l, m, disp))
                dco.append(cfg.dl[l])
        idx_all.append(idx)
        disp_all.append(disp)
        beta_all.append(np.stack(rows).ravel())
        d_all.append(np.asarray(dco))
        sph_off.append(sph_off[-1] + len(idx))
        chan_off.append(chan_off[-1] + len(rows))
    cat = lambda xs, dt, shape: (np.ascontiguousarray(np.concatenate(xs)).astype(dt) if xs else np.zeros(shape, dt))
    return Projectors(
        natoms=len(pos),
        sph_off=np.asarray(sph_off, dtype=np.int64),
        sph_idx=cat(idx_all, np.int32, (0,)),
        sph_disp=cat(disp_all, np.float64, (0, 3)),
        chan_off=np.asarray(chan_off, dtype=np.int32),
        beta=cat(beta_all, np.float64, (0,)),
        dcoef=cat(d_all, np.float64, (0,)),
    )


# ----------------------------------------------------------------------------------------------
# states
# ----------------------------------------------------------------------------------------------
def state(cfg: Config, s: int) -> np.ndarray:
    """State s of the config: complex128, shape n, i.i.d. complex Gaussian, dV*sum|psi|^2 = 1 (R14)."""
    rng = np.random.default_rng([BASE_SEED + cfg.cid, 2, int(s)])
    npts = cfg.npts
    re = rng.standard_normal(npts)
    im = rng.standard_normal(npts)
    psi = re + 1j * im
    psi /= math.sqrt(cfg.dv * float(np.sum(re * re + im * im)))
    return psi.reshape(cfg.n)


def states(cfg: Config, s0: int = 0, s1: Optional[int] = None, out: Optional[np.ndarray] = None) -> np.ndarray:
    """Block of states [s0, s1) as one contiguous (s1-s0, n0, n1, n2) complex128 array."""
    if s1 is None:
        s1 = cfg.nst
    if out is None:
        out = np.empty((s1 - s0,) + tuple(cfg.n), dtype=np.complex128)
    for s in range(s0, s1):
        out[s - s0] = state(cfg, s)
    return out


@dataclasses.dataclass
class Workload:
    cfg: Config
    pos: np.ndarray
    v: np.ndarray
    proj: Projectors


def make(cfg: Config) -> Workload:
    """Everything except psi (which is generated per state / per chunk on demand)."""
    pos = atom_positions(cfg)
    return Workload(cfg=cfg, pos=pos, v=local_potential(cfg, pos), proj=projectors(cfg, pos))
