"""ctypes front end of the CPU oracle (oracle/ref_tdh.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this module.
It does not import the CUDA package's binding; arguments are plain numpy arrays on the host.

Functions mirror the C exports one to one (see the header comment of ref_tdh.c for the passages they follow):
    dft3d, kinetic, local, nonlocal_, apply_hamiltonian, propagate, num_threads
``backend``: 0 = direct O(N^2)-per-pencil DFT (the definition), 1 = naive recursive radix-2/3 FFT.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build

DIRECT, NAIVE_FFT = 0, 1

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        for name in ("ref_dft3d", "ref_kinetic", "ref_local", "ref_nonlocal", "ref_apply_hamiltonian",
                     "ref_propagate", "ref_taylor_pair", "ref_etrs_step", "ref_density", "ref_hartree", "ref_overlap", "ref_sd_step", "ref_gradient", "ref_forces", "ref_num_threads"):
            getattr(_lib, name).restype = C.c_int
    return _lib


def _i3(x):
    return (C.c_int * 3)(*[int(v) for v in x])


def _d3(x):
    return (C.c_double * 3)(*[float(v) for v in x])


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


class _Proj:
    """Marshalled projector tables (keeps the contiguous arrays alive)."""

    def __init__(self, proj):
        if proj is None or proj.natoms == 0:
            self.natoms = 0
            self.args = (C.c_int(0), None, None, None, None, None, None)
            return
        self.natoms = int(proj.natoms)
        self.sph_off = np.ascontiguousarray(proj.sph_off, dtype=np.int64)
        self.sph_idx = np.ascontiguousarray(proj.sph_idx, dtype=np.int32)
        self.sph_disp = None if proj.sph_disp is None else np.ascontiguousarray(proj.sph_disp, dtype=np.float64)
        self.chan_off = np.ascontiguousarray(proj.chan_off, dtype=np.int32)
        self.beta = np.ascontiguousarray(proj.beta, dtype=np.float64)
        self.dcoef = np.ascontiguousarray(proj.dcoef, dtype=np.float64)
        self.args = (C.c_int(self.natoms), _ptr(self.sph_off), _ptr(self.sph_idx), _ptr(self.sph_disp),
                     _ptr(self.chan_off), _ptr(self.beta), _ptr(self.dcoef))


def num_threads() -> int:
    return int(lib().ref_num_threads())


def dft3d(a: np.ndarray, sign: int, backend: int = DIRECT) -> np.ndarray:
    """3-D DFT of a block (nst, n0, n1, n2) (or one state (n0, n1, n2)); sign -1 forward, +1 inverse (1/N_p)."""
    a = _c128(a).copy()
    n = a.shape[-3:]
    nst = 1 if a.ndim == 3 else a.shape[0]
    _check(lib().ref_dft3d(_i3(n), C.c_int(nst), _ptr(a), C.c_int(sign), C.c_int(backend)), "dft3d")
    return a


def kinetic(n, length, kpt, ecut, psi, backend: int = DIRECT) -> np.ndarray:
    psi = _c128(psi)
    out = np.empty_like(psi)
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    _check(lib().ref_kinetic(_i3(n), _d3(length), _d3(kpt), C.c_double(ecut), C.c_int(nst), _ptr(psi), _ptr(out),
                             C.c_int(backend)), "kinetic")
    return out


def local(n, v, psi) -> np.ndarray:
    psi = _c128(psi)
    out = np.empty_like(psi)
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
    _check(lib().ref_local(_i3(n), _ptr(v), C.c_int(nst), _ptr(psi), _ptr(out)), "local")
    return out


def nonlocal_(n, length, kpt, proj, psi) -> np.ndarray:
    psi = _c128(psi)
    out = np.empty_like(psi)
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    p = _Proj(proj)
    _check(lib().ref_nonlocal(_i3(n), _d3(length), _d3(kpt), *p.args, C.c_int(nst), _ptr(psi), _ptr(out)), "nonlocal")
    return out


def apply_hamiltonian(n, length, kpt, ecut, v, proj, psi, backend: int = NAIVE_FFT) -> np.ndarray:
    """H psi for a block (nst, n0, n1, n2) or a single state (n0, n1, n2).  Returns a new array."""
    psi = _c128(psi)
    out = np.empty_like(psi)
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
    p = _Proj(proj)
    _check(lib().ref_apply_hamiltonian(_i3(n), _d3(length), _d3(kpt), C.c_double(ecut), _ptr(v), *p.args,
                                       C.c_int(nst), _ptr(psi), _ptr(out), C.c_int(backend)), "apply_hamiltonian")
    return out


def propagate(n, length, kpt, ecut, v, proj, psi, dt: float, nsteps: int, order: int = 4,
              backend: int = NAIVE_FFT) -> np.ndarray:
    """nsteps Taylor-`order` steps of exp(-i dt H).  Returns a new array (the input is not modified)."""
    psi = _c128(psi).copy()
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
    p = _Proj(proj)
    _check(lib().ref_propagate(_i3(n), _d3(length), _d3(kpt), C.c_double(ecut), _ptr(v), *p.args, C.c_int(nst),
                               _ptr(psi), C.c_double(dt), C.c_int(nsteps), C.c_int(order), C.c_int(backend)),
           "propagate")
    return psi


def taylor_pair(n, length, kpt, ecut, v, proj, psi, dt: float, order: int = 4, backend: int = NAIVE_FFT):
    """(exp(-i dt/2 H) psi, exp(-i dt H) psi) from one chain of powers H^k psi.  Returns new arrays."""
    psi = _c128(psi)
    half, full = np.empty_like(psi), np.empty_like(psi)
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
    p = _Proj(proj)
    _check(lib().ref_taylor_pair(_i3(n), _d3(length), _d3(kpt), C.c_double(ecut), _ptr(v), *p.args, C.c_int(nst), _ptr(psi),
                                 _ptr(half), _ptr(full), C.c_double(dt), C.c_int(order), C.c_int(backend)), "taylor_pair")
    return half, full


def etrs_step(n, length, kpt, ecut, v, v_next, proj, psi, dt: float, backend: int = NAIVE_FFT):
    """One ETRS step (Eq. 6-7) with V(t+dt) = v_next supplied.  Returns (psi(t+dt), approx = exp(-i dt H(t)) psi(t))."""
    out = _c128(psi).copy()
    approx = np.empty_like(out)
    nst = 1 if out.ndim == 3 else out.shape[0]
    v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
    v_next = None if v_next is None else np.ascontiguousarray(v_next, dtype=np.float64)
    p = _Proj(proj)
    _check(lib().ref_etrs_step(_i3(n), _d3(length), _d3(kpt), C.c_double(ecut), _ptr(v), _ptr(v_next), *p.args, C.c_int(nst),
                               _ptr(out), _ptr(approx), C.c_double(dt), C.c_int(backend)), "etrs_step")
    return out, approx


def density(n, psi, occ=None, accumulate_into=None) -> np.ndarray:
    """n(r) = sum_s occ[s] |psi_s(r)|^2 (Eq. 1); occ None: all 1.  accumulate_into: float64 array (n) that is added to."""
    psi = _c128(psi)
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    occ = None if occ is None else np.ascontiguousarray(occ, dtype=np.float64)
    out = np.zeros(tuple(n), dtype=np.float64) if accumulate_into is None else accumulate_into
    assert out.flags["C_CONTIGUOUS"] and out.dtype == np.float64
    _check(lib().ref_density(_i3(n), C.c_int(nst), _ptr(psi), _ptr(occ), _ptr(out),
                             C.c_int(0 if accumulate_into is None else 1)), "density")
    return out


def hartree(n, length, dens, backend: int = NAIVE_FFT) -> np.ndarray:
    """Periodic Hartree potential: v_hat(G) = 4 pi n_hat(G) / |G|^2, G = 0 dropped."""
    dens = np.ascontiguousarray(dens, dtype=np.float64)
    out = np.empty_like(dens)
    _check(lib().ref_hartree(_i3(n), _d3(length), _ptr(dens), _ptr(out), C.c_int(backend)), "hartree")
    return out


def overlap(n, dv: float, a, b) -> np.ndarray:
    """S[i][j] = dV sum_p conj(a_i[p]) b_j[p] for two state blocks (na, n0, n1, n2), (nb, n0, n1, n2)."""
    a, b = _c128(a), _c128(b)
    na, nb = a.shape[0], b.shape[0]
    s = np.empty((na, nb), dtype=np.complex128)
    _check(lib().ref_overlap(_i3(n), C.c_double(dv), C.c_int(na), _ptr(a), C.c_int(nb), _ptr(b), _ptr(s)), "overlap")
    return s


def rotate(psi, m) -> np.ndarray:
    """Rotation in the space of states: out_j = sum_i psi_i m[i][j]; psi (n_in, n0, n1, n2), m (n_in, n_out)."""
    psi = _c128(psi)
    m = _c128(m)
    out = np.zeros((m.shape[1],) + psi.shape[1:], dtype=np.complex128)
    for j in range(m.shape[1]):                 # literal loops over the two state indices
        for i in range(m.shape[0]):
            out[j] += psi[i] * m[i, j]
    return out


def orthonormalize(n, dv: float, psi) -> np.ndarray:
    """Cholesky orthonormalisation ("orthogonalization"): S = dV psi^H psi = L L^H (library Cholesky as one
    step), psi' = psi L^{-H}, so that dV psi'^H psi' = 1 and psi'_j only mixes psi_0..psi_j (the Gram-Schmidt order)."""
    s = overlap(n, dv, psi, psi)
    l = np.linalg.cholesky(0.5 * (s + s.conj().T))
    w = np.linalg.inv(l)                         # lower triangular L^{-1}
    return rotate(psi, w.conj().T)


def sd_step(n, length, kpt, ecut, v, proj, psi, lam: float, backend: int = NAIVE_FFT):
    """One Teter-preconditioned steepest-descent update of every state (fixed step lam).  Returns (new psi, eps before)."""
    out = _c128(psi).copy()
    nst = 1 if out.ndim == 3 else out.shape[0]
    v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
    eig = np.empty(nst, dtype=np.float64)
    p = _Proj(proj)
    _check(lib().ref_sd_step(_i3(n), _d3(length), _d3(kpt), C.c_double(ecut), _ptr(v), *p.args, C.c_int(nst), _ptr(out),
                             C.c_double(lam), _ptr(eig), C.c_int(backend)), "sd_step")
    return out, eig


def subspace_diag(n, dv: float, psi, hpsi):
    """Subspace diagonalisation of an orthonormal block: M = dV psi^H (H psi), M = V diag(w) V^H (library
    Hermitian eigensolver as one step, w ascending), psi' = psi V.  Returns (w, psi', V); V's columns are unique only up
    to a phase (and within degenerate eigenspaces)."""
    m = overlap(n, dv, psi, hpsi)
    w, v = np.linalg.eigh(0.5 * (m + m.conj().T))
    return w, rotate(psi, v), v


def gradient(n, length, kpt, axis: int, psi, backend: int = NAIVE_FFT) -> np.ndarray:
    """d_axis psi = DFT^-1(i (G_a + k_a) DFT psi) for a block or a single state."""
    psi = _c128(psi)
    out = np.empty_like(psi)
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    _check(lib().ref_gradient(_i3(n), _d3(length), _d3(kpt), C.c_int(axis), C.c_int(nst), _ptr(psi), _ptr(out),
                              C.c_int(backend)), "gradient")
    return out


def forces(n, length, kpt, proj, psi, occ=None, vloc_atoms=None, backend: int = NAIVE_FFT) -> np.ndarray:
    """Eq. 11: F[I][a] = sum_s f_s (<d_a psi_s|v_I|psi_s> + c.c.); vloc_atoms: (natoms, n0, n1, n2) float64 or None."""
    psi = _c128(psi)
    nst = 1 if psi.ndim == 3 else psi.shape[0]
    p = _Proj(proj)
    occ = None if occ is None else np.ascontiguousarray(occ, dtype=np.float64)
    vl = None if vloc_atoms is None else np.ascontiguousarray(vloc_atoms, dtype=np.float64)
    out = np.zeros((p.natoms, 3), dtype=np.float64)
    _check(lib().ref_forces(_i3(n), _d3(length), _d3(kpt), *p.args, _ptr(vl), C.c_int(nst), _ptr(psi), _ptr(occ), _ptr(out),
                            C.c_int(backend)), "forces")
    return out


def apply_workload(wl, psi, backend: int = NAIVE_FFT) -> np.ndarray:
    """Convenience: H psi with a workloads.Workload."""
    c = wl.cfg
    return apply_hamiltonian(c.n, c.length, c.kpt, c.ecut_abi, wl.v, wl.proj, psi, backend)


def propagate_workload(wl, psi, dt=None, nsteps=None, backend: int = NAIVE_FFT) -> np.ndarray:
    c = wl.cfg
    return propagate(c.n, c.length, c.kpt, c.ecut_abi, wl.v, wl.proj, psi, c.dt if dt is None else dt,
                     c.nsteps if nsteps is None else nsteps, 4, backend)
