"""Thin ctypes binding of libtdh.so (include/tdh.h).  Argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch supplies device memory and the stream.
There is no CPU fallback: importing this module without the built library, or creating a grid without a CUDA
device, raises.

    g = Grid(n, length, kpt, ecut, max_states)           # tdh_create_grid on torch's current stream
    g.set_potential(v)                                    # torch float64 CUDA tensor (n0, n1, n2)
    g.set_projectors(proj)                                # workloads.Projectors (host numpy tables)
    hpsi = g.apply_hamiltonian(psi)                       # torch complex128 CUDA tensor (nst, n0, n1, n2)
    g.propagate(psi, dt, nsteps)                          # in place
    g.apply_hamiltonian_host(psi_host, out_host)          # numpy / pinned torch CPU tensors
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtdh.so")

#: every symbol include/tdh.h declares
SYMBOLS = (
    "tdh_create_grid", "tdh_destroy_grid", "tdh_set_potential", "tdh_set_projectors", "tdh_apply_hamiltonian",
    "tdh_propagate", "tdh_taylor_pair", "tdh_etrs_step", "tdh_density", "tdh_hartree", "tdh_overlap", "tdh_rotate", "tdh_orthonormalize", "tdh_subspace_diag", "tdh_sd_step", "tdh_gradient", "tdh_forces", "tdh_apply_hamiltonian_host", "tdh_propagate_host", "tdh_fft3d", "tdh_last_launch_count",
    "tdh_create_slab_grid", "tdh_slab_buffers", "tdh_slab_set_peers", "tdh_slab_apply_phase", "tdh_slab_fft_phase", "tdh_work_layout",
    "tdh_ipc_export", "tdh_ipc_import", "tdh_ipc_close", "tdh_last_jacobi_sweeps",
    "tdh_set_profiling", "tdh_last_kernel_seconds", "tdh_kernel_name", "tdh_set_chunk_states", "tdh_reserve", "tdh_last_error",
    "tdh_overlap_noalloc",
)
NKERNELS = 6

TDH_OK, TDH_EINVAL, TDH_EUNSUPPORTED, TDH_ENOMEM, TDH_ECUDA, TDH_EINDEX = 0, -1, -2, -3, -4, -5


class TdhError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libtdh error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Load libtdh.so (fails loudly if it has not been built: python -m paper_2106_03872_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing; build it with `python -m paper_2106_03872_b200.build` "
                          "(there is no CPU fallback)")
    l = C.CDLL(LIB_PATH)
    vp, i, d = C.c_void_p, C.c_int, C.c_double
    l.tdh_create_grid.argtypes = [C.POINTER(i), C.POINTER(d), C.POINTER(d), d, i, vp, C.POINTER(vp)]
    l.tdh_destroy_grid.argtypes = [vp]
    l.tdh_set_potential.argtypes = [vp, vp]
    l.tdh_set_projectors.argtypes = [vp, i, vp, vp, vp, vp, vp, vp]
    l.tdh_apply_hamiltonian.argtypes = [vp, i, vp, vp]
    l.tdh_propagate.argtypes = [vp, i, vp, d, i, i]
    l.tdh_taylor_pair.argtypes = [vp, i, vp, vp, d, i]
    l.tdh_etrs_step.argtypes = [vp, i, vp, vp, d, vp]
    l.tdh_density.argtypes = [vp, i, vp, vp, vp, i]
    l.tdh_hartree.argtypes = [vp, vp, vp]
    l.tdh_overlap.argtypes = [vp, i, vp, i, vp, vp]
    l.tdh_rotate.argtypes = [vp, i, vp, i, vp, vp]
    l.tdh_orthonormalize.argtypes = [vp, i, vp, vp]
    l.tdh_sd_step.argtypes = [vp, i, vp, vp, d, vp]
    l.tdh_subspace_diag.argtypes = [vp, i, vp, vp, vp, vp]
    l.tdh_gradient.argtypes = [vp, i, vp, i, vp]
    l.tdh_forces.argtypes = [vp, i, vp, vp, vp, vp]
    l.tdh_apply_hamiltonian_host.argtypes = [vp, i, vp, vp]
    l.tdh_propagate_host.argtypes = [vp, i, vp, d, i, i]
    l.tdh_fft3d.argtypes = [vp, i, vp, i]
    l.tdh_last_launch_count.argtypes = [vp]
    l.tdh_create_slab_grid.argtypes = [C.POINTER(i), C.POINTER(d), C.POINTER(d), d, i, i, i, vp, C.POINTER(vp)]
    l.tdh_slab_buffers.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    l.tdh_slab_set_peers.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    l.tdh_slab_apply_phase.argtypes = [vp, i, i, vp, vp]
    l.tdh_slab_fft_phase.argtypes = [vp, i, i, i, vp]
    l.tdh_work_layout.argtypes = [vp, C.POINTER(i), C.POINTER(i)]
    l.tdh_ipc_export.argtypes = [vp, C.c_char_p]
    l.tdh_ipc_import.argtypes = [C.c_char_p, C.POINTER(vp)]
    l.tdh_ipc_close.argtypes = [vp]
    l.tdh_last_jacobi_sweeps.argtypes = [vp]
    l.tdh_set_profiling.argtypes = [vp, i]
    l.tdh_last_kernel_seconds.argtypes = [vp, C.POINTER(d)]
    l.tdh_kernel_name.argtypes = [i]
    l.tdh_kernel_name.restype = C.c_char_p
    l.tdh_set_chunk_states.argtypes = [vp, i]
    l.tdh_overlap_noalloc.argtypes = [C.c_size_t, d, i, vp, i, vp, vp, vp]
    l.tdh_last_error.argtypes = []
    l.tdh_last_error.restype = C.c_char_p
    for s in SYMBOLS:
        if s not in ("tdh_kernel_name", "tdh_last_error"):
            getattr(l, s).restype = i
    _lib = l
    return l


def _check(rc: int):
    if rc != 0:
        raise TdhError(rc, lib().tdh_last_error().decode(errors="replace"))


NOALLOC_MAX_STATES = 256          # TDH_NOALLOC_MAX_STATES
NOALLOC_SCRATCH_BYTES = 8 << 20   # TDH_NOALLOC_SCRATCH_BYTES


def overlap_noalloc(a, b=None, dv: float = 1.0, out=None, stream: Optional[int] = None):
    """S[i][j] = dv sum_p conj(a_i[p]) b_j[p] through tdh_overlap_noalloc: no handle, and nothing is allocated inside the
    call (its scratch is a fixed 8 MiB array inside libtdh.so), for programs whose own pool owns the device memory or
    that cannot take an allocation's synchronisation in their time loop.  a, b: complex128 device tensors (states, ...)
    with the same number of points per state, at most 256 states each; pass `out` (na, nb) to keep this wrapper from
    allocating the result as well.  Every call shares the scratch array: keep calls on one stream.  Make the first call
    on a device at start-up (it looks up the array's address there)."""
    import torch
    if b is None:
        b = a
    for t in (a, b):
        assert t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous() and t.dim() >= 2
    na, nb = int(a.shape[0]), int(b.shape[0])
    npts = a[0].numel()
    assert b[0].numel() == npts, "a and b must have the same number of grid points per state"
    if out is None:
        out = torch.empty((na, nb), dtype=torch.complex128, device=a.device)
    assert out.is_cuda and out.dtype == torch.complex128 and out.is_contiguous() and out.numel() == na * nb
    if stream is None:
        stream = torch.cuda.current_stream(a.device).cuda_stream
    with torch.cuda.device(a.device):
        _check(lib().tdh_overlap_noalloc(npts, float(dv), na, C.c_void_p(a.data_ptr()), nb, C.c_void_p(b.data_ptr()),
                                         C.c_void_p(out.data_ptr()), C.c_void_p(stream)))
    return out


def _host_ptr(a) -> int:
    """Address of a contiguous host buffer: numpy array or CPU torch tensor."""
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert not a.is_cuda and a.is_contiguous()
    return a.data_ptr()


class Grid:
    """Owns one tdh_grid handle.  All tensors passed in must live on the device that was current at creation."""

    def __init__(self, n: Sequence[int], length: Sequence[float], kpt: Sequence[float] = (0.0, 0.0, 0.0),
                 ecut: float = -1.0, max_states: int = 1, stream: Optional[int] = None,
                 slab: Optional[Sequence[int]] = None):
        """slab = (rank, world): the handle of one rank of a slab decomposition (tdh_create_slab_grid); self.n is then
        the shape of the rank's real-space planes and self.n_full the whole grid."""
        import torch
        l = lib()
        if stream is None:
            if not torch.cuda.is_available():
                raise TdhError(TDH_ECUDA, "no CUDA device available (there is no CPU fallback)")
            stream = torch.cuda.current_stream().cuda_stream
        self.n_full = tuple(int(x) for x in n)
        self.slab = None if slab is None else (int(slab[0]), int(slab[1]))
        self.n = self.n_full if slab is None else (self.n_full[0] // self.slab[1],) + self.n_full[1:]
        self.npts = self.n[0] * self.n[1] * self.n[2]
        self.max_states = int(max_states)
        self.natoms = 0
        self._h = C.c_void_p()
        a3 = ((C.c_int * 3)(*self.n_full), (C.c_double * 3)(*[float(x) for x in length]),
              (C.c_double * 3)(*[float(x) for x in kpt]), float(ecut), int(max_states))
        if slab is None:
            _check(l.tdh_create_grid(*a3, C.c_void_p(stream), C.byref(self._h)))
        else:
            _check(l.tdh_create_slab_grid(*a3, self.slab[0], self.slab[1], C.c_void_p(stream), C.byref(self._h)))

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().tdh_destroy_grid(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- set-up
    def set_potential(self, v):
        if v is None:
            _check(lib().tdh_set_potential(self._h, None))
            return
        import torch
        assert v.is_cuda and v.dtype == torch.float64 and v.is_contiguous() and v.numel() == self.npts
        _check(lib().tdh_set_potential(self._h, C.c_void_p(v.data_ptr())))

    def set_projectors(self, proj):
        """proj: workloads.Projectors-like object with host numpy tables, or None to clear."""
        if proj is None or proj.natoms == 0:
            _check(lib().tdh_set_projectors(self._h, 0, None, None, None, None, None, None))
            self.natoms = 0
            return
        sph_off = np.ascontiguousarray(proj.sph_off, dtype=np.int64)
        sph_idx = np.ascontiguousarray(proj.sph_idx, dtype=np.int32)
        sph_disp = None if proj.sph_disp is None else np.ascontiguousarray(proj.sph_disp, dtype=np.float64)
        chan_off = np.ascontiguousarray(proj.chan_off, dtype=np.int32)
        beta = np.ascontiguousarray(proj.beta, dtype=np.float64)
        dcoef = np.ascontiguousarray(proj.dcoef, dtype=np.float64)
        p = lambda a: None if a is None else C.c_void_p(a.ctypes.data)
        _check(lib().tdh_set_projectors(self._h, int(proj.natoms), p(sph_off), p(sph_idx), p(sph_disp), p(chan_off),
                                        p(beta), p(dcoef)))
        # the handle's atom count sizes the result of tdh_forces; a table without any channel clears the projectors
        self.natoms = int(proj.natoms) if int(chan_off[-1]) > 0 else 0

    # -- device entry points
    def _block(self, psi):
        import torch
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous()
        assert psi.numel() % self.npts == 0
        return psi.numel() // self.npts

    def apply_hamiltonian(self, psi, out=None):
        import torch
        nst = self._block(psi)
        if out is None:
            out = torch.empty_like(psi)
        assert self._block(out) == nst
        _check(lib().tdh_apply_hamiltonian(self._h, nst, C.c_void_p(psi.data_ptr()), C.c_void_p(out.data_ptr())))
        return out

    def propagate(self, psi, dt: float, nsteps: int, order: int = 4):
        nst = self._block(psi)
        _check(lib().tdh_propagate(self._h, nst, C.c_void_p(psi.data_ptr()), float(dt), int(nsteps), int(order)))
        return psi

    def taylor_pair(self, psi, dt: float, full=None, order: int = 4):
        """psi <- exp(-i dt/2 H) psi in place; returns full = exp(-i dt H) psi (both Taylor order 4, one chain of powers)."""
        import torch
        nst = self._block(psi)
        if full is None:
            full = torch.empty_like(psi)
        assert self._block(full) == nst
        _check(lib().tdh_taylor_pair(self._h, nst, C.c_void_p(psi.data_ptr()), C.c_void_p(full.data_ptr()), float(dt), int(order)))
        return full

    def etrs_step(self, psi, dt: float, v_next, approx=None):
        """One ETRS step in place with V(t+dt) = v_next (device float64 tensor or None); returns approx = exp(-i dt H(t)) psi."""
        import torch
        nst = self._block(psi)
        if approx is None:
            approx = torch.empty_like(psi)
        assert self._block(approx) == nst
        vp_ = None
        if v_next is not None:
            assert v_next.is_cuda and v_next.dtype == torch.float64 and v_next.is_contiguous() and v_next.numel() == self.npts
            vp_ = C.c_void_p(v_next.data_ptr())
        _check(lib().tdh_etrs_step(self._h, nst, C.c_void_p(psi.data_ptr()), C.c_void_p(approx.data_ptr()), float(dt), vp_))
        return approx

    def density(self, psi, occ=None, out=None, accumulate: bool = False):
        """n(r) = sum_s occ[s] |psi_s(r)|^2 (Eq. 1) of the block on this device; occ: host numpy array or None (all 1)."""
        import torch
        nst = self._block(psi)
        if out is None:
            assert not accumulate
            out = torch.empty(self.n, dtype=torch.float64, device=psi.device)
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.npts
        occ_arr = None if occ is None else np.ascontiguousarray(occ, dtype=np.float64)
        assert occ_arr is None or occ_arr.size == nst
        _check(lib().tdh_density(self._h, nst, C.c_void_p(psi.data_ptr()),
                                 None if occ_arr is None else C.c_void_p(occ_arr.ctypes.data),
                                 C.c_void_p(out.data_ptr()), 1 if accumulate else 0))
        return out

    def hartree(self, dens, out=None):
        """Periodic Hartree potential of a density (device float64 tensor of the grid's shape)."""
        import torch
        assert dens.is_cuda and dens.dtype == torch.float64 and dens.is_contiguous() and dens.numel() == self.npts
        if out is None:
            out = torch.empty_like(dens)
        _check(lib().tdh_hartree(self._h, C.c_void_p(dens.data_ptr()), C.c_void_p(out.data_ptr())))
        return out

    def overlap(self, a, b=None, out=None):
        """S[i][j] = dV sum_p conj(a_i[p]) b_j[p] (b = a if omitted); returns a (na, nb) complex128 device tensor."""
        import torch
        if b is None:
            b = a
        na, nb = self._block(a), self._block(b)
        if out is None:
            out = torch.empty((na, nb), dtype=torch.complex128, device=a.device)
        assert out.is_cuda and out.dtype == torch.complex128 and out.is_contiguous() and out.numel() == na * nb
        _check(lib().tdh_overlap(self._h, na, C.c_void_p(a.data_ptr()), nb, C.c_void_p(b.data_ptr()),
                                 C.c_void_p(out.data_ptr())))
        return out

    def rotate(self, psi, m, out=None):
        """out_j = sum_i psi_i m[i][j]; m: (n_in, n_out) complex128 device tensor."""
        import torch
        n_in = self._block(psi)
        assert m.is_cuda and m.dtype == torch.complex128 and m.is_contiguous() and m.dim() == 2 and m.shape[0] == n_in
        n_out = int(m.shape[1])
        if out is None:
            out = torch.empty((n_out,) + self.n, dtype=torch.complex128, device=psi.device)
        assert self._block(out) == n_out
        _check(lib().tdh_rotate(self._h, n_in, C.c_void_p(psi.data_ptr()), n_out, C.c_void_p(m.data_ptr()),
                                C.c_void_p(out.data_ptr())))
        return out

    def orthonormalize(self, psi, out=None):
        """Cholesky orthonormalisation of a block (out-of-place)."""
        import torch
        nst = self._block(psi)
        if out is None:
            out = torch.empty_like(psi)
        _check(lib().tdh_orthonormalize(self._h, nst, C.c_void_p(psi.data_ptr()), C.c_void_p(out.data_ptr())))
        return out

    def gradient(self, psi, axis: int, out=None):
        """d_axis psi through Fourier space."""
        import torch
        nst = self._block(psi)
        if out is None:
            out = torch.empty_like(psi)
        _check(lib().tdh_gradient(self._h, nst, C.c_void_p(psi.data_ptr()), int(axis), C.c_void_p(out.data_ptr())))
        return out

    def forces(self, psi, natoms: Optional[int] = None, occ=None, vloc_atoms=None):
        """Eq. 11 per atom and axis -> (natoms, 3) host numpy; vloc_atoms: device float64 (natoms, n0, n1, n2) or None.
        natoms is the atom count of the installed projector table (checked when given: it sizes the result buffer)."""
        import torch
        nst = self._block(psi)
        if natoms is None:
            natoms = self.natoms
        if natoms != self.natoms:
            raise TdhError(TDH_EINVAL, f"forces: natoms = {natoms} but the installed projector table has {self.natoms} atoms")
        occ_arr = None if occ is None else np.ascontiguousarray(occ, dtype=np.float64)
        assert occ_arr is None or occ_arr.size == nst
        if vloc_atoms is not None:
            assert vloc_atoms.is_cuda and vloc_atoms.dtype == torch.float64 and vloc_atoms.is_contiguous()
            assert vloc_atoms.numel() == natoms * self.npts
        out = np.zeros((natoms, 3), dtype=np.float64)
        _check(lib().tdh_forces(self._h, nst, C.c_void_p(psi.data_ptr()),
                                None if occ_arr is None else C.c_void_p(occ_arr.ctypes.data),
                                None if vloc_atoms is None else C.c_void_p(vloc_atoms.data_ptr()),
                                C.c_void_p(out.ctypes.data)))
        return out

    def subspace_diag(self, psi, hpsi, out=None, want_eig: bool = True):
        """Ritz values (ascending, host numpy; None with want_eig=False) and Ritz vectors out = psi V of an orthonormal
        block; hpsi = H psi with a Hermitian H.  Raises TdhError when the eigensolver has not converged."""
        import torch
        nst = self._block(psi)
        assert self._block(hpsi) == nst
        if out is None:
            out = torch.empty_like(psi)
        eig = np.empty(nst, dtype=np.float64) if want_eig else None
        _check(lib().tdh_subspace_diag(self._h, nst, C.c_void_p(psi.data_ptr()), C.c_void_p(hpsi.data_ptr()),
                                       C.c_void_p(out.data_ptr()), None if eig is None else C.c_void_p(eig.ctypes.data)))
        return eig, out

    def sd_step(self, psi, lam: float, work=None, want_eig: bool = True):
        """One Teter-preconditioned steepest-descent update in place; returns the Rayleigh quotients before the update."""
        import torch
        nst = self._block(psi)
        if work is None:
            work = torch.empty_like(psi)
        assert self._block(work) == nst
        eig = np.empty(nst, dtype=np.float64) if want_eig else None
        _check(lib().tdh_sd_step(self._h, nst, C.c_void_p(psi.data_ptr()), C.c_void_p(work.data_ptr()), float(lam),
                                 None if eig is None else C.c_void_p(eig.ctypes.data)))
        return eig

    def fft3d(self, psi, sign: int):
        nst = self._block(psi)
        _check(lib().tdh_fft3d(self._h, nst, C.c_void_p(psi.data_ptr()), int(sign)))
        return psi

    # -- slab decomposition (one handle per rank; shard.SlabGroup drives the phases)
    def slab_buffers(self):
        """(fs, rs, dpi) device addresses of this rank's exchange buffers (dpi is 0 without projectors)."""
        fs, rs, dp = C.c_void_p(), C.c_void_p(), C.c_void_p()
        _check(lib().tdh_slab_buffers(self._h, C.byref(fs), C.byref(rs), C.byref(dp)))
        return fs.value or 0, rs.value or 0, dp.value or 0

    def slab_set_peers(self, fs: Sequence[int], rs: Sequence[int], dpi: Optional[Sequence[int]] = None):
        w = len(fs)
        arr = lambda xs: (C.c_void_p * w)(*[C.c_void_p(int(x)) for x in xs])
        _check(lib().tdh_slab_set_peers(self._h, arr(fs), arr(rs), None if dpi is None else arr(dpi)))

    def slab_apply_phase(self, phase: int, psi, out=None):
        nst = self._block(psi)
        _check(lib().tdh_slab_apply_phase(self._h, int(phase), nst, C.c_void_p(psi.data_ptr()),
                                          None if out is None else C.c_void_p(out.data_ptr())))

    def slab_fft_phase(self, sign: int, phase: int, block):
        nst = self._block(block)
        _check(lib().tdh_slab_fft_phase(self._h, int(sign), int(phase), nst, C.c_void_p(block.data_ptr())))

    def work_layout(self):
        """(rowmap, colmap): plane row rowmap[ky] / column colmap[kz] of the work layout holds frequency index ky / kz."""
        ny, nz = self.n_full[1], self.n_full[2]
        r, c = (C.c_int * ny)(), (C.c_int * nz)()
        _check(lib().tdh_work_layout(self._h, r, c))
        return np.array(r[:], dtype=np.int64), np.array(c[:], dtype=np.int64)

    # -- host entry points (end-to-end path)
    def apply_hamiltonian_host(self, psi_host, out_host):
        nst = psi_host.size // self.npts if isinstance(psi_host, np.ndarray) else psi_host.numel() // self.npts
        _check(lib().tdh_apply_hamiltonian_host(self._h, int(nst), C.c_void_p(_host_ptr(psi_host)),
                                                C.c_void_p(_host_ptr(out_host))))
        return out_host

    def propagate_host(self, psi_host, dt: float, nsteps: int, order: int = 4):
        nst = psi_host.size // self.npts if isinstance(psi_host, np.ndarray) else psi_host.numel() // self.npts
        _check(lib().tdh_propagate_host(self._h, int(nst), C.c_void_p(_host_ptr(psi_host)), float(dt), int(nsteps),
                                        int(order)))
        return psi_host

    # -- statistics / knobs
    def last_jacobi_sweeps(self) -> int:
        return int(lib().tdh_last_jacobi_sweeps(self._h))

    def last_launch_count(self) -> int:
        return int(lib().tdh_last_launch_count(self._h))

    def set_profiling(self, on: bool):
        _check(lib().tdh_set_profiling(self._h, 1 if on else 0))

    def last_kernel_seconds(self) -> dict:
        buf = (C.c_double * NKERNELS)()
        _check(lib().tdh_last_kernel_seconds(self._h, buf))
        return {lib().tdh_kernel_name(i).decode(): buf[i] for i in range(NKERNELS)}

    def set_chunk_states(self, chunk: int):
        _check(lib().tdh_set_chunk_states(self._h, int(chunk)))

    def reserve(self, rotation_states: int = 0, forces_local_term: bool = False, host_buffers: bool = False):
        _check(lib().tdh_reserve(self._h, int(rotation_states), int(bool(forces_local_term)), int(bool(host_buffers))))


def ipc_export(dev_ptr: int) -> bytes:
    """64-byte CUDA IPC token of a handle-owned device buffer."""
    buf = C.create_string_buffer(64)
    _check(lib().tdh_ipc_export(C.c_void_p(int(dev_ptr)), buf))
    return buf.raw


def ipc_import(token: bytes) -> int:
    p = C.c_void_p()
    _check(lib().tdh_ipc_import(C.create_string_buffer(token, 64), C.byref(p)))
    return p.value


def ipc_close(dev_ptr: int):
    _check(lib().tdh_ipc_close(C.c_void_p(int(dev_ptr))))


def grid_for(wl, max_states: Optional[int] = None, device_v=None) -> Grid:
    """Create a Grid for a workloads.Workload and load its potential and projectors."""
    import torch
    c = wl.cfg
    g = Grid(c.n, c.length, c.kpt, c.ecut_abi, max_states or c.nst)
    v = device_v if device_v is not None else torch.from_numpy(wl.v).cuda()
    g.set_potential(v)
    g.set_projectors(wl.proj)
    return g
