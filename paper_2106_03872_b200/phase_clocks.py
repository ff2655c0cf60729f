"""Phase clocks of tile_inv: where a tile's time goes, per warp group (diagnostic, not on the product path).

Needs a library built with the phase marks compiled in:

    TDH_NVCC_FLAGS=-DTDH_PHASE_CLOCKS python -m paper_2106_03872_b200.build --force
    python -m paper_2106_03872_b200.phase_clocks large 128 full      # workload, states, full | noproj
    python -m paper_2106_03872_b200.build --force                    # back to the product build

Thread 0 of every warp group accumulates clock64() ticks between the marks of tile_kernels.cuh (TDH_MARK); the
library sums them over all groups (tdh_debug_phase_ticks, exported only by such a build).  TDH_NL_MODE=0 selects the
fused back-projection (records inside tile_inv), which is what the 'record layers' column measures.
"""
from __future__ import annotations

import ctypes as C
import sys

NAMES = ["wait X", "yA'", "yB'", "zA'", "zB' in place", "record layers", "epilogue", "release+issue"]


def main(argv):
    import torch
    from . import binding, workloads as W
    name = argv[1] if len(argv) > 1 else "large"
    nst = int(argv[2]) if len(argv) > 2 else 128
    variant = argv[3] if len(argv) > 3 else "full"
    lib = binding.lib()
    if not hasattr(lib, "tdh_debug_phase_ticks"):
        raise SystemExit("this libtdh.so was built without -DTDH_PHASE_CLOCKS (see the module docstring)")
    cfg = W.CONFIGS[name]
    wl = W.make(cfg)
    torch.manual_seed(W.BASE_SEED + cfg.cid)
    psi = torch.randn(nst, *cfg.n, dtype=torch.complex128, device="cuda")
    out = torch.empty_like(psi)
    with binding.Grid(cfg.n, cfg.length, cfg.kpt, cfg.ecut_abi, nst) as g:
        g.set_potential(torch.from_numpy(wl.v).cuda())
        g.set_projectors(wl.proj if variant == "full" else None)
        buf = (C.c_ulonglong * 16)()
        for _ in range(2):
            g.apply_hamiltonian(psi, out)
        lib.tdh_debug_phase_ticks(buf)                      # reading resets the counters
        reps = 3
        for _ in range(reps):
            g.apply_hamiltonian(psi, out)
        lib.tdh_debug_phase_ticks(buf)
    split = 2 if cfg.n[1] * cfg.n[2] >= 6144 else 1          # plane parts per (state, x) plane
    ntiles = nst * cfg.n[0] * split * reps
    print(f"{name} {variant}: ticks per tile and warp group: " +
          " | ".join(f"{n} {buf[i] / ntiles:.0f}" for i, n in enumerate(NAMES)) + f" | total {sum(buf[:8]) / ntiles:.0f}")


if __name__ == "__main__":
    main(sys.argv)
