"""Chunk-size sweep: python -m paper_2106_03872_b200.tune <workload> <nst> <c1,c2,...>  (tuning aid; needs a GPU)."""
import sys, os, statistics
import torch, numpy as np
from paper_2106_03872_b200 import workloads as W, binding as B
name = sys.argv[1] if len(sys.argv) > 1 else "large"
nst = int(sys.argv[2]) if len(sys.argv) > 2 else 256
chunks = [int(x) for x in sys.argv[3].split(",")] if len(sys.argv) > 3 else [1,2,4,8,16,32,64]
cfg = W.CONFIGS[name]; wl = W.make(cfg)
psi = torch.randn((nst,)+cfg.n, dtype=torch.complex128, device="cuda")
out = torch.empty_like(psi)
g = B.grid_for(wl, max_states=nst)
units = nst*cfg.npts
for c in chunks:
    g.set_chunk_states(c)
    for _ in range(2): g.apply_hamiltonian(psi, out=out)
    torch.cuda.synchronize()
    ts=[]
    for _ in range(5):
        e0=torch.cuda.Event(enable_timing=True); e1=torch.cuda.Event(enable_timing=True)
        e0.record(); g.apply_hamiltonian(psi, out=out); e1.record(); torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1)*1e-3)
    t=statistics.median(ts)
    g.set_profiling(True); g.apply_hamiltonian(psi,out=out); torch.cuda.synchronize(); ks=g.last_kernel_seconds(); g.set_profiling(False)
    print(f"{name} nst={nst} chunk={c:4d}: {t*1e3:8.3f} ms  {units/t:.3e} st.pt/s  strict {32*units/t*1e-9:7.1f} GB/s  launches {g.last_launch_count()}  " + " ".join(f"{k}={v*1e3:.3f}" for k,v in ks.items()), flush=True)
