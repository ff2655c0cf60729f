#!/usr/bin/env python
"""bench.py -- H|psi> throughput of libtdh.so on B200 (one JSON line on stdout, rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload large] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one tdh_apply_hamiltonian call (rows a1-a6 of DESIGN.md section 1) over the whole state block of the
workload; metric = states*gridpoints/s in complex128.  Default workload: "large" (BASELINE.json configs[3]:
96^3 grid, 1024 states, 13.5 GiB block -- far larger than the 126 MB L2, so no flush is needed between steps).
Row a7 (Taylor-4 propagate, 4 H applications + fused axpys per step) is timed beside it on the "tddft" config and
reported under "propagate"; the other configs are reported under "workloads" (context, not the headline).

Keys beyond the driver's contract: "roofline" (dominant kernel family, CUDA events on the launching stream),
"cpu_baseline" (the CPU oracle as it stands on a bounded sample; N=1 only), "kernels" (per-family seconds per step),
"propagate", "workloads".

--impl reference times the CPU oracle (oracle/ref_tdh.c, OpenMP over states) on the host cores, each step a bounded
sample of the same workload.  The oracle is imported only by that leg and by the cpu_baseline leg.
With N > 1 every rank owns its own block of `nst` states (distinct seeds; weak scaling, no data-path collective:
PAPER.md:438 -- states are independent); torch.distributed only carries the barrier and the max-over-ranks time.
"""
from __future__ import annotations

import argparse
import concurrent.futures as cf
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

from paper_2106_03872_b200 import workloads as W

METRIC = "H|psi> states*gridpoints/s (complex128)"
UNIT = "states*gridpoints/s"

# Algorithmic bytes per state*gridpoint of each kernel family: what the launch must read and
# write if nothing were cached.  plane_inv: spectrum in (16) + phi for V*phi (16) + out (16); +16 with an axpy addend.
# nl_project / nl_scatter: 16 / 32 bytes per sphere point and state (filled in per workload by alg_bytes).
# small_h (the one-launch on-chip kernel of 16^3 / 32^3 grids): psi in (16) + H psi out (16), the strict bound; +16 with
# an axpy addend.
ALG_BYTES = {"nl_project": None, "plane_fwd": 32.0, "xpencil": 32.0, "plane_inv": 48.0, "nl_scatter": None, "small_h": 32.0}


def parse_args():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=10)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--workload", default="large", choices=list(W.CONFIG_ORDER))
    p.add_argument("--states", type=int, default=0, help="override the number of states per GPU (0 = the config's)")
    p.add_argument("--chunk", type=int, default=0, help="tdh_set_chunk_states (0 = library default)")
    p.add_argument("--no-sweep", action="store_true", help="skip the other configs / propagate legs")
    p.add_argument("--no-e2e", action="store_true")
    p.add_argument("--no-cpu-baseline", action="store_true")
    p.add_argument("--cpu-sample-states", type=int, default=0, help="states in the cpu_baseline sample (0 = auto)")
    return p.parse_args()


# ----------------------------------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------------------------------
def host_states(cfg, s0, s1, pinned=True):
    """States [s0, s1) of the config as a (pinned) host torch tensor; generated per state (seeded) on a thread pool."""
    import torch
    t = torch.empty((s1 - s0,) + tuple(cfg.n), dtype=torch.complex128, pin_memory=pinned)
    a = t.numpy()

    def fill(s):
        a[s - s0] = W.state(cfg, s)

    with cf.ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1)) as ex:
        list(ex.map(fill, range(s0, s1)))
    return t


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while a timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def fp64_gemm_ceiling(torch, n=8192, reps=3):
    """Measured FP64 ceiling of this GPU in the same run: cuBLAS DGEMM n^3 through torch.matmul (a measurement of the
    hardware, not part of the product path).  Returns TFLOP/s."""
    a = torch.randn(n, n, dtype=torch.float64, device="cuda")
    b = torch.randn(n, n, dtype=torch.float64, device="cuda")
    c = torch.matmul(a, b)
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b, out=c)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1) * 1e-3)
    del a, b, c
    return 2.0 * n ** 3 / best * 1e-12


def fp64_tensor_peak(torch, B):
    """FP64 tensor-core ceiling for the contraction legs, measured in this run two ways: a dependent-free
    mma.sync.m8n8k4.f64 issue loop (probe_fp64_mma_peak of libtdh_probe.so, registers only) and cuBLAS DGEMM 8192^3 (torch.matmul).
    The roofline denominator is the larger of the two; the bf16-scaled nominal figure is reported for context only."""
    import ctypes
    from paper_2106_03872_b200 import build as tdh_build
    probe = ctypes.CDLL(tdh_build.build_probe())            # measurement helper, outside the product ABI
    v = ctypes.c_double()
    rc = probe.probe_fp64_mma_peak(ctypes.byref(v))
    if rc != 0:
        raise RuntimeError(f"probe_fp64_mma_peak failed: {rc}")
    issue = float(v.value)
    dgemm = fp64_gemm_ceiling(torch)
    out = {"mma_issue_loop_tflops": round(issue, 2), "cublas_dgemm_8192_tflops": round(dgemm, 2),
           "peak": round(max(issue, dgemm), 2),
           "peak_source": "larger of the mma.sync.m8n8k4.f64 issue loop and cuBLAS DGEMM 8192^3, both measured in this run"}
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            out["bf16_scaled_nominal_tflops"] = round(float(json.load(open(path))["bf16_tflops"]) * 45.0 / 2250.0, 2)
        except Exception:
            pass
    return out


class Dist:
    """torch.distributed plumbing: barrier and max-over-ranks only (no data-path collective)."""

    def __init__(self, want_gpus):
        import torch
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.torch = torch
        if self.world > 1:
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29500")
            torch.cuda.set_device(self.local)
            dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
            self.dist = dist
        else:
            self.dist = None
            if torch.cuda.is_available():
                torch.cuda.set_device(0)
        if want_gpus != self.world and self.rank == 0:
            sys.stderr.write(f"bench.py: --gpus {want_gpus} but WORLD_SIZE={self.world}; using WORLD_SIZE\n")

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max(self, x):
        if self.dist is None:
            return float(x)
        t = self.torch.tensor([x], dtype=self.torch.float64, device="cuda")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


def timed_device(D, fn, steps, warmup):
    """`warmup` untimed calls, then exactly `steps` calls between CUDA events on torch's current stream (the handle's
    stream), barrier + synchronize on both sides; returns max-over-ranks seconds for the `steps` calls."""
    torch = D.torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    D.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    D.barrier()
    return D.max(e0.elapsed_time(e1) * 1e-3)


def timed_each(torch, fn, reps, flush=None):
    """Per-call device times (s); `flush` (a big tensor) is overwritten before each call to evict L2."""
    out = []
    for _ in range(reps):
        if flush is not None:
            flush.add_(1.0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        out.append(e0.elapsed_time(e1) * 1e-3)
    return out


def upload_states(torch, cfg, s0, nst, keep_host):
    """Device block of states [s0, s0+nst); returns (device tensor, pinned host tensor of the first keep_host states)."""
    dev = torch.empty((nst,) + tuple(cfg.n), dtype=torch.complex128, device="cuda")
    step = max(1, min(nst, (1 << 30) // (cfg.npts * 16)))
    host_keep = None
    if keep_host > 0:
        host_keep = host_states(cfg, s0, s0 + keep_host)
        dev[:keep_host].copy_(host_keep, non_blocking=True)
    for a in range(keep_host, nst, step):
        b = min(nst, a + step)
        h = host_states(cfg, s0 + a, s0 + b)
        dev[a:b].copy_(h, non_blocking=True)
        torch.cuda.synchronize()
    torch.cuda.synchronize()
    return dev, host_keep


# ----------------------------------------------------------------------------------------------------------------
# legs
# ----------------------------------------------------------------------------------------------------------------
def kernel_breakdown(torch, g, fn, steps):
    """Per-family device seconds per step from the library's own CUDA events on its stream (profiling pass)."""
    g.set_profiling(True)
    tot, launches = {}, 0
    for _ in range(steps):
        fn()
        torch.cuda.synchronize()
        launches = g.last_launch_count()
        for k, v in g.last_kernel_seconds().items():
            tot[k] = tot.get(k, 0.0) + v
    g.set_profiling(False)
    return {k: v / steps for k, v in tot.items()}, launches


# DRAM bytes per launch measured by ncu (dram__bytes_read.sum + dram__bytes_write.sum, `ncu --set full`), one row per
# kernel family and workload, written from the .ncu-rep of the command named in profiles/r03_ncu_dram.md.  Read at bench
# time for roofline.traffic; a family without a row has traffic null (never a stale constant).
NCU_DRAM_CSV = os.path.join(ROOT, "profiles", "r03_ncu_dram.csv")


def ncu_dram_bytes_per_unit(workload):
    """{family: DRAM bytes per state*gridpoint} for `workload` from the committed ncu table; {} if absent."""
    out = {}
    try:
        with open(NCU_DRAM_CSV) as f:
            head = f.readline().strip().split(",")
            for line in f:
                row = dict(zip(head, line.strip().split(",")))
                if row.get("workload") == workload:
                    out[row["family"]] = (float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])) / float(row["units_per_launch"])
    except (OSError, KeyError, ValueError, ZeroDivisionError):
        return {}
    return out


def alg_bytes(wl):
    """ALG_BYTES with the gather of the projection kernel filled in: 16 bytes per sphere point and state."""
    b = dict(ALG_BYTES)
    b["nl_project"] = 16.0 * float(wl.proj.sph_off[-1]) / wl.cfg.npts if wl.proj.natoms else None
    # back-projection kernel (large grids): read-modify-write of the same points of the output block
    b["nl_scatter"] = 32.0 * float(wl.proj.sph_off[-1]) / wl.cfg.npts if wl.proj.natoms else None
    return b


def nl_flops_per_unit(wl):
    """Useful flop per state*gridpoint of each projector kernel: 8 * sum_I C_I P_I / N_p (real matrix x complex block)."""
    pr = wl.proj
    if not pr.natoms:
        return 0.0
    cp = sum(int(pr.chan_off[i + 1] - pr.chan_off[i]) * int(pr.sph_off[i + 1] - pr.sph_off[i]) for i in range(pr.natoms))
    return 8.0 * cp / wl.cfg.npts


def roofline_of(kern_s, units, peak_gbs, peak_src, bytes_per_unit, workload=None, units_per_launch=None, nl_flops=0.0,
                step_s=None):
    """Roofline object for the dominant kernel family (largest share of the step) + the fractions of the others, the
    step against its pass structure (sum of the families' algorithmic bytes) and against the 32 compulsory bytes."""
    cand = {k: v for k, v in kern_s.items() if bytes_per_unit.get(k) and v > 0}
    if not cand:
        return None
    top = max(cand, key=cand.get)
    achieved = bytes_per_unit[top] * units / cand[top] * 1e-9
    tot = sum(kern_s.values())
    others = {k: {"achieved": round(bytes_per_unit[k] * units / v * 1e-9, 1),
                  "frac": round(bytes_per_unit[k] * units / v * 1e-9 / peak_gbs, 4),
                  "algorithmic_bytes_per_unit": round(bytes_per_unit[k], 3),
                  "share_of_step": round(v / tot, 4)} for k, v in cand.items()}
    for k in ("nl_project", "nl_scatter"):
        if k in others and nl_flops > 0:
            # the contraction is byte bound: its useful FP64 rate is reported, the bytes govern
            others[k]["useful_tflops"] = round(nl_flops * units / cand[k] * 1e-12, 2)
    traffic = None
    per_unit = ncu_dram_bytes_per_unit(workload).get(top)
    if per_unit and units_per_launch:
        traffic = {"bytes_per_launch": per_unit * units_per_launch, "algorithmic_bytes_per_launch":
                   bytes_per_unit[top] * units_per_launch, "units_per_launch": units_per_launch,
                   "source": "profiles/r03_ncu_dram.csv (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum of one "
                             "launch per state*gridpoint, scaled to this run's launch size)"}
    t = step_s if step_s else tot
    pass_bytes = sum(bytes_per_unit[k] for k in cand)
    # what the step really moves: the ncu DRAM bytes per unit of every family that ran (committed captures), against the
    # step time -- the gather / scatter kernels fetch whole 128-byte lines around their z-runs, the FFT kernels move their
    # algorithmic bytes
    ncu_all = ncu_dram_bytes_per_unit(workload)
    dram = None
    if all(k in ncu_all for k in cand):
        dram_bytes = sum(ncu_all[k] for k in cand)
        dram = {"bytes_per_unit": round(dram_bytes, 2), "frac": round(dram_bytes * units / t * 1e-9 / peak_gbs, 4),
                "per_kernel_frac": {k: round(ncu_all[k] * units / cand[k] * 1e-9 / peak_gbs, 4) for k in cand},
                "note": "ncu dram__bytes (read + write) per state*gridpoint of every family (profiles/r03_ncu_dram.csv) x units "
                        "/ step time (per_kernel_frac: / the family's CUDA-event time) / HBM peak"}
    return {"kernel": top, "bound": "hbm", "achieved": round(achieved, 1), "peak": peak_gbs, "unit": "GB/s",
            "frac": round(achieved / peak_gbs, 4), "traffic": traffic, "peak_source": peak_src,
            "algorithmic_bytes_per_unit": bytes_per_unit[top], "units_per_step": units,
            "share_of_step": round(cand[top] / tot, 4), "all_kernels": others,
            "pass_structure": {"bytes_per_unit": round(pass_bytes, 2),
                               "frac": round(pass_bytes * units / t * 1e-9 / peak_gbs, 4),
                               "note": "sum of the families' algorithmic bytes x units / step time / HBM peak"},
            "strict_32B": {"frac": round(32.0 * units / t * 1e-9 / peak_gbs, 4),
                           "note": "compulsory traffic (read psi + write H psi) x units / step time / HBM peak"},
            "dram_traffic": dram,
            "note": "achieved = algorithmic bytes of all launches of this family in one step / their summed CUDA-event "
                    "time (separate profiling pass of the same steps)"}


def cpu_baseline(cfg, wl, sample_states, budget_s=12.0):
    """The CPU oracle as it stands on a bounded sample of the same workload (states [0, S)); the whole block when that
    takes less than `budget_s` seconds."""
    from oracle import ref
    cores = ref.num_threads()
    cal = W.states(cfg, 0, min(cfg.nst, cores))
    t0 = time.perf_counter()
    ref.apply_workload(wl, cal, ref.NAIVE_FFT)
    rate = cal.shape[0] * cfg.npts / (time.perf_counter() - t0)
    S = sample_states or int(min(cfg.nst, max(cores, cores * round(rate * budget_s / cfg.npts / cores))))
    S = max(1, min(S, cfg.nst))
    psi = W.states(cfg, 0, S)
    t0 = time.perf_counter()
    ref.apply_workload(wl, psi, ref.NAIVE_FFT)
    dt = time.perf_counter() - t0
    return {"value": S * cfg.npts / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"states [0,{S}) of '{cfg.name}' ({S} of {cfg.nst} states x {cfg.n[0]}^3 points), one "
                      f"ref_apply_hamiltonian call (naive radix-2/3 FFT back-end, OpenMP over states), {dt:.2f} s"}


def cpu_baseline_propagate(cfg, wl, budget_s=15.0):
    """ref_propagate (Eq. 8 literally) on a bounded state sample of the TDDFT config, all of its steps."""
    from oracle import ref
    cores = ref.num_threads()
    cal = W.states(cfg, 0, min(cfg.nst, cores))
    t0 = time.perf_counter()
    ref.propagate_workload(wl, cal, dt=cfg.dt, nsteps=1, backend=ref.NAIVE_FFT)
    per_state_step = (time.perf_counter() - t0) / cal.shape[0]
    S = int(max(cores, min(cfg.nst, cores * max(1, round(budget_s / (per_state_step * cfg.nsteps * cores))))))
    S = min(S, cfg.nst)
    psi = W.states(cfg, 0, S)
    t0 = time.perf_counter()
    ref.propagate_workload(wl, psi, dt=cfg.dt, nsteps=cfg.nsteps, backend=ref.NAIVE_FFT)
    dt = time.perf_counter() - t0
    return {"value": S * cfg.npts * 4 * cfg.nsteps / dt, "unit": UNIT + " (H-application equivalents)", "cores": cores,
            "kind": "oracle", "steps_per_s": cfg.nsteps / dt * S / cfg.nst,
            "sample": f"states [0,{S}) of '{cfg.name}' ({S} of {cfg.nst} states), one ref_propagate call of {cfg.nsteps} "
                      f"Taylor-4 steps, {dt:.2f} s; steps_per_s scaled to the whole block"}


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores; each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import ref
    cfg = W.CONFIGS[args.workload]
    wl = W.make(cfg)
    cores = ref.num_threads()
    S = args.cpu_sample_states or min(cfg.nst, 4 * cores)
    psi = W.states(cfg, 0, S)
    for _ in range(args.warmup):
        ref.apply_workload(wl, psi, ref.NAIVE_FFT)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ref.apply_workload(wl, psi, ref.NAIVE_FFT)
    dt = time.perf_counter() - t0
    val = args.steps * S * cfg.npts / dt
    sample = f"each step = states [0,{S}) of '{cfg.name}' through ref_apply_hamiltonian (naive FFT back-end)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "grid": list(cfg.n), "states_per_step": S, "atoms": cfg.natoms},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# The general-axis-length path (any 2^a 3^b length; generic_fft.cuh) on a grid outside the tuned set: five launches per
# application -- forward z and forward y booked under plane_fwd (2 x 32 B), x under xpencil (32 B), inverse y and
# inverse z + epilogue under plane_inv (32 + 48 B): 176 B per state*gridpoint against the tuned path's 112 (DESIGN.md
# section 15).  72^3 is what a cutoff-derived grid between the 64^3 and 96^3 configs looks like.
GENERAL_72 = W.test_config(172, (72, 72, 72), (24.0, 24.0, 24.0), nst=256, natoms=32, placement="lattice", lattice=(4, 4, 2),
                           lmax=1, rc=2.5, dl=(2.0, -0.8))
GENERAL_BYTES = {"plane_fwd": 64.0, "xpencil": 32.0, "plane_inv": 80.0}


def sweep_leg(torch, B, name, flush, peak, peak_src, cpu, reps=7, cfg=None, family_bytes=None):
    """One of the non-headline configs at its full size: apply_hamiltonian cold (L2 flushed) and L2-hot, its roofline
    object (dominant family, pass-structure and strict fractions) and the CPU oracle beside it.  cfg / family_bytes:
    a config outside W.CONFIGS and the algorithmic bytes of its kernel families where they differ from ALG_BYTES."""
    cfg = cfg or W.CONFIGS[name]
    wl = W.make(cfg)
    psi, _ = upload_states(torch, cfg, 0, cfg.nst, 0)
    out = torch.empty_like(psi)
    units = cfg.nst * cfg.npts
    with B.grid_for(wl) as g:
        fn = lambda: g.apply_hamiltonian(psi, out=out)
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        cold = statistics.median(timed_each(torch, fn, reps, flush))
        hot = statistics.median(timed_each(torch, fn, reps, None))
        res = {"states": cfg.nst, "grid": cfg.n[0], "value": units / cold, "ms": cold * 1e3,
               "value_l2_hot": units / hot, "ms_l2_hot": hot * 1e3, "launches": g.last_launch_count()}
        # per-family times (library events, L2 flushed before every call) -> this config's roofline object
        g.set_profiling(True)
        tot = {}
        for _ in range(5):
            flush.add_(1.0)
            fn()
            torch.cuda.synchronize()
            for k, v in g.last_kernel_seconds().items():
                tot[k] = tot.get(k, 0.0) + v / 5
        g.set_profiling(False)
        ab = alg_bytes(wl)                           # families that did not run (nl_scatter on whole-plane tiles) drop out
        ab.update(family_bytes or {})
        res["kernels_s_per_step"] = tot
        res["roofline"] = roofline_of(tot, units, peak, peak_src, ab, name, units, nl_flops_per_unit(wl), step_s=cold)
        if res["roofline"] and units * 32 < 100e6:
            res["roofline"]["note"] += ("; the block and its output fit the 126 MB L2 several times over, the bytes of this "
                                        "config are not the bound: launch latency is (see ms_per_call_in_a_100_call_loop)")
        if cpu:
            res["cpu_baseline"] = cpu_baseline(cfg, wl, 0)
        if name in ("tiny", "small"):
            # launch-latency regime: 100 back-to-back calls, one pair of events around the loop
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(100):
                fn()
            e1.record()
            torch.cuda.synchronize()
            res["ms_per_call_in_a_100_call_loop"] = e0.elapsed_time(e1) / 100
            # row a7 in the launch-latency regime: 20 Taylor-4 steps in one tdh_propagate call, replayed as one CUDA graph
            # (captured on the first call), and the same call as plain launches (a second handle with TDH_GRAPH=0)
            nsteps_p = 20
            work = psi.clone()

            def prop_ms(gg):
                gg.propagate(work, cfg.dt, nsteps_p)
                torch.cuda.synchronize()
                return statistics.median(timed_each(torch, lambda: gg.propagate(work, cfg.dt, nsteps_p), 5, None)) * 1e3
            ms_graph = prop_ms(g)
            launches = g.last_launch_count()
            old_env = os.environ.get("TDH_GRAPH")
            os.environ["TDH_GRAPH"] = "0"
            try:
                with B.grid_for(wl) as g2:
                    work.copy_(psi)
                    ms_plain = prop_ms(g2)
            finally:
                if old_env is None:
                    del os.environ["TDH_GRAPH"]
                else:
                    os.environ["TDH_GRAPH"] = old_env
            res["propagate"] = {"steps": nsteps_p, "dt": cfg.dt, "ms_cuda_graph": ms_graph, "ms_plain_launches": ms_plain,
                                "launches": launches,
                                "h_application_equivalents_per_s": units * 4 * nsteps_p / (ms_graph * 1e-3), "unit": UNIT}
            del work
        if name == "tddft":
            # row a7: the config's 20 Taylor-4 steps (80 H applications + fused axpys) in one tdh_propagate call
            work = psi.clone()
            g.propagate(work, cfg.dt, 1)
            torch.cuda.synchronize()
            work.copy_(psi)
            ts = timed_each(torch, lambda: g.propagate(work, cfg.dt, cfg.nsteps), 1, flush)
            t = ts[0]
            res["propagate"] = {"steps": cfg.nsteps, "dt": cfg.dt, "seconds": t, "steps_per_s": cfg.nsteps / t,
                                "h_application_equivalents_per_s": units * 4 * cfg.nsteps / t, "unit": UNIT,
                                "launches": g.last_launch_count(),
                                "pass_structure_frac": round((ALG_BYTES["plane_fwd"] + ALG_BYTES["xpencil"] + ALG_BYTES["plane_inv"]
                                                              + 16.0 + (ab["nl_project"] or 0.0)) * units * 4 * cfg.nsteps / t
                                                             * 1e-9 / peak, 4),
                                "strict_32B_frac": round(32.0 * units * 4 * cfg.nsteps / t * 1e-9 / peak, 4)}
            if cpu:
                res["propagate"]["cpu_baseline"] = cpu_baseline_propagate(cfg, wl)
            # NEXT-1: ETRS steps (Eq. 6-7) with the shared-powers pair: 8 H applications per step
            # instead of the 12 of three separate exponentials
            work.copy_(psi)
            vdev = torch.from_numpy(wl.v).cuda()
            g.etrs_step(work, cfg.dt, vdev, approx=out)
            torch.cuda.synchronize()
            work.copy_(psi)
            nsteps_e = 5

            def etrs():
                for _ in range(nsteps_e):
                    g.etrs_step(work, cfg.dt, vdev, approx=out)
            te = timed_each(torch, etrs, 1, flush)[0]
            res["etrs"] = {"steps": nsteps_e, "dt": cfg.dt, "seconds_per_step": te / nsteps_e,
                           "h_applications_per_step": 8, "h_application_equivalents_per_s": units * 8 * nsteps_e / te,
                           "unit": UNIT, "note": "tdh_etrs_step: taylor pair (4 H) + potential switch + half step (4 H)"}
            # NEXT-2: density (Eq. 1) of the whole block, Hartree solve, and the self-consistent (Hartree-only) ETRS step
            dens = g.density(psi)
            vh = g.hartree(dens)
            torch.cuda.synchronize()
            td = statistics.median(timed_each(torch, lambda: g.density(psi, out=dens), 5, flush))
            th = statistics.median(timed_each(torch, lambda: g.hartree(dens, out=vh), 5, None))
            work.copy_(psi)

            def scf_step():
                g.set_potential(vdev + g.hartree(g.density(work)))
                approx = g.taylor_pair(work, cfg.dt, full=out)
                g.set_potential(vdev + g.hartree(g.density(approx)))
                g.propagate(work, 0.5 * cfg.dt, 1)
            scf_step()
            torch.cuda.synchronize()
            work.copy_(psi)
            ts = timed_each(torch, scf_step, 1, flush)[0]
            res["density_hartree"] = {
                "density_seconds": td, "density_gbs": units * 16 / td * 1e-9, "hartree_seconds": th,
                "self_consistent_etrs_seconds_per_step": ts,
                "note": "tdh_density over the whole block (16 B per state*gridpoint read), tdh_hartree (one-state FFT pair, "
                        "launch bound), and one ETRS step with V(t+dt) = V_ext + v_H[n(t+dt)] rebuilt from Eq. 7's states"}
            g.set_potential(vdev)
            # overlap matrix S = dV psi^H psi of the whole block: the one flop-bound contraction (FP64 tensor cores)
            smat = g.overlap(psi, out)                   # two different blocks: every tile is computed
            torch.cuda.synchronize()
            to = statistics.median(timed_each(torch, lambda: g.overlap(psi, out, out=smat), 5, flush))
            tg = statistics.median(timed_each(torch, lambda: g.overlap(psi, out=smat), 5, flush))
            pk = fp64_tensor_peak(torch, B)
            tf = 8.0 * cfg.nst * cfg.nst * cfg.npts / to * 1e-12
            res["overlap"] = {"seconds": to, "bound": "tensor", "achieved": round(tf, 2), "peak": pk["peak"],
                              "unit": "TFLOP/s", "frac": round(tf / pk["peak"], 4), "peak_source": pk["peak_source"],
                              "flops": "8 * nst^2 * N_p (complex128 GEMM, K = N_p)", "gram_seconds": tg,
                              "fp64_peaks_same_run": pk,
                              "frac_of_cublas_dgemm": round(tf / pk["cublas_dgemm_8192_tflops"], 4),
                              "frac_of_mma_issue_loop": round(tf / pk["mma_issue_loop_tflops"], 4),
                              "frac_of_nominal_45": round(tf / 45.0, 4),
                              "note": "tdh_overlap of two blocks: mma.sync.m8n8k4.f64, 64x64 tiles, split-K with ordered reduction; "
                                      "gram_seconds: one block with itself (tiles below the diagonal mirrored)"}
            work.copy_(psi)
            tsd = statistics.median(timed_each(torch, lambda: g.sd_step(work, 0.05, work=out, want_eig=False), 3, flush))
            res["sd_step"] = {"seconds": tsd, "launches": g.last_launch_count(),
                              "note": "tdh_sd_step on the whole block: H psi, T psi, Rayleigh quotients, residual, Teter "
                                      "preconditioner pass with the fused update (about 2.7 H-application equivalents)"}
            tfo = statistics.median(timed_each(torch, lambda: g.forces(psi, cfg.natoms), 3, flush))
            res["forces"] = {"seconds": tfo, "launches": g.last_launch_count(),
                             "note": "tdh_forces (Eq. 11, non-local part) of the whole block: forward transform, three gradient "
                                     "chains, four projector gathers per state (host timer incl. the result copy)"}
            hps = g.apply_hamiltonian(work)
            tsub = statistics.median(timed_each(torch, lambda: g.subspace_diag(work, hps, out=out), 3, flush))
            res["subspace_diag"] = {"seconds": tsub, "launches": g.last_launch_count(),
                                    "note": "tdh_subspace_diag: overlap psi^H (H psi), cooperative parallel Jacobi eigensolver of "
                                            "the nst x nst matrix, rotation psi V (host timer incl. the eigenvalue copy)"}
            del hps
            tor = statistics.median(timed_each(torch, lambda: g.orthonormalize(psi, out=out), 3, flush))
            res["orthonormalize"] = {"seconds": tor, "launches": g.last_launch_count(),
                                     "effective_tflops": round(12.0 * cfg.nst * cfg.nst * cfg.npts / tor * 1e-12, 2),
                                     "note": "tdh_orthonormalize: overlap (8 n^2 N_p flop) + cooperative Cholesky + triangular "
                                             "inverse + upper-triangular rotation (4 n^2 N_p flop)"}
    del psi, out
    torch.cuda.empty_cache()
    return res


def block_sweep(torch, g, psi, out, cfg, blocks=(32, 128, 512, 1024)):
    """Config 4's sweep: the whole block submitted as consecutive sub-blocks of b states (PAPER.md:456 batching claim)."""
    res = {}
    nst = psi.shape[0]
    for b in blocks:
        if b > nst:
            continue

        def fn():
            for s0 in range(0, nst, b):
                g.apply_hamiltonian(psi[s0:s0 + b], out=out[s0:s0 + b])

        fn()
        torch.cuda.synchronize()
        t = statistics.median(timed_each(torch, fn, 3, None))
        res[str(b)] = nst * cfg.npts / t
    return res


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    from paper_2106_03872_b200 import binding as B
    B.lib()                                            # fails loudly if libtdh.so is missing (no fallback)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback (use --impl reference for the oracle)")
    D = Dist(args.gpus)
    cfg = W.CONFIGS[args.workload]
    nst = args.states or cfg.nst
    wl = W.make(cfg)
    units = nst * cfg.npts                              # per GPU and step
    s_first = D.rank * nst                              # weak scaling: every rank its own states (distinct seeds)
    # e2e host buffers: the whole block when it fits the host comfortably, else a bounded part (stated in the output)
    e2e_states = 0 if args.no_e2e else (nst if D.world <= 2 else min(nst, 256))
    psi, host_in = upload_states(torch, cfg, s_first, nst, e2e_states)
    hpsi = torch.empty_like(psi)
    g = B.grid_for(wl, max_states=nst)
    if args.chunk:
        g.set_chunk_states(args.chunk)
    fn = lambda: g.apply_hamiltonian(psi, out=hpsi)

    # ---- headline: device-resident, K steps
    sampler = ClockSampler(D.local)
    fn(); torch.cuda.synchronize()
    sampler.start()
    t = timed_device(D, fn, args.steps, args.warmup)
    clocks = sampler.stop()
    launches = g.last_launch_count() * args.steps
    value = D.world * units * args.steps / t

    # ---- per-kernel times (same steps, library events on the launching stream) -> roofline of the dominant family
    kern_s, _ = kernel_breakdown(torch, g, fn, max(1, min(args.steps, 5)))
    peak, peak_src = measured_peaks()
    cap = max(1, (4 << 30) // (cfg.npts * 16))                                   # the library's default chunk
    states_per_launch = args.chunk or (nst if cap >= nst else (cap // 8 * 8 if cap >= 8 else cap))
    ab = alg_bytes(wl)
    roof = roofline_of(kern_s, units, peak, peak_src, ab, args.workload, states_per_launch * cfg.npts,
                       nl_flops_per_unit(wl), step_s=t / args.steps)

    # ---- end to end through the host-buffer entry point (pinned host in/out, copies inside the timed region)
    e2e = None
    if e2e_states > 0:
        host_out = torch.empty_like(host_in).pin_memory()
        efn = lambda: g.apply_hamiltonian_host(host_in, host_out)
        for _ in range(min(args.warmup, 2)):
            efn()
        torch.cuda.synchronize(); D.barrier()
        esteps = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(esteps):
            efn()                                        # returns when host_out is complete
        torch.cuda.synchronize()
        te = D.max(time.perf_counter() - t0)
        D.barrier()
        nbytes = e2e_states * cfg.npts * 16
        e2e = {"value": D.world * e2e_states * cfg.npts * esteps / te, "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": esteps, "states_per_gpu": e2e_states,
               "ms_per_step": te / esteps * 1e3,
               "pcie_gbs_per_direction": round(nbytes * esteps / te * 1e-9, 2),
               "bound": "host link: the step moves the block in and out over PCIe (both directions overlap); the kernels "
                        "take %.1f ms of the %.1f ms" % (t / args.steps * 1e3 * e2e_states / nst, te / esteps * 1e3),
               "timer": "host perf_counter around the blocking tdh_apply_hamiltonian_host calls, max over ranks"}
        del host_out
    host_in = None

    extra = {}
    if D.rank == 0 and D.world == 1 and not args.no_sweep:
        # context only: the vendor-library route the paper takes -- cuFFT forward + inverse of a sub-block,
        # nothing else of H; not on the product path
        try:
            sub = psi[:min(nst, 64)]
            tmp = torch.fft.ifftn(torch.fft.fftn(sub, dim=(1, 2, 3)), dim=(1, 2, 3))
            torch.cuda.synchronize()
            ts = []
            for _ in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                tmp = torch.fft.ifftn(torch.fft.fftn(sub, dim=(1, 2, 3)), dim=(1, 2, 3))
                e1.record()
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1) * 1e-3)
            extra["cufft_context"] = {"states": int(sub.shape[0]), "seconds": min(ts), "value": sub.shape[0] * cfg.npts / min(ts),
                                      "unit": UNIT, "note": "torch.fft.fftn + ifftn (cuFFT) of a sub-block: the two transforms "
                                                            "alone, without kinetic scale, V, projectors; context, not a target"}
            del tmp, sub
        except Exception as exc:                            # context line only
            extra["cufft_context"] = {"unavailable": str(exc)[:200]}
        flush = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")       # 256 MB > 126 MB L2
        if args.workload == "large":
            extra["block_sweep_states_per_call"] = block_sweep(torch, g, psi, hpsi, cfg)
        g.close()
        del psi, hpsi
        torch.cuda.empty_cache()
        wls = {}
        for name in W.CONFIG_ORDER:
            if name != args.workload:
                wls[name] = sweep_leg(torch, B, name, flush, peak, peak_src, not args.no_cpu_baseline)
        wls["general_72"] = sweep_leg(torch, B, "general_72", flush, peak, peak_src, not args.no_cpu_baseline,
                                      cfg=GENERAL_72, family_bytes=GENERAL_BYTES)
        wls["general_72"]["note"] = ("general-axis-length path (shared-memory Stockham, five launches, 176 B per unit); "
                                     "72^3 x 256 states, Gamma, 32 atoms")
        extra["workloads"] = wls
        if "tddft" in wls and "propagate" in wls["tddft"]:
            extra["propagate"] = wls["tddft"].pop("propagate")
            extra["etrs"] = wls["tddft"].pop("etrs")
            extra["density_hartree"] = wls["tddft"].pop("density_hartree")
            extra["overlap"] = wls["tddft"].pop("overlap")
            extra["orthonormalize"] = wls["tddft"].pop("orthonormalize")
            extra["sd_step"] = wls["tddft"].pop("sd_step")
            extra["subspace_diag"] = wls["tddft"].pop("subspace_diag")
            extra["forces"] = wls["tddft"].pop("forces")
    else:
        g.close()

    cpu = None
    if D.rank == 0 and D.world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(cfg, wl, args.cpu_sample_states)

    if D.rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": D.world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name}: {cfg.n[0]}^3 grid, {nst} states/GPU complex128, {cfg.natoms} atoms, "
                                   f"{cfg.nchan_per_atom} KB channels/atom, rc={cfg.rc}",
                       "call": "tdh_apply_hamiltonian on the whole block", "states_per_gpu": nst,
                       "l2": "inputs larger than L2 (block of %.1f GB per GPU), no flush" % (units * 16 / 1e9)
                             if units * 16 > 512e6 else "L2-resident block, no flush (use the 'large' workload)",
                       "parallelism": f"states sharded over {D.world} GPU(s), no collective"},
            "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "roofline": roof, "cpu_baseline": cpu,
            "kernels_s_per_step": kern_s,
        }
        line.update(extra)
        print(json.dumps(line))
    D.close()


if __name__ == "__main__":
    main()
