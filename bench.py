#!/usr/bin/env python3
"""bench.py -- the TDDFT-ris derivative-integral hot path on B200 (contract: task prompt "Measurement").

One "step" = one pass of the whole hot path over one batch of synthetic input:
    ris_grad_J(D, c_aux) + ris_grad_K(C_occ, C_vir, B) + ris_grad_PQ(c_aux, d_aux)      (Eq. 27)
for all `nbatch` states of the workload, on a context built once by ris_setup (one-off per geometry, reported
separately as `setup_ms`).  Metric (BASELINE.json): TDDFT-ris gradient ms/state -- with the two other figures of
the metric string (3c2e-derivative primitive triplets/s, % FP64 peak) in the same JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

N > 1 (torchrun), default `--shard aux`: ONE batch of states sharded over the auxiliary index (DESIGN.md
"Multi-GPU"): rank r holds B[:, P_r] only and evaluates ris_grad_J_range / ris_grad_K_range on its block of aux functions,
one NCCL all-reduce of (nbatch_J + nbatch_K) natoms 3 doubles completes the gradients on every rank; total work is fixed,
value = time / nbatch ("scaling": "strong").  `--shard states`: every rank runs the same molecule with its own batch of
states (independent problems), no data-path collective; value = time / (N * nbatch)  ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "TDDFT-ris gradient ms/state"
UNIT = "ms/state"
# ncu counters of the committed `ncu --set full` captures, keyed by config and kernel (profiles/ncu_counters.json, written
# by hand from the profile summaries it names); a (config, kernel) without a committed capture reports null.
def ncu_counters(config: int) -> dict:
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_counters.json")) as f:
            return json.load(f).get(f"config{config}", {})
    except (OSError, ValueError):
        return {}


ORACLE_CUTOFF = {4: 1e-22}      # the oracle's documented primitive cutoff on config 4


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config (1-based); 4 = the largest")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--shard", default="aux", choices=["aux", "states"], help="N > 1: what the ranks split (see the module docstring)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the fit_step / resp_step blocks reported beside the metric "
                    "(profiler runs: the launch list then holds the setup, the peak probes and the steps only)")
    ap.add_argument("--cpu-baseline-full", action="store_true",
                    help="time the oracle over the WHOLE workload (minutes on config 3; not for config 4) and single-threaded")
    ap.add_argument("--oracle-aux", type=int, default=0, help="aux functions in the oracle's timed sample (0 = auto)")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: [self.lines.append(l) for l in self.proc.stdout], daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ oracle leg
def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.lower().startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def set_oracle_threads(n: int):
    """The oracle's OpenMP team size (it is loaded already: set through the OpenMP runtime it linked)."""
    import ctypes
    ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))


def oracle_sample_time(wl, cfg: int, n_aux: int, nstate: int = 1):
    """Time the oracle AS IT STANDS on a bounded sample of the workload: aux functions P in [0, n_aux) (of naux),
    `nstate` state(s): J, K (its Gamma^P assembly -- numpy matmul -- and its integral contraction timed separately) for
    the sample, PQ in full.  n_aux >= naux and nstate = all states: the whole workload, nothing extrapolated.
    Returns a dict: seconds of the sample, ms/state for the whole workload (extrapolated linearly in naux when the sample
    is a part), threads, parts, description."""
    from oracle import ris_oracle as orc
    mol = wl.mol
    cut = ORACLE_CUTOFF.get(cfg, 0.0)
    aux = list(range(min(n_aux, mol.natoms)))
    nsJ, nsK = min(nstate, wl.D.shape[0]), min(nstate, wl.B.shape[0])
    t0 = time.perf_counter()
    orc.grad_J(mol, wl.D[:nsJ], wl.c_aux[:nsJ], prim_cutoff=cut, aux=aux)
    tJ = time.perf_counter()
    orc.grad_K(mol, wl.C_occ, wl.C_vir, wl.B[:nsK], prim_cutoff=cut, aux=aux)
    tK = time.perf_counter()
    for P in aux:                       # the Gamma^P assembly step of grad_K once more, by itself
        for st in range(nsK):
            orc.gamma_P(wl.C_occ, wl.C_vir, wl.B[st, P])
    tG = time.perf_counter()
    orc.grad_PQ(mol, wl.c_aux[:nsJ], wl.d_aux[:nsJ])
    tQ = time.perf_counter()
    frac = len(aux) / mol.natoms
    sJ, sK, sG, sQ = tJ - t0, tK - tJ, tG - tK, tQ - tG
    ms_state = (sJ / nsJ / frac + sK / nsK / frac + sQ / nsJ) * 1e3
    full = frac >= 1.0 and nsJ == wl.D.shape[0] and nsK == wl.B.shape[0]
    desc = (("the whole workload, all aux functions and states" if full else
             f"aux P in [0,{len(aux)}) of {mol.natoms}, {nsJ} J / {nsK} K state(s) of the batch") +
            f": oracle grad_J {sJ:.2f}s + grad_K {sK:.2f}s (of which numpy Gamma^P assembly {sG:.2f}s, integral "
            f"contraction {max(sK - sG, 0.0):.2f}s), PQ in full {sQ:.3f}s"
            + ("" if full else f"; ms/state extrapolated x{1 / frac:.1f} in naux")
            + (f"; oracle primitive cutoff {cut:g}" if cut else ""))
    return {"seconds": sJ + sK + sQ, "ms_state": ms_state, "threads": orc.num_threads(), "desc": desc,
            "extrapolated": not full, "factor": round(1.0 / frac, 2),
            "parts_s": {"J": round(sJ, 3), "K_total": round(sK, 3), "K_gamma_assembly": round(sG, 3),
                        "K_integrals": round(max(sK - sG, 0.0), 3), "PQ": round(sQ, 4)}}


def auto_oracle_aux(wl) -> int:
    # about 10-30 s of CPU work on 16 threads: cost per aux ~ ordered primitive pairs + Gamma^P matmul
    est = {1: 3, 2: 30, 3: 12, 4: 40, 5: 6}
    return est.get(wl.meta.get("config", 0), 4)


def cpu_baseline_block(wl, cfg: int, n_aux: int, full: bool):
    """The `cpu_baseline` object of the JSON line.  full: the oracle over the whole workload (configs 1-3, 5: nothing
    extrapolated; `--cpu-baseline-full`), plus its single-thread time on configs 1-2 (whole) / 3 (a sample)."""
    nst = max(wl.D.shape[0], wl.B.shape[0]) if full else 1
    r = oracle_sample_time(wl, cfg, wl.mol.natoms if full else n_aux, nst)
    blk = {"value": round(r["ms_state"], 2), "unit": UNIT, "cores": r["threads"], "cpu_model": cpu_model(), "kind": "oracle",
           "sample": r["desc"], "sample_seconds": round(r["seconds"], 2), "extrapolated": r["extrapolated"],
           "extrapolation_factor": r["factor"] if r["extrapolated"] else 1.0, "parts_s": r["parts_s"]}
    if full and cfg in (1, 2, 3):
        nthr = r["threads"]
        set_oracle_threads(1)
        try:
            r1 = oracle_sample_time(wl, cfg, wl.mol.natoms if cfg < 3 else 2, nst if cfg < 3 else 1)
        finally:
            set_oracle_threads(nthr)
        blk["single_thread"] = {"value": round(r1["ms_state"], 2), "unit": UNIT, "sample": r1["desc"],
                                "extrapolated": r1["extrapolated"], "parts_s": r1["parts_s"]}
    return blk


# ------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2511_18233_b200 import probe_fp64_peak, ris_setup, synth
    from paper_2511_18233_b200.ris import probe_fp64_mma_peak
    counters = ncu_counters(args.config)

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the ris library has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    wl = synth.make_workload(args.config)
    mol = wl.mol
    nbJ, nbK = wl.D.shape[0], wl.B.shape[0]
    nstates = max(nbJ, nbK)

    t0 = time.perf_counter()
    ctx = ris_setup(mol, schwarz_tol=wl.schwarz_tol, profile=True)
    torch.cuda.synchronize()
    setup_first_ms = (time.perf_counter() - t0) * 1e3      # includes CUDA context creation and module load
    setup_ms = float("inf")                                # what a new geometry costs in a running process (best of 3)
    for _ in range(3):
        ctx.close()
        t0 = time.perf_counter()
        ctx = ris_setup(mol, schwarz_tol=wl.schwarz_tol, profile=True)
        torch.cuda.synchronize()
        setup_ms = min(setup_ms, (time.perf_counter() - t0) * 1e3)

    sharded = world > 1 and args.shard == "aux"
    host = {k: torch.from_numpy(np.ascontiguousarray(getattr(wl, k))).pin_memory()
            for k in ("D", "c_aux", "d_aux", "C_occ", "C_vir")}
    if sharded:
        from paper_2511_18233_b200 import shard
        my_aux = shard.aux_range(ctx.naux, rank, world)
        host["B"] = torch.from_numpy(np.ascontiguousarray(wl.B[:, my_aux.start:my_aux.stop])).pin_memory()   # this rank's slice only
        gJK = torch.empty((nbJ + nbK, mol.natoms, 3), dtype=torch.float64, device=dev)
    else:
        host["B"] = torch.from_numpy(np.ascontiguousarray(wl.B)).pin_memory()
    d = {k: v.to(dev, non_blocking=True) for k, v in host.items()}
    gJ = torch.empty((nbJ, mol.natoms, 3), dtype=torch.float64, device=dev)
    gK = torch.empty((nbK, mol.natoms, 3), dtype=torch.float64, device=dev)
    gQ = torch.empty((nbJ, mol.natoms, 3), dtype=torch.float64, device=dev)
    torch.cuda.synchronize()

    marks = []                              # per step: events before J, after J, after K, after PQ (same stream)

    def step(timed=False):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)] if timed else None
        if timed:
            ev[0].record()
        if sharded:         # J and K shares + the all-reduce (charged to the K interval below)
            if timed:
                ev[1].record()
            shard.grad_JK_sharded(ctx, d["D"], d["c_aux"], d["C_occ"], d["C_vir"], d["B"], out=gJK)
        else:
            ctx.grad_J(d["D"], d["c_aux"], out=gJ)
            if timed:
                ev[1].record()
            ctx.grad_K(d["C_occ"], d["C_vir"], d["B"], out=gK)
        if timed:
            ev[2].record()
        ctx.grad_PQ(d["c_aux"], d["d_aux"], out=gQ)
        if timed:
            ev[3].record()
            marks.append(ev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    fp64_peak = probe_fp64_peak()            # DFMA chains, TFLOP/s (MEASURED_PEAKS.json has no FP64 figure)
    mma_peak = probe_fp64_mma_peak()         # mma.sync f64 chains, TFLOP/s

    # The timed region runs WITHOUT the library's per-launch events (two event records per launch are a tenth of a
    # small molecule's step); the per-kernel table comes from a second, profiled pass of the same steps below.
    ctx.profile_enable(False)
    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step(timed=True)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    ctx.profile_enable(True)
    step()
    barrier()
    ctx.profile_reset()
    for _ in range(args.steps):
        step()
    barrier()
    prof = ctx.profile()
    ctx.profile_enable(False)                # the end-to-end loop below is timed without it as well
    ms_J = sum(ev[0].elapsed_time(ev[1]) for ev in marks)
    ms_K = sum(ev[1].elapsed_time(ev[2]) for ev in marks)
    ms_Q = sum(ev[2].elapsed_time(ev[3]) for ev in marks)
    if world > 1:
        t = torch.tensor([ms_total, ms_J, ms_K, ms_Q], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total, ms_J, ms_K, ms_Q = (float(x) for x in t.tolist())
    ms_step = ms_total / args.steps
    # ms per state: every term divided by ITS OWN number of states (config 2 runs 2 J/PQ states and 1 K state); the
    # remainder of the step (launch gaps between the calls) is charged to the larger batch.  Equal batches: ms_step/nbatch.
    gap = max(ms_total - (ms_J + ms_K + ms_Q), 0.0)
    value = (ms_J / nbJ + ms_K / nbK + ms_Q / nbJ + gap / nstates) / args.steps / (1 if sharded else world)
    per_term = {"J_ms_per_state": round(ms_J / nbJ / args.steps, 4), "K_ms_per_state": round(ms_K / nbK / args.steps, 4),
                "PQ_ms_per_state": round(ms_Q / nbJ / args.steps, 4), "nbatch_J": nbJ, "nbatch_K": nbK}
    if sharded:
        per_term["note"] = "aux-sharded: K_ms_per_state holds this step's J share + K share + the all-reduce (max over ranks)"

    # ---- per-kernel accounting from the CUDA events the library records around every launch (same stream)
    groups = {}
    for name, ms, fl, by in prof:
        g = groups.setdefault(name, {"launches": 0, "ms": 0.0, "flops": 0.0, "bytes": 0.0})
        g["launches"] += 1; g["ms"] += ms; g["flops"] += fl; g["bytes"] += by
    ksum = sum(g["ms"] for g in groups.values())
    dom_name = max(groups, key=lambda k: groups[k]["ms"])
    dom = groups[dom_name]
    is_gemm = dom_name.startswith("ris_gemm")
    peak = mma_peak if is_gemm else fp64_peak
    achieved = dom["flops"] / (dom["ms"] * 1e-3) * 1e-12 if dom["ms"] > 0 else 0.0
    roofline = {"kernel": dom_name, "bound": "tensor" if is_gemm else "alu", "achieved": round(achieved, 3),
                "peak": round(peak, 3), "unit": "TFLOP/s", "frac": round(achieved / peak, 4) if peak else None,
                "traffic": counters.get(dom_name, {}).get("dram_bytes_per_launch"), "launches": dom["launches"],
                "avg_launch_ms": round(dom["ms"] / dom["launches"], 4),
                "share_of_kernel_time": round(dom["ms"] / ksum, 4),
                "kernel_times_overlap": bool(ctx.p_batch >= 0 and mol.natoms <= 64),   # small molecules: class kernels run side by side
                "traffic_unit": "bytes per launch, dram__bytes_read.sum + dram__bytes_write.sum; source: "
                                + str(counters.get(dom_name, {}).get("source", "no committed ncu capture of this (config, kernel)")),
                "algorithmic_bytes_per_launch": round(dom["bytes"] / dom["launches"]),
                "peak_source": ("measured in this run by ris_probe_fp64_mma_peak (mma.sync f64 chains)" if is_gemm else
                                "measured in this run by ris_probe_fp64_peak (independent DFMA chains)")
                               + "; MEASURED_PEAKS.json carries no FP64 figure"}
    cls = [g for n, g in groups.items() if n.startswith("ris_grad_kernel")]
    cls_ms = sum(g["ms"] for g in cls)
    cls_fl = sum(g["flops"] for g in cls)
    ncalls = 2 * args.steps                      # J and K each run the class kernels over all triplets
    integrals = {"tflops_model": round(cls_fl / (cls_ms * 1e-3) * 1e-12, 3) if cls_ms else None,
                 "frac_model": round(cls_fl / (cls_ms * 1e-3) * 1e-12 / fp64_peak, 4) if cls_ms else None,
                 "frac_model_note": "textbook operation model of SURVEY.md 8(d) / live time; NOT the ncu instruction count",
                 "frac_ncu": counters.get("integral_kernels"),
                 "fp64_peak_tflops": round(fp64_peak, 2), "ms_per_step": round(cls_ms / args.steps, 4),
                 "triplets_per_s": round(ctx.ntriplets * ncalls / (cls_ms * 1e-3), 1) if cls_ms else None,
                 "ntriplets": ctx.ntriplets, "ntriplets_unscreened": ctx.ntriplets_unscreened}
    gemm_ms = sum(g["ms"] for n, g in groups.items() if n.startswith("ris_gemm"))
    gemm_fl = sum(g["flops"] for n, g in groups.items() if n.startswith("ris_gemm"))
    kernels = {n: {"launches": g["launches"], "ms_per_step": round(g["ms"] / args.steps, 4),
                   "tflops": round(g["flops"] / (g["ms"] * 1e-3) * 1e-12, 3) if g["ms"] > 0 else None,
                   "gbs": round(g["bytes"] / (g["ms"] * 1e-3) * 1e-9, 1) if g["ms"] > 0 else None}
               for n, g in sorted(groups.items(), key=lambda kv: -kv[1]["ms"])}

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D + kernels + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        hJ = np.empty((nbJ, mol.natoms, 3)); hK = np.empty((nbK, mol.natoms, 3)); hQ = np.empty((nbJ, mol.natoms, 3))

        def step_host():
            if sharded:     # this rank's inputs up, its shares + the all-reduce, the gradients down
                t = {k: v.to(dev, non_blocking=True) for k, v in host.items()}
                a, b = shard.grad_JK_sharded(ctx, t["D"], t["c_aux"], t["C_occ"], t["C_vir"], t["B"], out=gJK)
                q = ctx.grad_PQ(t["c_aux"], t["d_aux"], out=gQ)
                hJ[...] = a.cpu().numpy(); hK[...] = b.cpu().numpy(); hQ[...] = q.cpu().numpy()
            else:
                ctx.grad_host(host["D"], host["c_aux"], host["d_aux"], host["C_occ"], host["C_vir"], host["B"], out=(hJ, hK, hQ))

        for _ in range(max(1, min(args.warmup, 3))):    # (small molecules: the J part is captured into a CUDA graph on its second call)
            step_host()
        barrier()
        n_e2e = max(1, min(args.steps, 5 if ms_step > 20.0 else 50))      # sub-millisecond steps: more repetitions (host jitter)
        reps = []
        for _ in range(n_e2e):
            t0 = time.perf_counter()
            step_host()
            torch.cuda.synchronize()
            reps.append((time.perf_counter() - t0) * 1e3)
        t_e2e = sum(reps) / n_e2e
        if world > 1:
            t = torch.tensor([t_e2e], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            t_e2e = float(t.item())
        # the end-to-end result is the resident-input result (same kernels, other copy schedule)
        if sharded:
            gJ, gK = gJK[:nbJ], gJK[nbJ:]
        e2e_err = max(float(np.abs(h - g.cpu().numpy()).max() / max(1e-300, float(g.abs().max())))
                      for h, g in ((hJ, gJ), (hK, gK), (hQ, gQ)))
        if not e2e_err <= 5e-14:
            raise SystemExit(f"bench.py: ris_grad_host deviates from the resident-input path by {e2e_err:.3g} of the scale")
        h2d = 8 * (host["D"].numel() + host["c_aux"].numel() + host["d_aux"].numel() + host["C_occ"].numel()
                   + host["C_vir"].numel() + host["B"].numel())
        d2h = 8 * (hJ.size + hK.size + hQ.size)
        e2e = {"value": round(t_e2e / ((1 if sharded else world) * nstates), 4), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": n_e2e, "e2e_checked": True, "e2e_max_dev_of_scale": e2e_err, "ms_per_step_each": [round(r, 2) for r in reps],
               "median_ms_per_state": round(sorted(reps)[len(reps) // 2] / ((1 if sharded else world) * nstates), 4),
               "how": ("aux-sharded: per rank, its inputs (B[:, P_r] only) from pinned host memory, ris_grad_J_range + ris_grad_K_range, "
                       "the NCCL all-reduce, ris_grad_PQ, gradients back to the host; host wall clock, max over ranks; bytes are per rank") if sharded else
                      ("ris_grad_host (J + K + PQ in one call) on pinned host buffers; host wall clock around the call, which returns "
                       "after the D2H copy of the gradients; B goes up in P chunks on a copy stream under the J kernels and the GEMMs")}

    fit = None
    if not args.no_extras and not sharded:
        # ---- NEXT-1 (reported beside the metric, outside the timed step): the J-type fitting step on the same workload
        ctx.fit_J(d["D"])                                       # builds the metric's Cholesky factor (one-off per geometry)
        torch.cuda.synchronize()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record()
        for _ in range(3):
            ctx.fit_J(d["D"])
        f1.record()
        torch.cuda.synchronize()
        fit = {"ris_fit_J_ms_per_state": round(f0.elapsed_time(f1) / 3 / nbJ, 4), "nbatch": nbJ,
               "what": "v_P = sum D (mu nu|P) on the undifferentiated class kernels + Cholesky solve c = M^-1 v"}
        ctx.fit_K(d["C_occ"], d["C_vir"])                       # builds M^-1, sizes the scratch
        torch.cuda.synchronize()
        ctx.profile_reset()
        f0.record()
        ctx.fit_K(d["C_occ"], d["C_vir"])
        f1.record()
        torch.cuda.synchronize()
        fit["ris_fit_K_ms"] = round(f0.elapsed_time(f1), 3)
        fit["ris_fit_K_kernels"] = {}
        for name, ms, fl, by in ctx.profile():
            g = fit["ris_fit_K_kernels"].setdefault(name, {"ms": 0.0, "tflops": 0.0})
            g["ms"] = round(g["ms"] + ms, 3); g["tflops"] += fl
        for g in fit["ris_fit_K_kernels"].values():
            g["tflops"] = round(g["tflops"] / (g["ms"] * 1e-3) * 1e-12, 2) if g["ms"] > 0 else None

    # ---- NEXT-3 / NEXT-4c (reported beside the metric): the ris coupling-matrix products for a block of 8 trial vectors
    resp = None
    try:
        if args.no_extras or sharded:
            raise StopIteration
        torch.cuda.synchronize()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        ctx.resp_setup(d["C_occ"], d["C_vir"])
        r1.record()
        torch.cuda.synchronize()
        resp = {"ris_resp_setup_ms": round(r0.elapsed_time(r1), 2), "nvec": 8,
                "what": "sigma = sum_jb [cJ (ia|jb) - cKA (ij|ab) - cKB (ib|ja)]^ris X_jb, 8 vectors per call"}
        Xv = torch.randn((8, wl.nocc, wl.nvir), dtype=torch.float64, device=dev, generator=torch.Generator(device=dev).manual_seed(7))
        sg = torch.empty_like(Xv)
        for label, coef in (("tda_A_ms", (2.0, 0.25, 0.0)), ("z_vector_ApB_ms", (4.0, 0.25, 0.25))):
            ctx.resp_matvec(Xv, *coef, out=sg)
            torch.cuda.synchronize()
            ctx.profile_reset()
            r0.record()
            for _ in range(3):
                ctx.resp_matvec(Xv, *coef, out=sg)
            r1.record()
            torch.cuda.synchronize()
            resp[label] = round(r0.elapsed_time(r1) / 3, 3)
            kk = {}
            for name, ms, fl, by in ctx.profile():
                g = kk.setdefault(name, {"ms": 0.0, "tflops": 0.0, "gbs": 0.0})
                g["ms"] += ms / 3; g["tflops"] += fl / 3; g["gbs"] += by / 3
            for g in kk.values():
                t = g["ms"] * 1e-3
                g["tflops"] = round(g["tflops"] / t * 1e-12, 2) if t > 0 else None
                g["gbs"] = round(g["gbs"] / t * 1e-9, 1) if t > 0 else None
                g["ms"] = round(g["ms"], 3)
            resp[label.replace("_ms", "_kernels")] = kk
            gm = [g for n, g in kk.items() if n.startswith("ris_gemm")]
            if gm:
                tot = sum(g["ms"] for g in gm)
                resp[label.replace("_ms", "_gemm_frac_of_dmma_peak")] = round(sum(g["tflops"] * g["ms"] for g in gm) / tot / mma_peak, 4)
        ctx.resp_free()
    except StopIteration:
        resp = None
    except Exception as exc:                  # the block is an extra: a failure here must not lose the metric line
        resp = {"error": repr(exc)}

    line = {
        "metric": METRIC, "value": round(value, 4), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round(ms_step, 4), "higher_is_better": False,
        "scaling": "strong" if sharded else "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "natoms": mol.natoms, "nao": mol.nao, "naux": mol.natoms, "nocc": wl.nocc,
                   "nvir": wl.nvir, "nbatch_J": nbJ, "nbatch_K": nbK, "schwarz_tol": wl.schwarz_tol,
                   "p_batch": ctx.p_batch, "l2": "inputs larger than L2 (B alone is %.2f GB)" % (host["B"].numel() * 8e-9)
                   if host["B"].numel() * 8 > 200e6 else "inputs smaller than L2; no flush (latency-bound case)",
                   "step": "ris_grad_J + ris_grad_K + ris_grad_PQ, all states; ris_setup excluded (one-off per geometry)",
                   "parallelism": ("aux%d: one batch of states, aux index split over %d ranks, one all-reduce" % (world, world)) if sharded
                                  else ("replicas%d: every rank its own batch of states" % world if world > 1 else "single GPU")},
        "per_term": per_term,
        "setup_ms": round(setup_ms, 2), "setup_first_ms": round(setup_first_ms, 2), "e2e": e2e, "gpu_launches": len(prof),
        "roofline": roofline, "integral_kernels": integrals,
        "gamma_gemm": {"ms_per_step": round(gemm_ms / args.steps, 4),
                       "tflops": round(gemm_fl / (gemm_ms * 1e-3) * 1e-12, 3) if gemm_ms else None,
                       "fp64_mma_peak_tflops": round(mma_peak, 2)},
        "kernels": kernels, "fit_step": fit, "resp_step": resp, "clocks": clocks,
    }
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            n_aux = args.oracle_aux or auto_oracle_aux(wl)
            line["cpu_baseline"] = cpu_baseline_block(wl, args.config, n_aux, args.cpu_baseline_full)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """The oracle, as it stands, on the host cores (rank 0 only).  Exactly `--warmup` untimed and `--steps` timed steps;
    each step = one bounded sample of the workload (a few aux functions of one state; the whole workload on configs 1-2),
    so that the run ends within minutes.  `ms_per_step` is the MEASURED time of one such step; `value` is ms/state of the
    whole workload, extrapolated linearly in naux from the sample (`cpu_baseline.extrapolated`, `.extrapolation_factor`)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2511_18233_b200 import synth        # input generator only (no arithmetic of the method)
    wl = synth.make_workload(args.config)
    n_aux = args.oracle_aux or {1: 3, 2: 30, 3: 3, 4: 6, 5: 2}[args.config]
    for _ in range(max(0, args.warmup)):
        oracle_sample_time(wl, args.config, n_aux)
    vals, secs, r = [], [], None
    steps = max(1, args.steps)
    for _ in range(steps):
        r = oracle_sample_time(wl, args.config, n_aux)
        vals.append(r["ms_state"]); secs.append(r["seconds"])
    v = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": round(v, 2), "unit": UNIT,
            "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": steps, "warmup": max(0, args.warmup),
            "ms_per_step": round(float(np.mean(secs)) * 1e3, 2), "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "natoms": wl.mol.natoms, "nao": wl.mol.nao, "nocc": wl.nocc, "nvir": wl.nvir,
                       "step": "one bounded sample of the workload (see cpu_baseline.sample); ms_per_step is its measured time"},
            "cpu_baseline": {"value": round(v, 2), "unit": UNIT, "cores": r["threads"], "cpu_model": cpu_model(), "kind": "oracle",
                             "sample": r["desc"], "sample_seconds": round(float(np.mean(secs)), 2),
                             "extrapolated": r["extrapolated"], "extrapolation_factor": r["factor"] if r["extrapolated"] else 1.0,
                             "parts_s": r["parts_s"]},
            "e2e": {"value": round(v, 2), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
