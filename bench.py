#!/usr/bin/env python
"""bench.py -- fp64 DOF-updates/s per RK stage of the DG-SWEM hot path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--repeats R] [--workload C3|C1|C2p1|C2p2|C2p3|C4|C5|C5p3|H[+perturbed]]
                  [--dtype f64|f32] [--also LIST|none] [--impl ours|reference]

A "step" is one full explicit time step of the workload: WIND (if on) and, per RK stage, EDGE ->
GATHER+AREA+RK(+wet/dry) -> (limiter+wet/dry), i.e. every row of SURVEY.md section 8(a).  Default
workload: C3, the largest p=1 mesh (4,494,002 elements; BASELINE.json configs[2], the one the
north_star quotes the roofline target on).  value = 3*ndof*N_e*n_stage*K / t (DOF-updates/s per RK
stage), t = CUDA-event time of K steps on the stream the kernels run on, state resident in HBM: the MEDIAN of R = 5
such runs, the state re-set and W warm-up steps before each; min / max under `repeats`.  After the
headline the default run also times, briefly and in the same process, the storm-surge configurations from their recipe
states and from perturbed states (where the limiter pass has work everywhere) and the paper-size mesh in binary32; those
go under the `also` key and do not touch the headline's keys.
N > 1: independent replicas of the same workload, one per GPU ("replicas only"), weak
scaling, max over ranks.  --impl reference times the CPU oracle on the host cores.
Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import numpy as np  # noqa: E402

METRIC = "fp64 DOF-updates/sec per RK stage"          # BASELINE.json metric; with --dtype f32 the line says fp32
UNIT = "DOF-updates/s"


_LAST_BASE: dict = {}


def make_workload(name: str, scale: float = 1.0):
    """Workload by name; NAME+perturbed = the same recipe started from a non-smooth state (seeded waves + noise in every
    mode, workloads.perturbed): the limiter + wet/dry pass writes only what it changes, so on the BASELINE recipes'
    almost-at-rest states (C4, C5) it is timed at its best case; the perturbed start makes it limit nearly everywhere.
    The last base workload is kept, so that X followed by X+perturbed builds the mesh once."""
    if name.endswith("+perturbed"):
        from workloads import perturbed
        return perturbed(make_workload(name[:-len("+perturbed")], scale), amp_z=0.2)
    if _LAST_BASE.get("key") != (name, scale):
        _LAST_BASE.update(key=(name, scale), w=_build_workload(name, scale))
    return _LAST_BASE["w"]


def _build_workload(name: str, scale: float):
    from workloads import c1, c2, c3, c4, c5
    if name == "C3":
        nn = max(20, int(round(1500 * scale)))
        return c3(nn=nn)
    if name == "H":
        # the paper's Harvey / TX2008 mesh size (6,675,517 elements) on the C3 recipe: 2 x 1827^2 = 6,675,858
        return c3(nn=max(20, int(round(1828 * scale))))
    if name == "C1":
        return c1()
    if name == "C2p1":
        return c2(nq=max(8, int(512 * scale)), p=1)
    if name == "C2p2":
        return c2(nq=max(8, int(512 * scale)), p=2)
    if name == "C2p3":
        return c2(nq=max(8, int(512 * scale)), p=3)
    if name == "C5p3":      # the C5 mesh and recipe at p = 3
        return c5(nn=max(20, int(round(1323 * scale))), p=3)
    if name == "C4":
        return c4(nqx=max(16, int(1024 * scale)), nqy=max(8, int(512 * scale)))
    if name == "C5":
        return c5(nn=max(20, int(round(1323 * scale))))
    raise SystemExit(f"unknown workload {name}")


# ---------------------------------------------------------------------------------------------
# algorithmic bytes: what the two-kernel design must move per launch, every
# array counted once (unique-read assumption: each element's state is read once by EDGE although
# three edges use it; each flux value once by the element kernel although two elements use it).
def alg_bytes(w, kind: str, stage_first: bool, fused: bool = False, rb: int = 8) -> float:
    """rb = bytes per value of the working precision (8: fp64, 4: fp32); index tables are int32, masks bytes."""
    ne, nd = w.mesh.n_elem, w.mesh.n_edge
    nn = w.mesh.n_nodes
    ndof, nqe = w.ndof, w.params["p"] + 1
    lim, wd, wind = w.params["limiter"], w.params["wetdry"], w.holland is not None
    st = 3 * ndof * rb
    if kind == "edge":
        return nd * (8 + 4 + 2 * rb + 2 * rb + 3 * nqe * rb) + ne * st
    if kind == "elem" and fused:
        # element-centric stage kernel (A1-A5, A7): state once (the neighbours' rows are other elements' own
        # rows: unique-read assumption), neighbour table 12, normals 48, L/A 24, Jacobian 32, vertex bathymetry
        # 24, wet flag 1, new state; no flux buffer, no edge records
        b = ne * (st + 12 + 6 * rb + 3 * rb + 4 * rb + 3 * rb + 1 + st)
        if not stage_first:
            b += ne * st
        if wd and not lim:
            b += ne * 1
        if lim:
            b += ne * 3 * rb
        if wind:
            b += ne * 12 + nn * 2 * rb
        return b
    if kind == "elem":
        b = nd * 3 * nqe * rb + ne * (st + 12 + 3 * rb + 4 * rb + 3 * rb + 1 + st)
        if not stage_first:
            b += ne * st
        if wd and not lim:
            b += ne * 1
        if lim:
            b += ne * 3 * rb
        if wind:
            b += ne * 12 + nn * 2 * rb
        return b
    if kind == "limwd":
        # what a write-if-changed pass must READ: the state rows the two steps look at (p = 2: not the quadratic momentum
        # modes), neighbour table, the neighbours' means (once per element), vertex bathymetry, wet flag.  What it writes
        # depends on the data (only values a step changed) and is NOT credited: the fraction is a lower bound.
        rows = 9 if w.params["p"] == 1 else w.ndof + 6
        return ne * (rows * rb + 12 + 3 * rb + 3 * rb + 1)
    if kind == "wind":
        return nn * 4 * rb
    raise ValueError(kind)


def stage_bytes_total(w, fused: bool = False, rb: int = 8) -> float:
    """Algorithmic bytes of one whole time step (all stages)."""
    tot = alg_bytes(w, "wind", True, rb=rb) if w.holland is not None else 0.0
    for s in range(w.n_stage):
        tot += (0.0 if fused else alg_bytes(w, "edge", s == 0, rb=rb)) + alg_bytes(w, "elem", s == 0, fused, rb=rb)
        if w.params["limiter"]:
            tot += alg_bytes(w, "limwd", s == 0, rb=rb)
    return tot


def read_traffic():
    """profiles/traffic.csv: per (workload, kernel) the DRAM bytes per launch and, where the capture has it, the FP64
    instructions per element (smsp__inst_executed_pipe_fp64 x 32 / elements... stored per element), each with the prefix
    of the ncu summary under profiles/ it was read from.  A committed measurement, not live."""
    out = {}
    f = ROOT / "profiles" / "traffic.csv"
    if not f.exists():
        return out
    for ln in f.read_text().splitlines()[1:]:
        c = [x.strip() for x in ln.split(",")]
        if len(c) < 4 or not c[0]:
            continue
        out[(c[0], c[1])] = {"dram_bytes": float(c[2]) if c[2] else None, "source": c[3],
                             "fp64_inst_per_elem": float(c[4]) if len(c) > 4 and c[4] else None}
    return out


def plain_stages(w) -> int:
    """Stages of the Shu-Osher form that do not read w^n (a_s = 0, b_s = 1; R-2, R-19): the first stage of
    SSP(2,2) and SSP(3,3); all but the last of SSP(s,2); all but the third of SSP(4,3)."""
    return 1 if w.n_stage == w.params["rk_order"] else w.n_stage - 1


def fp64_roof(w, wname, fused, dom, avg_ms, dfma_rate, traffic):
    """Second roof of the dominant kernel: its FP64 instruction count (from the committed ncu capture named in `source`)
    against the DFMA rate the library's probe measures on this device in this run."""
    key = (wname, "stage" if (fused and dom == "elem") else dom)
    out = {"dfma_per_s_measured": dfma_rate, "tflops_measured": 2.0 * dfma_rate / 1e12,
           "how": "dgswem_fp64_peak: 8 dependent-DFMA chains per thread, 8 x 256 threads per SM, best of 3 launches"}
    rec = traffic.get(key)
    n = rec and rec["fp64_inst_per_elem"]
    if n and dfma_rate > 0:
        floor_ms = n * w.mesh.n_elem / dfma_rate * 1e3
        out.update({"fp64_inst_per_element": n, "floor_ms": floor_ms, "frac": floor_ms / avg_ms,
                    "source": f"profiles/{rec['source']}_*: thread-level FP64-pipe instructions per launch / elements (profiles/traffic.csv)"})
    return out


def load_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        d = json.loads(f.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------
# N > 1: independent replicas (the path does not shard in this build), no collective on the
# data path; the ranks only agree on the slowest replica's time.
def max_over_ranks(x: float, world: int, device) -> float:
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def whole_job_value(world: int, dofs_stage: int, steps: int, seconds: float) -> float:
    """DOF-updates/s of the whole job: every replica advances `steps` steps in `seconds` (max over ranks)."""
    return world * dofs_stage * steps / seconds


def workload_config(w) -> dict:
    """What names the workload: the SAME dict on both arms (the driver compares them); how an arm ran it is in `run`."""
    return {"workload": w.name, "n_elem": w.mesh.n_elem, "n_edge": w.mesh.n_edge, "n_nodes": w.mesh.n_nodes, "p": w.params["p"],
            "rk_order": w.params["rk_order"], "dt": w.dt, "limiter": w.params["limiter"], "wetdry": w.params["wetdry"],
            "flux": w.params.get("flux", 0), "wind": w.holland is not None, "tide": w.tide is not None,
            # timing hygiene: no L2 flush between iterations where one stage buffer alone exceeds the 126 MB L2
            "l2": "inputs larger than L2 (no flush)" if 3 * w.ndof * w.mesh.n_elem * 8 > 130e6 else "working set fits L2, not flushed between steps"}


def run_reference(args, rank: int):
    """The CPU oracle, as it stands, on the host cores (bench contract: reference arm)."""
    if rank != 0:
        return
    if args.dtype == "f32":
        from oracle import oracle32 as orc
    else:
        from oracle import oracle as orc
    orc.build()
    total = args.steps + args.warmup
    # bounded sample: the full mesh if the run stays within a few minutes, else a smaller mesh of the same recipe
    est_full = 2.4 * total + 20.0           # s: about 1.2 s per RK stage at 4.5 M elements on 8 cores
    scale = 1.0 if (args.workload != "C3" or est_full < 150.0) else max(0.1, (150.0 / est_full) ** 0.5)
    w = make_workload(args.workload, scale)
    o = orc.Oracle.from_workload(w)
    o.step(args.warmup, w.dt)
    t0 = time.perf_counter()
    o.step(args.steps, w.dt)
    dt = time.perf_counter() - t0
    value = w.dofs * w.n_stage * args.steps / dt
    sample = f"{w.name}: {w.mesh.n_elem} elements, {args.steps} steps after {args.warmup} warm-up"
    cfg = workload_config(w if scale == 1.0 else make_workload(args.workload))     # the arm's config names the full workload
    line = {"impl": "reference", "metric": METRIC.replace("fp64", "fp32") if args.dtype == "f32" else METRIC, "value": value, "unit": UNIT,
            "n_gpus": int(os.environ.get("WORLD_SIZE", args.gpus)), "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": cfg,
            "run": {"kind": "CPU oracle (oracle/dgswem_oracle.c, gcc -O2 -ffp-contract=off, OpenMP)", "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_decomp(args, rank: int, world: int, local_rank: int):
    """--decomp P: ONE mesh split into partitions with halo exchange every RK stage (strong scaling).
    world == 1: P partitions on this GPU (LocalTransport; measures the cost of the decomposition machinery itself).
    world > 1: one partition per rank, NCCL isend/irecv of the packed halos on the communication stream, overlapped with
    the interior elements by default (the one-graph-per-step form is LocalTransport only; not measurable on this one-GPU box)."""
    import torch
    import torch.distributed as dist
    from paper_2508_21208_b200 import build as b
    if rank == 0:
        b.build()
    if world > 1:
        dist.barrier()
    from paper_2508_21208_b200.decomp import PartitionedDgswem, DistTransport
    torch.cuda.set_device(local_rank)
    w = make_workload(args.workload)
    m = w.mesh
    n_parts = world if world > 1 else max(1, args.decomp)
    pd = PartitionedDgswem.from_workload(w, n_parts, reorder=args.reorder, device=local_rank,
                                         parts=[rank] if world > 1 else None, transport=DistTransport() if world > 1 else None,
                                         overlap=None if args.decomp_overlap < 0 else bool(args.decomp_overlap),
                                         graph=bool(args.decomp_graph) and world == 1)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    pd.step(max(args.warmup, 3), w.dt)
    barrier()
    l0 = sum(g.launch_count() for g in pd.handles)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    pd.step(args.steps, w.dt)
    pd.join()                                   # the current stream waits for every partition's stream
    ev1.record()
    barrier()
    ms = max_over_ranks(ev0.elapsed_time(ev1), world, "cuda")
    launches = sum(g.launch_count() for g in pd.handles) - l0
    if pd.graph:
        # replays of the caller's graph are not seen by dgswem_launch_count: kernels recorded per step x steps replayed
        launches = pd.launches_per_graph_step * args.steps
    if rank != 0:
        return
    value = w.dofs * w.n_stage * args.steps / (ms * 1e-3)      # the whole (single) mesh, whatever the number of ranks
    ghosts = sum(s.n_local - s.n_owned for s in pd.subs)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": w.name, "n_elem": m.n_elem, "p": w.params["p"], "rk_order": w.params["rk_order"], "dt": w.dt,
                       "parallelism": f"domain decomposition: {n_parts} partitions on {world} GPU(s), halo exchange every RK stage",
                       "ghost_elements": int(ghosts), "overlap": bool(pd.overlap), "one_graph_per_step": bool(pd.graph), "transport": "NCCL isend/irecv" if world > 1 else "device copies (one GPU)"},
            "gpu_launches": int(launches), "e2e": None, "roofline": None, "cpu_baseline": None}
    print(json.dumps(line), flush=True)
    pd.close()


def timed_repeats(g, w, steps, warmup, repeats, barrier, hin):
    """`repeats` timed runs of exactly `steps` time steps, the state re-set (dgswem_set_state from the pinned
    host arrays, untimed) and `warmup` untimed steps before each; CUDA events on the stream the kernels are launched on.
    Returns the list of milliseconds and the kernel launches of one run."""
    import torch
    ms, launches = [], 0
    for _ in range(repeats):
        g.set_state(0.0, *hin)
        g.step(warmup, w.dt)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        l0 = g.launch_count()
        ev0.record(g.stream)
        g.step(steps, w.dt)       # dgswem_step replays its captured step graphs here (the production path: no per-launch events)
        ev1.record(g.stream)
        barrier()
        ms.append(ev0.elapsed_time(ev1))
        launches = g.launch_count() - l0
    return ms, launches


def profiled_pass(g, w, steps, barrier):
    """The same `steps` steps once more with the library's per-launch CUDA events on (plain stream launches, every kernel
    bracketed by two events on its stream): per-kernel durations for the roofline."""
    import torch
    g.profile(True)
    g.profile_read()
    evp0, evp1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    evp0.record(g.stream)
    g.step(steps, w.dt)
    evp1.record(g.stream)
    barrier()
    ms_prof = evp0.elapsed_time(evp1)
    prof = g.profile_read()
    g.profile(False)
    return prof, ms_prof


def kernel_table(w, wname, prof, ms_prof, fused, rb, peak, traffic):
    """Per kernel kind: launches, mean launch time, algorithmic bytes per launch (stages without / with the w^n read
    weighted by the scheme), achieved GB/s, share of the step, and the fraction of the peak by the DRAM bytes of the
    committed ncu capture where one exists (the honest numerator for the write-if-changed limiter pass)."""
    per_kind = {}
    for k, (tms, cnt) in prof.items():
        if not cnt:
            continue
        nfirst = cnt * plain_stages(w) // w.n_stage if k in ("edge", "elem", "limwd") else cnt
        byts = (alg_bytes(w, k, True, fused, rb) * nfirst + alg_bytes(w, k, False, fused, rb) * (cnt - nfirst)) / cnt
        per_kind[k] = {"launches": cnt, "avg_ms": tms / cnt, "alg_bytes_per_launch": byts,
                       "achieved_gbs": byts / (tms / cnt * 1e-3) / 1e9, "share_of_step": tms / ms_prof}
        rec = traffic.get((wname, "stage" if (fused and k == "elem") else k))
        if rec and rec["dram_bytes"]:
            per_kind[k]["ncu_dram_bytes_per_launch"] = rec["dram_bytes"]
            per_kind[k]["ncu_source"] = rec["source"]
            per_kind[k]["frac_of_peak_by_ncu_dram_bytes"] = rec["dram_bytes"] / (per_kind[k]["avg_ms"] * 1e-3) / 1e9 / peak
    return per_kind


def also_run(pk, name, dtype, args, local_rank, peak, traffic):
    """A short run of another workload in the same process (the `also` key: the storm-surge configurations and the
    paper's mesh size in its own precision next to the C3 / f64 headline): median of 3 repeats of 10 steps."""
    import torch
    w = make_workload(name)
    f32 = dtype == "f32"
    rb = 4 if f32 else 8
    g = pk.Dgswem.from_workload(w, reorder=args.reorder, device=local_rank, precision=32 if f32 else 64)
    fused = g.stage_form() >= 1
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    hin = [pin(w.ze), pin(w.qx), pin(w.qy)]
    steps = 10
    ms, launches = timed_repeats(g, w, steps, 3, 3, torch.cuda.synchronize, hin)
    med = float(np.median(ms))
    prof, ms_prof = profiled_pass(g, w, steps, torch.cuda.synchronize)
    wet = g.get_wetdry()
    g.close()
    kt = kernel_table(w, name + ("_f32" if f32 else ""), prof, ms_prof, fused, rb, peak, traffic)
    sb = stage_bytes_total(w, fused, rb)
    return {"workload": w.name, "dtype": dtype, "n_elem": w.mesh.n_elem, "p": w.params["p"], "rk_stages": w.n_stage,
            "limiter": w.params["limiter"], "wetdry": w.params["wetdry"], "wind": w.holland is not None,
            "value": w.dofs * w.n_stage * steps / (med * 1e-3), "unit": UNIT, "steps": steps, "repeats": len(ms),
            "ms_per_step": med / steps, "ms_per_step_min": min(ms) / steps, "ms_per_step_max": max(ms) / steps,
            "gpu_launches": int(launches), "dry_fraction": float(1.0 - wet.mean()),
            "whole_step_frac_of_measured_peak": sb / (med / steps * 1e-3) / 1e9 / peak,
            "kernels": {k: {kk: v[kk] for kk in ("launches", "avg_ms", "achieved_gbs", "share_of_step", "frac_of_peak_by_ncu_dram_bytes") if kk in v}
                        for k, v in kt.items()}}


def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    t_start = time.perf_counter()
    from paper_2508_21208_b200 import build as b
    if rank == 0:
        b.build()
    if world > 1:
        dist.barrier()
    import paper_2508_21208_b200 as pk
    torch.cuda.set_device(local_rank)
    w = make_workload(args.workload)
    f32 = args.dtype == "f32"
    rb = 4 if f32 else 8
    metric = METRIC.replace("fp64", "fp32") if f32 else METRIC
    g = pk.Dgswem.from_workload(w, reorder=args.reorder, device=local_rank, precision=32 if f32 else 64)
    dofs_stage = w.dofs * w.n_stage
    fused = g.stage_form() >= 1
    warm = max(args.warmup, 3)
    repeats = max(1, args.repeats)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    hin = [pin(w.ze), pin(w.qx), pin(w.qy)]
    hout = [pin(np.empty_like(w.ze)) for _ in range(3)]
    # ---- warm-up
    g.step(warm, w.dt)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    # ---- timed region: `repeats` runs of exactly K steps each, device-resident state, state re-set + warm-up before each
    ms_all, launches = timed_repeats(g, w, args.steps, warm, repeats, barrier, hin)
    prof, ms_prof = profiled_pass(g, w, args.steps, barrier)
    clocks = sampler.stop() if rank == 0 else None
    dfma_rate = g.fp64_peak() if rank == 0 else 0.0        # the device's measured DFMA rate: second roof of the stage kernel
    ms_all = [max_over_ranks(x, world, "cuda") for x in ms_all]     # every repeat: the slowest rank's time
    ms = float(np.median(ms_all))
    value = whole_job_value(world, dofs_stage, args.steps, ms * 1e-3)

    # ---- end to end through the C ABI with host buffers: set_state (H2D) + K steps + get_state/get_wetdry (D2H)
    g.set_state(0.0, *hin); g.step(1, w.dt); g.get_state(out=hout)      # warm the path
    barrier()
    t0 = time.perf_counter()
    g.set_state(0.0, *hin)
    g.step(args.steps, w.dt)
    g.get_state(out=hout)
    g.get_wetdry()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, world, "cuda")
    state_bytes = 3 * w.ndof * w.mesh.n_elem * 8          # the ABI's host arrays are binary64 in both precisions
    e2e = {"value": whole_job_value(world, dofs_stage, args.steps, e2e_s), "unit": UNIT,
           "h2d_bytes_per_step": state_bytes / args.steps, "d2h_bytes_per_step": (state_bytes + w.mesh.n_elem) / args.steps,
           "call": f"dgswem_set_state + dgswem_step({args.steps}) + dgswem_get_state + dgswem_get_wetdry, pinned host buffers, "
                   f"wall clock; bytes are the per-job copies divided by the {args.steps} steps"}
    stage_form = g.stage_form()
    g.close()
    if rank != 0:
        return

    # ---- roofline of the dominant kernel (per-launch CUDA-event times from inside the timed region)
    peak, peak_src = load_peaks()
    traffic = read_traffic()
    tkey = args.workload + ("_f32" if f32 else "")          # key into profiles/traffic.csv
    per_kind = kernel_table(w, tkey, prof, ms_prof, fused, rb, peak, traffic)
    dom = max(per_kind, key=lambda k: per_kind[k]["avg_ms"] * per_kind[k]["launches"])
    d = per_kind[dom]
    kname = "k_stage" if (fused and dom == "elem") else f"k_{dom}"
    sb = stage_bytes_total(w, fused, rb)
    # SURVEY.md section 8(d)'s figure for the flux-buffer design (591 B per element-stage at p = 1), for reference
    sb_survey = stage_bytes_total(w, False, rb)
    roofline = {"bound": "hbm", "kernel": f"{kname}<{w.params['p']}>", "achieved": d["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": d["achieved_gbs"] / peak, "traffic": d.get("ncu_dram_bytes_per_launch"), "traffic_source": d.get("ncu_source"),
                "peak_source": peak_src,
                "alg_bytes_per_launch": d["alg_bytes_per_launch"], "avg_launch_ms": d["avg_ms"], "kernels": per_kind,
                "fp64_roof": None if f32 else fp64_roof(w, tkey, fused, dom, d["avg_ms"], dfma_rate, traffic),
                "whole_step": {"alg_bytes": sb, "achieved_gbs": sb / (ms / args.steps * 1e-3) / 1e9,
                               "frac_of_measured_peak": sb / (ms / args.steps * 1e-3) / 1e9 / peak,
                               "frac_of_8TBs_nominal": sb / (ms / args.steps * 1e-3) / 1e9 / 8000.0,
                               "alg_bytes_flux_buffer_design": sb_survey,
                               "frac_of_measured_peak_at_flux_buffer_bytes": sb_survey / (ms / args.steps * 1e-3) / 1e9 / peak}}

    # ---- CPU baseline: the oracle on a bounded sample of the same workload, on this box's cores
    cpu = None
    if not args.no_cpu:
        if f32:
            from oracle import oracle32 as orc
        else:
            from oracle import oracle as orc
        orc.build()
        o = orc.Oracle.from_workload(w)
        nsamp = max(1, min(args.steps, int(round(45.0 / (w.mesh.n_elem * w.n_stage * 0.28e-6 + 1e-3)))))   # about 10-15 s on 16 cores
        o.step(1, w.dt)
        t0 = time.perf_counter()
        o.step(nsamp, w.dt)
        cs = time.perf_counter() - t0
        cpu = {"value": dofs_stage * nsamp / cs, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
               "sample": f"{nsamp} steps of {w.name} (full mesh, {w.mesh.n_elem} elements) after 1 warm-up step, {cs:.1f} s"}
        del o

    # ---- `also`: short runs of the storm-surge configurations and the paper-size mesh in fp32, same process, one GPU
    also = None
    if world == 1 and args.also and args.also != "none":
        also = {}
        for item in args.also.split(","):
            name, _, dt_ = item.partition(":")
            if time.perf_counter() - t_start > args.also_budget:
                also[item] = {"skipped": f"wall-clock budget of {args.also_budget:.0f} s for the whole run reached"}
                continue
            try:
                also[item] = also_run(pk, name, dt_ or "f64", args, local_rank, peak, traffic)
            except Exception as e:    # the headline line must still be printed
                also[item] = {"error": f"{type(e).__name__}: {e}"}

    line = {"metric": metric, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
            "ms_per_step": ms / args.steps, "ms_per_step_with_per_launch_events": ms_prof / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
            "data": "synthetic",
            "config": workload_config(w),
            "repeats": {"n": len(ms_all), "statistic": "median", "ms_per_step_min": min(ms_all) / args.steps, "ms_per_step_max": max(ms_all) / args.steps,
                        "value_min": whole_job_value(world, dofs_stage, args.steps, max(ms_all) * 1e-3),
                        "value_max": whole_job_value(world, dofs_stage, args.steps, min(ms_all) * 1e-3),
                        "protocol": f"state re-set (dgswem_set_state) and {warm} untimed steps before each of the {len(ms_all)} timed runs of {args.steps} steps (SURVEY.md 8(d))"},
            "run": {"reorder": args.reorder, "stage_form": ("element-centric stage kernel, TMA-staged operands (no flux buffer)" if stage_form == 3 else "element-centric stage kernel, shared-memory edge tile (no flux buffer)" if stage_form == 2 else "element-centric stage kernel (no flux buffer)") if fused
                    else "edge kernel + element kernel (flux buffer)", "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                    "l2": f"state {state_bytes // 8 * rb / 1e6:.0f} MB per buffer exceeds the 126 MB L2 (inputs larger than L2, no flush needed)"
                          if state_bytes // 8 * rb > 130e6 else "working set fits L2: a >L2 buffer is NOT flushed between steps; see DESIGN.md"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu, "also": also}
    print(json.dumps(line), flush=True)


def spawn_ranks(n: int) -> int:
    """Re-run this command line under torch.distributed.run with n ranks on this node; returns its exit code."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(Path(__file__).resolve()), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"], help="working precision of the path (f32: SURVEY 8(f) NEXT-2, "
                    "the paper's own precision; the driver's default line stays C3 / f64)")
    ap.add_argument("--reorder", type=int, default=1, help="internal renumbering: 0 none, 1 Hilbert curve (default), 2 reverse Cuthill-McKee")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--repeats", type=int, default=5, help="timed runs of --steps steps each; value = the median (SURVEY.md 8(d))")
    ap.add_argument("--also", default=None, help="comma list of workload[:dtype] run briefly after the headline and reported under "
                    "the `also` key; default for the default workload: C4,C4+perturbed,C5,C5+perturbed,H:f32; `none` = skip")
    ap.add_argument("--also-budget", type=float, default=170.0, help="no further `also` run is started once the whole run has taken this many seconds")
    ap.add_argument("--decomp", type=int, default=0, help="domain decomposition instead of replicas: one partition per rank "
                    "(N > 1), or this many partitions on the one GPU (N = 1)")
    ap.add_argument("--decomp-graph", type=int, default=0, help="--decomp on one GPU: record the whole decomposed step into one CUDA graph and replay it")
    ap.add_argument("--decomp-overlap", type=int, default=-1, help="--decomp: 1 = every stage first on the send-list elements, whose "
                    "exchange then overlaps the interior elements; 0 = unsplit; -1 = on when there is one partition per rank")
    args = ap.parse_args()
    if args.also is None:
        args.also = "C4,C4+perturbed,C5,C5+perturbed,H:f32" if (args.workload == "C3" and args.dtype == "f64" and args.gpus == 1) else "none"
    if args.gpus > 1 and "RANK" not in os.environ:
        # not under torchrun: spawn the N ranks ourselves (one process per GPU, rendezvous on 127.0.0.1) and hand over
        raise SystemExit(spawn_ranks(args.gpus))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    try:
        if args.decomp > 0:
            run_decomp(args, rank, world, local_rank)
        else:
            run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
