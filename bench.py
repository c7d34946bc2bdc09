#!/usr/bin/env python
"""bench.py -- cell-updates/s of the Dormand-Prince RK45 LLG step with FFT demag on one B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl mmx|reference] [--config c4]

A "step" is one pass of the whole hot path: one DP45 step (6 effective-field evaluations with
the full demag convolution, torque, stage combinations, error norm, controller) of BASELINE.json
configs[3] (256x256x64 cells, padded FFT 512x512x128, fp32) -- the configuration the metric is
quoted on -- at a fixed step size with forced acceptance ("Measurement").  One JSON
line is printed by rank 0.  N > 1 runs N independent replicas (the path does not shard: DESIGN.md
"Multi-GPU"), one process per GPU, timed as the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads as wl  # noqa: E402

METRIC = "cell-updates/s (RK45 LLG w/ demag)"
UNIT = "cell-updates/s"
DT = {"c1": 1e-13, "c2": 2e-14, "c3": 5e-15, "c4": 1e-13, "c5": 5e-15}

def ncu_traffic(category):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernel behind a profiler category, from the
    committed `ncu --set full` capture (profiles/ncu_traffic.csv, command in the .md beside it).  The row is
    used only while the kernel's source file still has the hash it was captured with; otherwise None."""
    import csv
    import hashlib
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        for row in csv.DictReader(f):
            if row["category"] != category:
                continue
            src = os.path.join(ROOT, row["source_file"])
            if not os.path.exists(src):
                return None
            with open(src, "rb") as g:
                if hashlib.sha1(g.read()).hexdigest() != row["source_sha1"]:
                    return None
            return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
    return None


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def algorithmic_bytes(spec):
    """Algorithmic HBM bytes per launch of every kernel category:
    a pruned pass reads only non-zero input and writes only kept output."""
    nx, ny, nz = spec.grid
    N = nx * ny * nz
    S = spec.S
    def pad(n, p):
        if p > 0:
            return n
        if n == 1:
            return 1
        q = 1
        while q < n:
            q *= 2
        return 2 * q
    px, py, pz = max(2, pad(nx, spec.pbc[0])), pad(ny, spec.pbc[1]), pad(nz, spec.pbc[2])
    xc = px // 2 + 1
    spec1 = 3 * nz * ny * xc * 8
    spec2 = 3 * nz * py * xc * 8
    ky, kz = (py // 2 + 1 if py > 1 else 1), (pz // 2 + 1 if pz > 1 else 1)
    three_d = nz > 1
    out = {
        "demag_x_fwd": 12 * N * S + spec1,
        "demag_x_inv": spec1 + 12 * N,
        "demag_mid_fwd": spec1 + spec2,
        "demag_mid_inv": spec2 + spec1,
        "demag_inner": (2 * spec2 + 6 * kz * ky * xc * 4) if three_d else (2 * spec1 + 4 * ky * xc * 4),
        # DP45: evaluation i = 1..5 moves (5 + i) fields, the last one 9: 49 fields of 12 N bytes / 6 launches
        "local": 12 * N * S * 49 / 6.0,
        "combine": 12 * N * S * 3,
    }
    return out


def survey_step_bytes(spec):
    """SURVEY 8d byte model of one DP45 step: one HBM sweep per 1-D FFT pass, innermost pass fused with the multiply,
    unit U = 12 N bytes, the (Nx+1)/Nx column ignored except in the kernel octant; 588 B/cell/sublattice for the
    local kernel.  3-D open: 26 U + octant; 2-D open: 10 U; 2-D periodic: 6 U per evaluation."""
    nx, ny, nz = spec.grid
    N = nx * ny * nz
    U = 12 * N
    if nz > 1:
        demag = 26 * U + 24 * (nx + 1) * (ny + 1) * (nz + 1)
    elif spec.pbc[0] > 0 and spec.pbc[1] > 0:
        demag = 6 * U + 4 * N
    else:
        demag = 10 * U + 16 * N + (12 * N if spec.S == 2 else 0)
    local = 588 * N if spec.S == 1 else (1104 + 12) * N
    return 6 * demag + local


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def wait_first_sample(self, timeout=3.0):
        """nvidia-smi needs ~0.1-0.3 s before its first line: call before the timed region."""
        t0 = time.time()
        while self.p is not None and time.time() - t0 < timeout:
            if os.path.getsize(self.f.name) > 0:
                return
            time.sleep(0.01)

    def mark(self):
        return time.time()

    def stop(self, t_begin=None, t_end=None):
        import datetime
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            if t_begin is not None:
                try:
                    ts = datetime.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                except ValueError:
                    continue
                if ts < t_begin - 0.02 or ts > t_end + 0.02:   # keep samples taken under load
                    continue
            c = c[1:]
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for nm, v in zip(names, c[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out["sm_mhz"] = float(np.median(sm))
            out["sm_max_mhz"] = float(max(mx))
            out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


def oracle_sample_grid(name, total_steps):
    """Bounded sample of the workload for the CPU oracle: a box of the same shape, cell size,
    material and seeded state recipe with fewer cells, sized so `total_steps` DP45 steps end
    within a few minutes on the host cores."""
    if name != "c4":
        return {"c1": (64, 16, 1), "c2": (128, 128, 1), "c3": (256, 64, 1), "c5": (256, 64, 1)}[name]
    if total_steps <= 3:
        return (128, 128, 32)
    if total_steps <= 60:
        return (64, 64, 16)
    return (32, 32, 8)


def time_oracle(name, grid, steps, warmup):
    """The oracle as it stands (never tuned), fixed-step DP45, wall clock on the host cores."""
    from oracle.world import World as OracleWorld
    spec = wl.make(name, grid)
    o = OracleWorld(spec)
    o.step_dp45_fixed(DT[name], max(warmup, 1))  # also builds its demag kernel (untimed setup)
    t0 = time.perf_counter()
    o.step_dp45_fixed(DT[name], steps)
    dt = time.perf_counter() - t0
    cells = grid[0] * grid[1] * grid[2]
    return cells * steps / dt, dt / steps


def run_reference(args, rank):
    if rank != 0:
        return
    grid = oracle_sample_grid(args.config, args.steps + args.warmup)
    value, s_per_step = time_oracle(args.config, grid, args.steps, args.warmup)
    cores = len(os.sched_getaffinity(0))
    sample = "oracle fp64 DP45 fixed-step on a %dx%dx%d box of the %s recipe (bounded sample)" % (*grid, args.config)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * s_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": "%s sample %dx%dx%d" % (args.config, *grid)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def max_over_ranks(ms, dist, device):
    """Replicas only: the job time is the slowest rank's device time."""
    if dist is None:
        return ms
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_seed(name, rank, world_size):
    """Every rank integrates an independent world of the same recipe (weak scaling)."""
    return None if world_size == 1 else 1000 + int(name[1]) + 100 * rank


def run_mmx(args, rank, local_rank, world_size):
    import torch

    import paper_2411_18194_b200 as mmx
    from paper_2411_18194_b200 import build as b

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libmmx has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world_size > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if rank == 0:
        b.build()
    if dist is not None:
        dist.barrier()

    name = args.config
    seed = replica_seed(name, rank, world_size)   # every rank: an independent replica, same recipe
    spec = wl.make(name) if seed is None else wl.make(name, seed=seed)
    N = spec.ncells
    stream = torch.cuda.current_stream()
    g = mmx.World.from_spec(spec, stream=stream.cuda_stream)
    dt = DT[name]
    K, W = args.steps, max(args.warmup, 3)

    def steps(n):
        return g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=n)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    clocks = ClockSampler(local_rank) if rank == 0 else None
    steps(W)
    if clocks:
        clocks.wait_first_sample()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_begin = time.time()
    e0.record(stream)
    st = steps(K)
    e1.record(stream)
    barrier()
    t_end = time.time()
    ms = e0.elapsed_time(e1)
    clk = clocks.stop(t_begin, t_end) if clocks else None
    ms = max_over_ranks(ms, dist, "cuda")
    value = N * K * world_size / (ms * 1e-3)
    launches = int(st["launches"])

    # ---- roofline of the dominant kernel: CUDA events around every launch, on the launching stream
    g.profile_enable(True)
    steps(K)
    prof = g.profile_read()
    g.profile_enable(False)
    alg = algorithmic_bytes(spec)
    total_prof_ms = sum(v[0] for v in prof.values())
    dom = max((k for k in prof if k in alg and prof[k][1] > 0), key=lambda k: prof[k][0])
    peak, peak_src = measured_peaks()
    dom_ms = prof[dom][0] / prof[dom][1]
    achieved = alg[dom] / (dom_ms * 1e-3) / 1e9
    kernels = {k: {"ms_per_launch": v[0] / v[1], "launches_per_step": v[1] / K, "share": v[0] / total_prof_ms,
                   "GBs": (alg[k] / (v[0] / v[1] * 1e-3) / 1e9) if k in alg else None}
               for k, v in prof.items() if v[1] > 0}
    step_bytes = sum(alg[k] * prof[k][1] / K for k in prof if k in alg and prof[k][1] > 0)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": ncu_traffic(dom), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg[dom], "ms_per_launch": dom_ms,
                # two byte models of a step: "as built" counts the passes this design launches (the Nx+1 column,
                # the k_combine1 pass); "survey" is SURVEY 8d's model (2608 B/cell/step on c4: 10.94 GB), the one
                # BASELINE.md's >= 50 % of 8 TB/s target is stated on
                "step_algorithmic_bytes": step_bytes,
                "step_frac_of_peak": step_bytes / (ms / K * 1e-3) / 1e9 / peak,
                "step_frac_of_8TBs": step_bytes / (ms / K * 1e-3) / 8e12,
                "step_bytes_survey_model": survey_step_bytes(spec),
                "step_frac_of_peak_survey_model": survey_step_bytes(spec) / (ms / K * 1e-3) / 1e9 / peak,
                "step_frac_of_8TBs_survey_model": survey_step_bytes(spec) / (ms / K * 1e-3) / 8e12,
                "kernels": kernels}

    # ---- end to end through the C-ABI, host buffers in and out every step (bytes counted from the tensors copied).
    # (1) serial: mmx_set_state(HOST) + one DP45 step + mmx_get_state(HOST), each call synchronous;
    # (2) overlapped, the way a caller that owns streams uses the same ABI: the step's input travels host -> device
    #     staging buffer on a copy stream while the previous step runs, enters the world with mmx_set_state(DEVICE),
    #     the result leaves with mmx_get_state(DEVICE) into a second staging buffer and travels device -> host on a
    #     third stream while the next step runs.  Every step still moves 12 N S bytes in and 12 N bytes out of pinned
    #     host memory and recomputes k1 (7 evaluations).  `e2e` is (2); (1) is kept beside it.
    Ke = min(K, 8)
    hin = [torch.from_numpy(np.ascontiguousarray(spec.m[s])).pin_memory() for s in range(spec.S)]
    hout = [torch.empty_like(hin[0]).pin_memory() for _ in range(2)]
    def e2e_step_serial():
        for s in range(spec.S):
            g.set_state(mmx.F_M[s], hin[s])
        g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=1)
        g.get_state(mmx.F_M0, hout[0])
    e2e_step_serial()
    barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        e2e_step_serial()
    torch.cuda.synchronize()
    te_serial = time.perf_counter() - t0

    cs, ds = torch.cuda.Stream(), torch.cuda.Stream()
    din = [[torch.empty(hin[s].shape, dtype=torch.float32, device="cuda") for s in range(spec.S)] for _ in range(2)]
    dout = [torch.empty(hin[0].shape, dtype=torch.float32, device="cuda") for _ in range(2)]
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_used = [torch.cuda.Event() for _ in range(2)]
    ev_res = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]
    def h2d(i):
        b = i & 1
        cs.wait_event(ev_used[b])                      # the staging buffer has been consumed by set_state two steps ago
        with torch.cuda.stream(cs):
            for s in range(spec.S):
                din[b][s].copy_(hin[s], non_blocking=True)
            ev_in[b].record(cs)
    def run_overlapped(n):
        for e in ev_used + ev_out:
            e.record(stream)
        h2d(0)
        for i in range(n):
            b = i & 1
            if i + 1 < n:
                h2d(i + 1)                             # overlaps step i
            stream.wait_event(ev_in[b])
            for s in range(spec.S):
                g.set_state(mmx.F_M[s], din[b][s])     # device -> device, on the world's stream
            ev_used[b].record(stream)
            stream.wait_event(ev_out[b])               # the result buffer has left for the host two steps ago
            g.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=dt, nsteps=1)
            g.get_state(mmx.F_M0, dout[b])
            ev_res[b].record(stream)
            ds.wait_event(ev_res[b])
            with torch.cuda.stream(ds):
                hout[b].copy_(dout[b], non_blocking=True)   # overlaps step i + 1
                ev_out[b].record(ds)
        torch.cuda.synchronize()
    run_overlapped(2)
    barrier()
    t0 = time.perf_counter()
    run_overlapped(Ke)
    te = time.perf_counter() - t0
    if dist is not None:
        t = torch.tensor([te, te_serial], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        te, te_serial = float(t[0].item()), float(t[1].item())
    e2e = {"value": N * Ke * world_size / te, "unit": UNIT, "h2d_bytes_per_step": 12 * N * spec.S,
           "d2h_bytes_per_step": 12 * N, "steps": Ke, "ms_per_step": 1e3 * te / Ke,
           "serial": {"value": N * Ke * world_size / te_serial, "ms_per_step": 1e3 * te_serial / Ke},
           "note": "per step: pinned host -> device staging (copy stream) -> mmx_set_state(DEVICE) -> 1 DP45 step (7 evaluations: "
                   "k1 is recomputed after set_state) -> mmx_get_state(DEVICE) -> device staging -> pinned host (third stream); "
                   "copies of neighbouring steps overlap the step; 'serial' = the same with the synchronous HOST calls"}

    # ---- separate adaptive run: accepted / rejected counts (not the timed figure)
    ad = g.step_rk45(method=mmx.DP45, tol=1e-5, dt0=dt, nsteps=10)
    adaptive = {"accepted": ad["accepted"], "rejected": ad["rejected"], "dt": ad["dt"]}
    dev_bytes = g.device_bytes()
    g.destroy()

    # ---- the other BASELINE.json configs (parity cases, small 2-D grids that fit in L2): DP45 fixed dt, same timing
    # rules, reported beside the headline (they are latency-bound: DESIGN.md section 8)
    others = None
    if rank == 0 and world_size == 1 and name == "c4" and not args.no_other_configs:
        others = {}
        for oname in ("c1", "c2", "c3", "c5"):
            ospec = wl.make(oname)
            og = mmx.World.from_spec(ospec, stream=stream.cuda_stream)
            run = lambda n: og.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=DT[oname], nsteps=n)
            run(5)
            ko = 100
            o0, o1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            o0.record(stream)
            run(ko)
            o1.record(stream)
            torch.cuda.synchronize()
            oms = o0.elapsed_time(o1) / ko
            others[oname] = {"grid": list(ospec.grid), "S": ospec.S, "ms_per_step": oms, "steps_per_s": 1e3 / oms,
                             "cell_updates_per_s": ospec.ncells * 1e3 / oms,
                             "frac_of_8TBs_survey_model": survey_step_bytes(ospec) / (oms * 1e-3) / 8e12}
            og.destroy()
            # a parameter sweep (the paper's demo 2.1 sweeps current and exchange reduction): independent worlds of
            # the same recipe, one stream and one host thread each; aggregate throughput over all of them
            import threading
            nw = 8
            ws = []
            for k in range(nw):
                stk = torch.cuda.Stream()
                ws.append((mmx.World.from_spec(wl.make(oname, seed=2000 + k), stream=stk.cuda_stream), stk))
            stepk = lambda gw, n: gw.step_rk45(method=mmx.DP45, fixed_dt=True, dt0=DT[oname], nsteps=n)
            for gw, _ in ws:
                stepk(gw, 5)
            torch.cuda.synchronize()
            tw0 = time.perf_counter()
            th = [threading.Thread(target=stepk, args=(gw, ko)) for gw, _ in ws]
            for t_ in th:
                t_.start()
            for t_ in th:
                t_.join()
            torch.cuda.synchronize()
            tw = time.perf_counter() - tw0
            others[oname]["sweep_of_8_worlds_cell_updates_per_s"] = nw * ospec.ncells * ko / tw
            for gw, _ in ws:
                gw.destroy()

    cpu = None
    if rank == 0 and world_size == 1 and not args.no_cpu_baseline:
        grid = oracle_sample_grid(name, 1)
        nstep_cpu = 5  # about 12 s of CPU work on the c4 sample box
        v, s_step = time_oracle(name, grid, nstep_cpu, 1)
        cpu = {"value": v, "unit": UNIT, "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
               "sample": "%d fixed-step DP45 steps of the fp64 numpy oracle on a %dx%dx%d box of the %s recipe "
                         "(%.1f s per step)" % (nstep_cpu, *grid, name, s_step)}
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world_size, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "%s %dx%dx%d DP45 fixed dt=%g, demag+exchange" % (name, *spec.grid, dt),
                       "cells": N, "field_evals_per_s": value * 6,
                       "l2": "working set %.2f GB >> 126 MB L2, no flush needed" % (dev_bytes / 1e9),
                       "parallelism": "replicas x%d" % world_size, "other_configs": others},
            "clocks": clk, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
            "cpu_baseline": cpu, "adaptive": adaptive,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="mmx", choices=["mmx", "reference"])
    ap.add_argument("--config", default="c4", choices=list(DT))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world_size = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if world_size != args.gpus and world_size == 1 and args.gpus > 1:
        raise SystemExit("launch with torch.distributed.run --nproc-per-node %d" % args.gpus)
    run_mmx(args, rank, local_rank, world_size)


if __name__ == "__main__":
    main()
