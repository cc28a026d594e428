#!/usr/bin/env python
"""bench.py -- Z4c RHS + KO + RK4 throughput of libsacra on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference] [--headline-only]

One "step" = one full RK4 step (5 halo fills + 4 fused RHS/KO/RK substages) of the whole workload through the
C ABI call sacra_rk4_step. Default workload: BASELINE.json configs[4], one 256^3 periodic patch, 25 FP64 fields,
Brill-Lindquist data + 1e-12 seeded noise (the configuration the north_star target is stated on; it fits one
GPU). N > 1 (torchrun): "replicas only" -- every rank advances its own independent 256^3 patch, no data-path
collective (Multi-GPU); value = points of all ranks / max-over-ranks time. With --decomp PXxPYxPZ the N
ranks instead share ONE periodic domain, a 256^3 block each, and exchange 3-layer halos over NCCL before every substage
(run_decomp).

Prints ONE JSON line (rank 0). Keys: see DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Z4c RHS+RK4 Mpoint-updates/s FP64"
UNIT = "Mpoint-updates/s"
NF = 25
# Algorithmic work per point: 16 field passes x 8 B x 25 fields per RK4 step (the
# minimum of any RK4 formulation, 3 + 5 + 5 + 3; the increment-form acc of this library moves 3 + 5 + 5 + 4 = 17 with
# SACRA_FLAG_SKIP_INCREMENT, which the timed steps set, and 18 without), i.e. 800 B per substage launch on average;
# FP64 work per RHS evaluation + RK update after CSE: 3 206 FP64 instructions (DADD 1 399, DMUL 818, DFMA 989 per
# point in the SASS of k_z4c<2>, profiles/r02_sass_histogram.md) = 4 195 flop with FMA = 2.
ALG_BYTES_PER_POINT_STEP = 16 * 8 * NF
ALG_FLOP_PER_POINT_STAGE = 4195.0
ALG_FP64_INSTR_PER_POINT_STAGE = 3206.0
FP64_LANES_PER_SM, N_SM = 64, 148
# The count SURVEY 8(d) asks for, beside the SASS one: the oracle's point-wise algebra instantiated with an
# operation-counting scalar (1 787 add + 1 777 mul + 12 div = 3 576, no CSE; tests/test_bench_counts.py checks the number
# against orc.count_ops()) plus the needed derivative operators in canonical form with shared inner differences
# (48 D1 x 5 + 33 D_aa x 9 + 33 D_ab x 5 + 25 upwind x 41 + 25 KO x 42 = 2 777). The roofline
# fraction is credited with the SMALLER of the two counts (the SASS one).
ORACLE_ALGEBRA_OPS = 1787 + 1777 + 12
CANONICAL_DERIVATIVE_OPS = 48 * 5 + 33 * 9 + 33 * 5 + 25 * 41 + 25 * 42
ORACLE_FLOP_PER_POINT_STAGE = float(ORACLE_ALGEBRA_OPS + CANONICAL_DERIVATIVE_OPS)
# Measured FP64 rate of this pool's B200 (BASELINE.md section 3, round-1 register-chain microbenchmark at 1 965 MHz):
# DFMA 17.06 Tinst/s = 34.1 TFLOP/s (58.7 of the 64 lanes per SM and clock); scaled with the SM clock of the run.
FP64_MEASURED_TFLOPS, FP64_MEASURED_AT_MHZ = 34.1, 1965.0
TIMED_FLAGS = ["SKIP_INCREMENT"]     # sacra_params_t.flags of every timed step (not the library default, see run_ours)


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


def _csrc_digest() -> str:
    """digest of the kernel sources (csrc/*, include/sacra.h) and of the nvcc flags"""
    import hashlib
    from paper_2607_08743_b200 import build as b
    h = hashlib.sha256(" ".join(b.FLAGS).encode())
    files = [os.path.join(ROOT, "include", "sacra.h")] + [os.path.join(b.CSRC, f) for f in os.listdir(b.CSRC)]
    for f in sorted(files):
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def _committed_traffic(workload: str):
    """dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/r03_traffic.json), or None
    when the capture was made for other kernel sources or another workload"""
    p = os.path.join(ROOT, "profiles", "r03_traffic.json")
    try:
        d = json.load(open(p))
    except (OSError, ValueError):
        return None
    if d.get("workload") != workload or d.get("csrc_digest") != _csrc_digest():
        return None
    return float(d["dram_bytes_per_launch_mean"])


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0=None, t1=None):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if (t0 is None or t >= t0 - 0.05) and (t1 is None or t <= t1 + 0.05)]
        rows = rows or [r for (_, r) in self.rows]
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def make_workload(idx: int, n: int | None):
    from paper_2607_08743_b200 import workloads as wl
    kw = {}
    if n:
        kw["n"] = n
    return wl.make(idx, **kw)


ORACLE_SAMPLE_N = 160     # both CPU legs (cpu_baseline and --impl reference) time the same sample


def oracle_sample(w, n_sample: int):
    """Bounded sample of the workload for the CPU legs: the central n_sample^3 block of patch 0 (same data,
    same spacing and parameters), advanced as its own periodic patch. Same work per point as the full run."""
    import numpy as np
    from paper_2607_08743_b200 import workloads as wl
    p = w.patches[0]
    m = min(n_sample, p.nx, p.ny, p.nz)
    ps, total = wl.make_layout([(m, m, m)], [p.dx], [p.dt], [(0.0, 0.0, 0.0)])
    s = wl.Workload("sample", ps, dict(w.params), np.zeros(total))
    o = [(d - m) // 2 for d in (p.nz, p.ny, p.nx)]
    for f in range(NF):
        s.active_view(s.state, 0, f)[...] = w.active_view(w.state, 0, f)[o[0]:o[0] + m, o[1]:o[1] + m, o[2]:o[2] + m]
    return s


def time_oracle(sample, steps, warmup):
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import orc
    u = sample.state.copy()
    for _ in range(warmup):
        orc.rk4_step(sample.patches, sample.params, u)
    ts = []
    for _ in range(steps):
        t = time.perf_counter()
        orc.rk4_step(sample.patches, sample.params, u)
        ts.append(time.perf_counter() - t)
    return ts, orc.num_threads()


def config_of(w, world: int):
    """the `config` object of the JSON line: the same for both arms, so that they can be compared key by key"""
    state_bytes = w.state.size * 8
    return {"workload": w.name, "patches": len(w.patches), "points": w.npoints, "fields": NF, "ghosts": 3,
            "state_bytes": state_bytes, "l2": "state (%.2f GB) larger than L2; no flush needed" %
            (state_bytes / 1e9) if state_bytes > 2.6e8 else "state fits L2: numbers are L2-resident",
            "parallelism": "replicas only" if world > 1 else "1 GPU"}


def run_reference(args):
    """the oracle, as it stands, on the host cores. Without --oracle-n it advances the WHOLE workload (config 4: the full
    256^3 patch, about 10 s per RK4 step on 16 cores), so both arms run the same configuration; --oracle-n M bounds it
    to the central M^3 block (the sample of the cpu_baseline leg)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.config, args.n)
    if args.oracle_n:
        s = oracle_sample(w, args.oracle_n)
        what = "central %d^3 block of %s as a periodic patch" % (s.patches[0].nx, w.name)
    else:
        s, what = w, "the whole of %s" % w.name
    ts, cores = time_oracle(s, args.steps, args.warmup)
    tot = sum(ts)
    val = s.npoints * len(ts) / tot / 1e6
    sample = "%s, %d RK4 steps" % (what, len(ts))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(ts),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_of(w, int(os.environ.get("WORLD_SIZE", "1"))),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2607_08743_b200 import sacra

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libsacra has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    from paper_2607_08743_b200 import replicas

    def max_over_ranks(x: float) -> float:
        return replicas.max_over_ranks(x, device="cuda")

    w = make_workload(args.config, args.n)
    # the timed steps do not store the increment S ("may be skipped outside verification"; the new
    # state is bit-identical, tests/test_gpu_multistep.py); the per-launch split below times the same kernels
    ps, prm = sacra.make_patches(w.patches), sacra.make_params(dict(w.params, flags=sacra.FLAG_SKIP_INCREMENT))
    npts = w.npoints
    n = w.state.size
    host_in = torch.from_numpy(w.state).pin_memory()
    host_out = torch.empty_like(host_in).pin_memory()
    u = torch.empty(n, dtype=torch.float64, device="cuda")
    work = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    K, W = args.steps, args.warmup

    def ev():
        return torch.cuda.Event(enable_timing=True)

    # ---- device-resident throughput: K consecutive steps, state stays in HBM -----------------------------
    u.copy_(host_in)
    for _ in range(W):
        sacra.rk4_step(ps, prm, u, work, n)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier()
    t0 = time.time()
    evs = [ev() for _ in range(K + 1)]
    evs[0].record(stream)
    for s in range(K):
        sacra.rk4_step(ps, prm, u, work, n)
        evs[s + 1].record(stream)
    barrier()
    t1 = time.time()
    step_ms = [evs[s].elapsed_time(evs[s + 1]) for s in range(K)]
    total_ms = max_over_ranks(evs[0].elapsed_time(evs[K]))
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    if not bool(torch.isfinite(u).all()):
        raise SystemExit("bench.py: non-finite state after the timed steps")
    # the same K steps with the library's default flags (stage 4 also stores S): reported beside the headline
    prm_default = sacra.make_params(dict(w.params, flags=0))
    sacra.rk4_step(ps, prm_default, u, work, n)
    d0, d1 = ev(), ev()
    barrier()
    d0.record(stream)
    for s in range(K):
        sacra.rk4_step(ps, prm_default, u, work, n)
    d1.record(stream)
    barrier()
    default_flags_ms = max_over_ranks(d0.elapsed_time(d1)) / K

    # ---- kernel split for the roofline: same nine calls, CUDA events around each -----------------------
    a, b, acc = work[:n], work[n:2 * n], work[2 * n:]
    seq = [(u, a), (a, b), (b, a), (a, u)]
    fill_ms, sub_ms = [], []
    for it in range(W + K):
        marks = []
        for stage, (src, dst) in enumerate(seq, start=1):
            e = [ev(), ev(), ev()]
            e[0].record(stream)
            sacra.fill_ghosts(ps, src)
            e[1].record(stream)
            sacra.rk4_substep(ps, prm, stage, u, src, dst, acc)
            e[2].record(stream)
            marks.append(e)
        e = [ev(), ev()]
        e[0].record(stream); sacra.fill_ghosts(ps, u); e[1].record(stream)
        torch.cuda.synchronize()
        if it >= W:
            fill_ms += [m[0].elapsed_time(m[1]) for m in marks] + [e[0].elapsed_time(e[1])]
            sub_ms += [m[1].elapsed_time(m[2]) for m in marks]
    sub_avg = sum(sub_ms) / len(sub_ms)
    fill_avg = sum(fill_ms) / len(fill_ms)

    # ---- constraint monitor on the evolved state: Eqs. 20-22, timed beside the step ------------
    con = work[:n]
    scratch = torch.zeros(sacra.constraint_scratch_doubles(ps), dtype=torch.float64, device="cuda")
    norms = torch.zeros(4, dtype=torch.float64, device="cuda")
    mon_ms = []
    for it in range(W + K):
        e = [ev(), ev(), ev()]
        e[0].record(stream)
        sacra.constraints(ps, u, con)
        e[1].record(stream)
        sacra.constraint_norms(ps, con, scratch, norms)
        e[2].record(stream)
        torch.cuda.synchronize()
        if it >= W:
            mon_ms.append((e[0].elapsed_time(e[1]), e[1].elapsed_time(e[2])))
    con_ms = sum(m[0] for m in mon_ms) / len(mon_ms)
    nrm_ms = sum(m[1] for m in mon_ms) / len(mon_ms)
    norms_host = [float(v) for v in norms.cpu()]

    # ---- end to end with HOST buffers: H2D of the state, one step, D2H of the new state, every step ----
    # (a) serial: copy in, step, copy out on one stream
    barrier()
    e0, e1 = ev(), ev()
    for it in range(min(W, 2) + K):
        if it == min(W, 2):
            barrier()
            e0.record(stream)
        u.copy_(host_in, non_blocking=True)
        sacra.rk4_step(ps, prm, u, work, n)
        host_out.copy_(u, non_blocking=True)
    e1.record(stream)
    barrier()
    e2e_serial_ms = max_over_ranks(e0.elapsed_time(e1))
    # (b) the same work per step as a stream of independent jobs: two device buffers, the copy-in of step i+1 and
    # the copy-out of step i-1 run on their own streams beside the kernels of step i (PCIe is full duplex)
    u2 = [u, torch.empty_like(u)]
    work2 = [work, torch.zeros_like(work)]
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_comp = [torch.cuda.Event() for _ in range(2)]
    ev_free = [torch.cuda.Event() for _ in range(2)]
    e0, e1 = ev(), ev()
    barrier()
    nwarm = min(W, 2)
    for it in range(nwarm + K):
        b = it & 1
        if it == nwarm:
            for st in (s_in, s_out):
                st.synchronize()
            barrier()
            e0.record(s_in)
        with torch.cuda.stream(s_in):
            if it >= 2:
                s_in.wait_event(ev_free[b])            # the copy-out of the job that used this buffer is done
            u2[b].copy_(host_in, non_blocking=True)
            ev_in[b].record(s_in)
        stream.wait_event(ev_in[b])
        sacra.rk4_step(ps, prm, u2[b], work2[b], n)
        ev_comp[b].record(stream)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_comp[b])
            host_out.copy_(u2[b], non_blocking=True)
            ev_free[b].record(s_out)
    e1.record(s_out)
    s_out.synchronize()
    barrier()
    e2e_ms = max_over_ranks(e0.elapsed_time(e1))
    del u2, work2

    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return

    hbm_gbs, sm_max_mhz, peak_src = _peaks()
    value = world * npts * K / (total_ms * 1e-3) / 1e6   # every rank advances an identical patch (replicas)
    e2e_val = world * npts * K / (e2e_ms * 1e-3) / 1e6
    # roofline of the dominant kernel (the fused substage kernel), per launch, averaged over the 4 stages
    alg_bytes = ALG_BYTES_PER_POINT_STEP / 4.0 * npts
    alg_flop = ALG_FLOP_PER_POINT_STAGE * npts
    fp64_peak_tf = N_SM * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12          # nominal
    fp64_meas_tf = FP64_MEASURED_TFLOPS * sm_max_mhz / FP64_MEASURED_AT_MHZ         # measured DFMA rate
    t_hbm = alg_bytes / (hbm_gbs * 1e9)
    t_alu = alg_flop / (fp64_meas_tf * 1e12)
    t_k = sub_avg * 1e-3
    # the metric's roofline: the slower of the compulsory bytes at the measured HBM rate and the flops at the MEASURED
    # FP64 rate; the nominal FP64 peak and both fractions are reported beside it
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": alg_flop / t_k / 1e12, "peak": fp64_meas_tf, "unit": "TFLOP/s"}
    else:
        roof = {"bound": "hbm", "achieved": alg_bytes / t_k / 1e9, "peak": hbm_gbs, "unit": "GB/s"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof.update({
        "t_hbm_ms": 1e3 * t_hbm, "t_alu_ms": 1e3 * t_alu, "t_alu_nominal_ms": 1e3 * alg_flop / (fp64_peak_tf * 1e12),
        "alu_peak_measured_tflops": fp64_meas_tf, "alu_peak_nominal_tflops": fp64_peak_tf,
        "alu_frac_measured_peak": (alg_flop / t_k / 1e12) / fp64_meas_tf,
        "alg_flop_per_point_stage": {"credited": ALG_FLOP_PER_POINT_STAGE,
                                     "kernel_sass_fma2": ALG_FLOP_PER_POINT_STAGE,
                                     "oracle_counting_scalar": ORACLE_FLOP_PER_POINT_STAGE,
                                     "note": "oracle: algebra %d ops (no CSE) + needed derivative operators %d; the "
                                             "smaller count is credited" % (ORACLE_ALGEBRA_OPS, CANONICAL_DERIVATIVE_OPS)},
        "traffic": args.traffic if args.traffic is not None else _committed_traffic(w.name),
        "traffic_source": "profiles/r03_traffic.json (ncu dram__bytes_read.sum + dram__bytes_write.sum, mean of the four "
                          "substage launches; null if the kernel sources changed since the capture)",
        "kernel": "k_z4c (fused derivative+algebra+KO+RK substage)",
        "kernel_ms": sub_avg, "kernel_share_of_step": 4 * sub_avg / (4 * sub_avg + 5 * fill_avg),
        "fill_ms": fill_avg, "alg_bytes_per_launch": alg_bytes, "alg_flop_per_launch": alg_flop,
        "hbm_frac": (alg_bytes / t_k / 1e9) / hbm_gbs, "alu_frac": (alg_flop / t_k / 1e12) / fp64_peak_tf,
        # FP64 instructions against the issue rate of the FP64 pipe (64 lanes per SM and clock): the tighter ALU
        # ceiling of this instruction mix (a quarter FMAs); measured DFMA/DADD rates: BASELINE.md section 3
        "fp64_issue_frac": ALG_FP64_INSTR_PER_POINT_STAGE * npts / t_k /
                           (N_SM * FP64_LANES_PER_SM * sm_max_mhz * 1e6),
        "peak_source": peak_src + "; FP64: measured DFMA rate 34.1 TFLOP/s at 1 965 MHz (BASELINE.md section 3) scaled "
                       "to sm_max_mhz; nominal = 148 SM x 64 lanes x 2 x sm_max_mhz (DESIGN.md section 7)"})

    # ---- CPU oracle beside it (reported baseline, bounded sample) -----------------------------------------
    cpu = None
    if not args.no_cpu:
        # bounded sample: about 10-20 s of oracle time on the box's host cores
        s = oracle_sample(w, args.oracle_n or ORACLE_SAMPLE_N)
        nst = 4 if s.npoints > 128 ** 3 else 8
        ts, cores = time_oracle(s, nst, 0)
        cpu = {"value": s.npoints * len(ts) / sum(ts) / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "central %d^3 block of %s as a periodic patch, %d RK4 steps (%.1f s)"
                         % (s.patches[0].nx, w.name, len(ts), sum(ts))}

    state_bytes = n * 8
    cfg = config_of(w, world)
    ghost_cells = sum((p.nx + 6) * (p.ny + 6) * (p.nz + 6) - p.nx * p.ny * p.nz for p in w.patches)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": total_ms / K, "ms_per_step_min": min(step_ms), "ms_per_step_median": sorted(step_ms)[K // 2],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": cfg,
        # sacra_params_t.flags of every timed step (value, e2e, roofline split, configs 0-3): stage 4 does not store the
        # increment S, one field pass less per step than the library default; the new state is the same bit for bit
        "flags": TIMED_FLAGS, "ms_per_step_default_flags": default_flags_ms,
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes,
                "ms_per_step": e2e_ms / K, "how": "pinned host state in and out every step; independent jobs, two device "
                "buffers, copy-in / kernels / copy-out on three streams",
                "serial_value": world * npts * K / (e2e_serial_ms * 1e-3) / 1e6, "serial_ms_per_step": e2e_serial_ms / K},
        "gpu_launches": 9 * K, "clocks": clocks, "roofline": roof, "cpu_baseline": cpu,
        # the other kernels of the step against HBM: the halo fill reads and writes the ghost cells once
        "kernels": {"k_fill_ghosts": {"ms": fill_avg, "hbm_frac": 2 * 8.0 * NF * ghost_cells / (fill_avg * 1e-3) / 1e9 / hbm_gbs},
                    "k_z4c": {"ms": sub_avg, "hbm_frac": (alg_bytes / t_k / 1e9) / hbm_gbs}},
        # the constraint monitor on the state after the timed steps: 15 fields read + 4 written = 152 B per point
        "constraint_monitor": {"constraints_ms": con_ms, "norms_ms": nrm_ms, "Mpoints_per_s": npts / (con_ms * 1e-3) / 1e6,
                               "hbm_frac": 152.0 * npts / (con_ms * 1e-3) / 1e9 / hbm_gbs,
                               "norms_H_Mx_My_Mz": norms_host},
    }
    if args.all_configs and world == 1 and args.config == 4 and not args.n:
        out["configs"] = [measure_config(i, args, hbm_gbs, fp64_meas_tf) for i in range(4)]
    print(json.dumps(out))


def run_decomp(args):
    """--decomp PXxPYxPZ: the sharded path of SURVEY 8(f) f-4. PX*PY*PZ = the number of
    ranks; every rank owns one block of a periodic (n PX) x (n PY) x (n PZ) domain and advances it with
    halo.rk4_step_distributed: pack -> NCCL point-to-point -> unpack of the 3-layer halos before every substage, overlapped
    with the interior cells. The domain is the periodic tiling of the workload's patch (config 4: 256^3 per rank), so
    every rank's block must come out equal, bit for bit, to the single-GPU periodic step of that patch: checked on one
    step before the timed region (`decomp_check`). Weak scaling: the work per GPU is fixed."""
    import torch
    import torch.distributed as dist
    from paper_2607_08743_b200 import halo, replicas, sacra

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dims = tuple(int(v) for v in args.decomp.lower().split("x"))
    if len(dims) != 3 or dims[0] * dims[1] * dims[2] != world:
        raise SystemExit("bench.py: --decomp %s does not match %d ranks" % (args.decomp, world))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libsacra has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = make_workload(args.config, args.n)
    if len(w.patches) != 1:
        raise SystemExit("bench.py: --decomp needs a single-patch workload")
    p = w.patches[0]
    prm = dict(w.params, flags=sacra.FLAG_SKIP_INCREMENT)
    topo = halo.CartTopology(dims)
    n = w.state.size
    host_in = torch.from_numpy(w.state).pin_memory()
    host_out = torch.empty_like(host_in).pin_memory()
    u = torch.empty(n, dtype=torch.float64, device="cuda")
    work = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    K, W = args.steps, args.warmup
    bufs = {}

    # one step against the single-GPU periodic step of the same patch: same bits
    v, wv = torch.from_numpy(w.state).cuda(), torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    sacra.rk4_step([p], prm, v, wv, n)
    u.copy_(host_in)
    halo.rk4_step_distributed(p, prm, u, work, topo, rank, buffers=bufs, overlap=True)
    torch.cuda.synchronize()
    same = float(bool(torch.equal(u, v)))
    same = replicas.sum_over_ranks(same, device="cuda") == world
    del v, wv

    def ev():
        return torch.cuda.Event(enable_timing=True)

    def timed(overlap, sampler=None):
        u.copy_(host_in)
        for _ in range(W):
            halo.rk4_step_distributed(p, prm, u, work, topo, rank, buffers=bufs, overlap=overlap)
        if sampler is not None and rank == 0:
            sampler.start()
            time.sleep(0.25)
        barrier()
        t0 = time.time()
        e0, e1 = ev(), ev()
        e0.record(stream)
        for _ in range(K):
            halo.rk4_step_distributed(p, prm, u, work, topo, rank, buffers=bufs, overlap=overlap)
        e1.record(stream)
        barrier()
        ms = replicas.max_over_ranks(e0.elapsed_time(e1), device="cuda")
        clocks = sampler.stop(t0, time.time()) if sampler is not None and rank == 0 else None
        return ms, clocks

    # the headline is the mode --overlap names (default off: on one GPU, where every exchange is a local copy, the split
    # into interior and shell launches costs more than it hides -- 36.0 against 27.1 ms per 256^3 step);
    # the other mode is timed beside it
    head = args.overlap == "on"
    other_ms, _ = timed(not head)
    total_ms, clocks = timed(head, ClockSampler(local))
    on_ms, plain_ms = (total_ms, other_ms) if head else (other_ms, total_ms)
    if not bool(torch.isfinite(u).all()):
        raise SystemExit("bench.py: non-finite state after the timed steps")
    # end to end: pinned host state in, one distributed step, new state out, every step
    barrier()
    e0, e1 = ev(), ev()
    for it in range(2 + K):
        if it == 2:
            barrier()
            e0.record(stream)
        u.copy_(host_in, non_blocking=True)
        halo.rk4_step_distributed(p, prm, u, work, topo, rank, buffers=bufs, overlap=head)
        host_out.copy_(u, non_blocking=True)
    e1.record(stream)
    barrier()
    e2e_ms = replicas.max_over_ranks(e0.elapsed_time(e1), device="cuda")
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return
    npts = w.npoints
    msgs = 2 * sum(1 for d in dims if d > 1)
    xbytes = 5 * 2 * 8 * sum(sacra.face_doubles(p, a) for a in range(3) if dims[a] > 1)      # sent per rank and step
    cfg = config_of(w, world)
    cfg.update({"parallelism": "3-D blocks %s, 3-layer halo, NCCL p2p, exchange %s" %
                               (args.decomp, "overlapped with the interior" if head else "before each substage"),
                "global_domain": [p.nx * dims[0], p.ny * dims[1], p.nz * dims[2]], "points_per_gpu": npts})
    print(json.dumps({
        "metric": METRIC, "value": world * npts * K / (total_ms * 1e-3) / 1e6, "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": W, "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": cfg, "flags": TIMED_FLAGS,
        "e2e": {"value": world * npts * K / (e2e_ms * 1e-3) / 1e6, "unit": UNIT, "h2d_bytes_per_step": n * 8,
                "d2h_bytes_per_step": n * 8, "ms_per_step": e2e_ms / K,
                "how": "per rank: pinned host state in, one distributed step, new state out, on one stream"},
        # 4 substage launches (overlap on: interior + shell each) + pack / unpack of 6 faces x 5 exchanges
        "gpu_launches": K * ((8 if head else 4) + 5 * 12), "clocks": clocks,
        "halo": {"messages_per_exchange": msgs, "exchanges_per_step": 5, "sent_bytes_per_rank_and_step": xbytes,
                 "overlap": args.overlap, "ms_per_step_overlap_on": on_ms / K, "ms_per_step_overlap_off": plain_ms / K},
        "decomp_check": "every rank's block after one step is bit-equal to sacra_rk4_step of the periodic patch: %s"
                        % ("yes" if same else "NO"),
        "roofline": None, "cpu_baseline": None}))
    if not same:
        raise SystemExit("bench.py: the distributed step differs from the single-GPU periodic step")


def measure_config(idx, args, hbm_gbs, fp64_peak_tf):
    """BASELINE.json configs 0-3 (the parity-test cases) timed the same way: K consecutive sacra_rk4_step calls from the
    initial data, and -- these are launch-bound -- the same step captured into a CUDA graph by the caller and replayed.
    frac: roofline fraction of the whole step (the slower of the algorithmic bytes at HBM bandwidth and the flops at the
    FP64 peak, over the measured time per step). States of configs 0-1 fit the L2: their numbers are L2-resident."""
    import torch
    from paper_2607_08743_b200 import sacra
    w = make_workload(idx, None)
    ps, prm = sacra.make_patches(w.patches), sacra.make_params(dict(w.params, flags=sacra.FLAG_SKIP_INCREMENT))
    n = w.state.size
    u0 = torch.from_numpy(w.state).cuda()
    u = u0.clone()
    work = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    K = max(args.steps, 20)
    stream = torch.cuda.current_stream()

    def timed(fn):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / K

    ms = timed(lambda: sacra.rk4_step(ps, prm, u, work, n))
    u.copy_(u0)
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        sacra.rk4_step(ps, prm, u, work, n, stream=side)        # warm-up on the capture stream (tensor maps cached)
        side.synchronize()
        with torch.cuda.graph(g, stream=side):
            sacra.rk4_step(ps, prm, u, work, n, stream=side)
    u.copy_(u0)
    ms_graph = timed(g.replay)
    npts = w.npoints
    t_roof = max(ALG_BYTES_PER_POINT_STEP * npts / (hbm_gbs * 1e9), 4 * ALG_FLOP_PER_POINT_STAGE * npts / (fp64_peak_tf * 1e12))
    best = min(ms, ms_graph)
    return {"workload": w.name, "patches": len(w.patches), "points": npts, "ms_per_step": ms,
            "ms_per_step_cuda_graph": ms_graph, "value": npts / (best * 1e-3) / 1e6, "unit": UNIT,
            "frac": t_roof / (best * 1e-3), "launches_per_step": 9 * ((len(w.patches) + 15) // 16),
            "l2": "state %.0f MB" % (n * 8 / 1e6)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index (default 4: 256^3)")
    ap.add_argument("--n", type=int, default=None, help="override the grid size (testing only)")
    ap.add_argument("--oracle-n", type=int, default=None, help="edge of the CPU oracle's sample block")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel (default: the committed ncu capture "
                         "profiles/r03_traffic.json if it was made for the current kernel sources)")
    ap.add_argument("--all-configs", action="store_true", default=True,
                    help="also time BASELINE.json configs 0-3 (default; the headline stays config 4, the line gains `configs`)")
    ap.add_argument("--headline-only", dest="all_configs", action="store_false", help="skip configs 0-3")
    ap.add_argument("--decomp", default=None, metavar="PXxPYxPZ",
                    help="run the sharded path: one block per rank of a periodic domain, halo exchange over NCCL "
                         "(default: replicas, no exchange)")
    ap.add_argument("--overlap", default="off", choices=["on", "off"],
                    help="--decomp: which mode the headline times (the other one is reported under `halo`)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.decomp:
        run_decomp(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
