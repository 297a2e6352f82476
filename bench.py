#!/usr/bin/env python
"""bench.py - BASELINE.json's metric on BASELINE.json's headline config.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one pass of the whole hot path (kick, jump, snapshot,
Kepler drift, encounter boxes + pair list, jump, O(N^2) K-weighted pair accelerations, kick)
= one ``mo_step`` over the N=65,536 planetesimal disk (config 3, seed 4; synthetic, recipe
in DESIGN.md).  ``value`` = ordered FP64 pair interactions per second, nb*(nb-1) per step,
with all state resident in HBM; ``e2e`` = the same through ``mo_step_host`` with pinned HOST
buffers (x, v, rcrit up; x, v, pair list, stats down inside the timed region).

One JSON line on stdout (rank 0).  The path does not shard (north_star: one GPU): under
torchrun every rank runs an independent replica, timing is the
max over ranks, ``value`` the total over replicas.

``--impl reference`` times the CPU oracle (test infrastructure, as it stands) on the box's
host cores on a bounded sample of the same step - a deliberately slow baseline.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "fp64_pair_interactions_per_s"
UNIT = "pairs/s"
FLOP_PER_PAIR = 26.0          # SURVEY.md 8(d) / DESIGN.md: K = 1 path, per ordered pair
FP64_LANES_PER_SM = 64        # DESIGN.md section "Rooflines": 148 SMs x 64 DFMA/clk x 2 x f
# executed FP64 flops per ORDERED pair of the two-sided kernel: 3 DADD + 6 DMUL + 11 DFMA = 31 flop per
# unordered pair (pair_sym.cuh; the ncu dadd/dmul/dfma counters in profiles/ show the same 3 : 6 : 11 mix)
EXECUTED_FLOP_PER_PAIR = 15.5
# one-sided kernels (pair_accel_kernel, pair_big_kernel): 3 DADD + 5 DMUL + 8 DFMA per ordered pair
EXECUTED_FLOP_PER_PAIR_ONE_SIDED = 24.0
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the pair kernel from the ncu --set full captures:
# pair_sym_kernel at config 3 (profiles/r1f_launches.md: 5.2 MB read + 91.1 MB written),
# pair_big_kernel at --bigsmall 1000000,100 (profiles/r1d_kernels_full.md: 56.0 MB read + 2.9 MB written)
PAIR_KERNEL_DRAM_TRAFFIC_BYTES = {3: 96.3e6, "1000000,100": 58.9e6}


def reduce_max_over_ranks(values, dist=None, device="cpu"):
    """MAX over ranks of a list of floats (timings): the job is as slow as its slowest rank."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def whole_job_value(world: int, units_per_rank_step: float, steps: int, total_ms_max: float) -> float:
    """Replicas only: every rank runs the same independent workload, so the job's throughput is
    world x units per rank over the slowest rank's time."""
    return world * units_per_rank_step * steps / (total_ms_max * 1e-3)


def _dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "20", "-i", str(self.idx)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def count(self) -> int:
        try:
            with open(self.f.name) as g:
                return sum(1 for _ in g)
        except OSError:
            return 0

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [t.strip() for t in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for n, val in zip(names, c[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(pw))
        return out


def _host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


# --------------------------------------------------------------------------- CPU oracle leg
def _workload(args):
    """(workload, nbig or None): BASELINE.json config, or with --bigsmall N,NBIG the paper's production
    regime - SURVEY.md 8(f) row 1, not a BASELINE.json config."""
    from paper_2601_19654_b200 import workloads as W
    if args.bigsmall:
        N, nbig = (int(t) for t in args.bigsmall.split(","))
        return W.make_bigsmall(N, nbig), nbig
    return W.make_config(args.config), None


def _pairs_per_step(w, nbig):
    """ordered (sink i, source j != i) evaluations of one mo_accel"""
    return w.nb * (w.nb - 1) if nbig is None else w.nb * nbig - nbig


def oracle_step_sample(w, budget_s: float, kind: str = "ld", nbig=None):
    """Times the oracle on a bounded sample of ONE hybrid step of workload w and scales it to
    the whole step: R sampled rows of the pair sum (each row is the full ascending-j loop),
    a strided row sample of the encounter pass, and the full O(N) drift.  Returns
    (estimated seconds per full step, description, seconds actually spent)."""
    import oracle
    cores = _host_cores()
    oracle.set_threads(cores)
    gm, mu = w.G * w.mass, w.G * w.m_star
    nb = w.nb
    t_start = time.perf_counter()
    # calibrate on a few rows, then size the sample for the budget
    rows = np.arange(0, nb, max(1, nb // (4 * cores)), dtype=np.int32)[: 4 * cores]
    t0 = time.perf_counter(); oracle.accel_rows(gm, w.x, w.rcrit, rows, kind=kind, nbig=nbig); t1 = time.perf_counter()
    per_row = (t1 - t0) / len(rows)
    R = int(min(nb, max(len(rows), 0.6 * budget_s / max(per_row, 1e-9))))
    rows = np.unique(np.linspace(0, nb - 1, R).astype(np.int32))
    t0 = time.perf_counter(); oracle.accel_rows(gm, w.x, w.rcrit, rows, kind=kind, nbig=nbig); t_acc = time.perf_counter() - t0
    t0 = time.perf_counter(); x1, v1, _ = oracle.drift(mu, w.dt, w.x, w.v, kind=kind); t_drift = time.perf_counter() - t0
    # encounter rows i % stride == 0 see on average the same number of j > i as any other phase
    stride = int(max(1, round(nb / max(len(rows) * 2, 1)))) if nbig is None else 1     # big x all: only nbig rows, all taken
    t0 = time.perf_counter()
    oracle.encounters(w.dt, w.x, w.v, x1, v1, w.rcrit, kind=kind, row_stride=stride, row_phase=0, nbig=nbig, cap=1 << 20)
    t_enc = time.perf_counter() - t0
    est = t_acc * nb / len(rows) + t_enc * stride + t_drift
    what = (f"one hybrid step estimated from {len(rows)} of {nb} pair-sum rows ({t_acc:.2f} s), encounter rows "
            f"i%{stride}==0 ({t_enc:.2f} s) and the full drift ({t_drift:.3f} s); oracle build '{kind}' "
            f"({'x87 long double' if kind == 'ld' else 'plain double'}), OpenMP over rows")
    return est, what, time.perf_counter() - t_start


def run_reference(args):
    rank, _, world = _dist_env()
    if rank != 0:
        return 0
    w, nbig = _workload(args)
    pairs = _pairs_per_step(w, nbig)
    cores = _host_cores()
    budget = max(2.0, min(20.0, 150.0 / max(args.steps + args.warmup, 1)))
    est = []
    what = ""
    for k in range(args.warmup + args.steps):
        e, what, _ = oracle_step_sample(w, budget, nbig=nbig)
        if k >= args.warmup:
            est.append(e)
    sec = sum(est) / len(est)
    val = pairs / sec
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nb": w.nb, "nbig": w.nb if nbig is None else nbig, "dt_days": w.dt, "seed": w.seed},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------- GPU leg
def run_ours(args):
    import torch
    rank, local_rank, world = _dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py: no CUDA device - libmopal has no CPU path (use --impl reference for the oracle)")
    dev = local_rank % torch.cuda.device_count()
    torch.cuda.set_device(dev)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", dev))
    from paper_2601_19654_b200 import mopal as M
    from paper_2601_19654_b200 import workloads as W

    w, nbig = _workload(args)
    nb, pairs = w.nb, _pairs_per_step(w, nbig)
    K, Wm = args.steps, max(args.warmup, 3)
    cap = 1 << 20
    m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=cap, device=f"cuda:{dev}")
    if nbig is not None:
        m.set_nbig(nbig)
    kname = m.pair_kernel_name()
    two_sided = kname == "pair_sym_kernel"
    exec_flop = EXECUTED_FLOP_PER_PAIR if two_sided else EXECUTED_FLOP_PER_PAIR_ONE_SIDED
    stream = m.stream
    geo = m.pair_geometry()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # FP64 issue peak of this GPU: burst (best launch) and sustained (1.5 s train of launches)
    peak_burst, _, peak_sust = M.probe_fp64_peak(160, with_mean=True)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=m.device)   # > 126 MB L2

    # ---- device-resident timing: K steps, L2 flushed between timed steps ------------------
    m.accel()
    for _ in range(Wm):
        m.step(w.dt, 1, sync=False)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    sampler = ClockSampler(dev)
    sampler.start()
    t_s = time.perf_counter()
    while sampler.p is not None and sampler.count() == 0 and time.perf_counter() - t_s < 2.0:
        m.step(w.dt, 1, sync=True)          # nvidia-smi takes ~0.1 s to start: keep the GPU on the same work until it samples
    n_idle = sampler.count()
    st0 = m.stats()
    m.set_kernel_timing(True)
    barrier()
    n0 = m.launch_count()
    t_wall0 = time.perf_counter()
    for k in range(K):
        flush.zero_()                       # untimed: evicts the 5.8 MB state from L2
        ev[k][0].record(stream)
        m.step(w.dt, 1, sync=False)
        ev[k][1].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    n_launch = m.launch_count() - n0
    pair_ms, n_pair = m.pair_kernel_ms()
    m.set_kernel_timing(False)
    st1 = m.stats()
    # a timed region shorter than a few sampling periods (20 ms): untimed repeats of the same step until 3 samples exist
    t_s = time.perf_counter()
    while sampler.p is not None and sampler.count() < n_idle + 3 and time.perf_counter() - t_s < 1.0:
        m.step(w.dt, 1, sync=True)
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = sum(step_ms)
    assert st1.steps_done - st0.steps_done == K and st1.drift_fail == 0, (st0, st1)

    # ---- end to end through the host-buffer entry point ------------------------------------
    ld = m.ld
    xh = torch.zeros((3, ld), dtype=torch.float64).pin_memory(); vh = torch.zeros((3, ld), dtype=torch.float64).pin_memory()
    xh[:, :nb] = torch.from_numpy(w.x); vh[:, :nb] = torch.from_numpy(w.v)
    rh = torch.from_numpy(w.rcrit.copy()).pin_memory()
    ph = torch.zeros((cap, 2), dtype=torch.int32).pin_memory()
    Ke = max(3, min(K, 10))
    m.step_host(w.dt, 1, xh, vh, rcrit_host=rh, a_is_current=False, pairs_host=ph)      # warm-up (computes a first)
    m.step_host(w.dt, 1, xh, vh, rcrit_host=rh, a_is_current=True, pairs_host=ph)
    barrier()
    d2h_pairs = 0
    t0 = time.perf_counter()
    for _ in range(Ke):
        s = m.step_host(w.dt, 1, xh, vh, rcrit_host=rh, a_is_current=True, pairs_host=ph)
        d2h_pairs += 8 * min(s.nce_last, cap)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    h2d = 2 * 3 * ld * 8 + nb * 8
    d2h = 2 * 3 * ld * 8 + 40 + d2h_pairs // Ke

    # ---- max over ranks --------------------------------------------------------------------
    total_ms_max, e2e_ms_max, pair_ms_max = reduce_max_over_ranks([total_ms, t_e2e * 1e3, pair_ms], dist, m.device)
    value = whole_job_value(world, pairs, K, total_ms_max)
    e2e_value = whole_job_value(world, pairs, Ke, e2e_ms_max)

    if rank == 0:
        achieved = FLOP_PER_PAIR * pairs / (pair_ms_max * 1e-3) / 1e12
        executed = exec_flop * pairs / (pair_ms_max * 1e-3) / 1e12
        nsm = torch.cuda.get_device_properties(dev).multi_processor_count
        sm_max = clocks.get("sm_max_mhz") or 1965.0
        nominal = nsm * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": total_ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nb": nb, "nbig": nb if nbig is None else nbig, "dt_days": w.dt, "seed": w.seed,
                       "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (path does not shard)",
                       "l2": f"flushed (256 MiB memset) between timed steps; the {88 * nb / 1e6:.1f} MB state is otherwise L2-resident",
                       "pair_kernel_geometry": geo, "encounter_pairs_last_step": st1.nce_last},
            "pct_fp64_peak": {"of_measured_sustained": 100 * achieved / peak_sust, "of_measured_burst": 100 * achieved / peak_burst,
                              "of_nominal": 100 * achieved / nominal, "flop_per_pair": FLOP_PER_PAIR},
            "roofline": {"bound": "alu", "kernel": kname, "achieved": achieved, "peak": peak_sust,
                         "unit": "TFLOP/s", "frac": achieved / peak_sust,
                         "traffic": PAIR_KERNEL_DRAM_TRAFFIC_BYTES.get(args.bigsmall if nbig is not None else args.config),
                         "note": ("achieved = 26 algorithmic flop per ORDERED pair (SURVEY.md 8(d)) / kernel time; the kernel "
                                  "evaluates each unordered pair once (Newton III), so frac can exceed 1; achieved_executed = "
                                  "the 15.5 flop per ordered pair it really issues (3 DADD + 6 DMUL + 11 DFMA per unordered pair)")
                                 if two_sided else
                                 ("achieved = 26 algorithmic flop per ordered (sink, source) pair (SURVEY.md 8(d)) / kernel time; "
                                  "achieved_executed = the 24 flop per pair it issues (3 DADD + 5 DMUL + 8 DFMA)"),
                         "achieved_executed": executed, "frac_executed": executed / peak_sust,
                         "peak_source": "mo_probe_fp64_peak: register-resident DFMA loop on this GPU, 160 launches back to "
                                        "back (sustained); MEASURED_PEAKS.json has no FP64 figure",
                         "peak_burst": peak_burst, "peak_nominal": nominal, "kernel_ms": pair_ms_max, "kernel_launches_timed": n_pair,
                         "kernel_share_of_step": pair_ms_max * n_pair / total_ms_max,
                         "pairs_per_s_kernel": pairs / (pair_ms_max * 1e-3)},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": Ke, "ms_per_step": e2e_ms_max / Ke, "api": "mo_step_host (pinned host x, v, rcrit in; x, v, pairs, stats out)"},
            "gpu_launches": n_launch,
            "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons", "samples", "power_w_max")},
            "wall_s_timed_region": t_wall,
        }
        if not args.no_cpu and world == 1:
            est, what, _ = oracle_step_sample(w, args.cpu_budget, nbig=nbig)
            line["cpu_baseline"] = {"value": pairs / est, "unit": UNIT, "cores": _host_cores(), "kind": "oracle",
                                    "sample": what, "ms_per_step": est * 1e3}
        print(json.dumps(line), flush=True)
    m.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_drift_sweep(args):
    """HBM roofline of the O(N) Kepler-drift kernel (north_star: 'achieved HBM GB/s for the drift kernel'):
    mo_drift alone at the five configs' sizes, where the state lives in L2, and at nb = 2^24, where
    the 96 B/body (x, v read and written) really come from HBM.  One JSON line."""
    import torch
    from paper_2601_19654_b200 import mopal as M
    from paper_2601_19654_b200 import workloads as W
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    hbm = float(peaks.get("hbm_gbs", 6550.0))
    out = []
    base = W.make_config(2)
    for nb in [255, 4095, 16383, 65535, 131071, 1 << 24]:
        reps = int(np.ceil(nb / base.nb))
        idx = np.arange(nb) % base.nb                     # tile the 16,383-body disk (orbits only matter here)
        x, v = base.x[:, idx].copy(), base.v[:, idx].copy()
        m = M.Mopal(np.full(nb, 1e-10), x, v, np.zeros(nb), m_star=base.m_star, G=base.G, cap=16)
        n_it = 200 if nb < 1 << 20 else 20
        for _ in range(3):
            m.drift(base.dt)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(m.stream)
        for _ in range(n_it):
            m.drift(base.dt)
        e1.record(m.stream); torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / n_it
        st = m.stats()
        out.append({"nb": nb, "us_per_launch": us, "GBps": 96.0 * nb / (us * 1e-6) / 1e9, "bodies_per_s": nb / (us * 1e-6),
                    "drift_fail": st.drift_fail, "max_newton": st.max_newton})
        m.close(); del m, reps
        torch.cuda.empty_cache()
    big = out[-1]
    print(json.dumps({"metric": "drift_kernel_hbm", "kernel": "drift_kernel", "algorithmic_bytes_per_body": 96,
                      "roofline": {"bound": "hbm", "achieved": big["GBps"], "peak": hbm, "unit": "GB/s", "frac": big["GBps"] / hbm,
                                   "at_nb": big["nb"], "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6550"},
                      "sweep": out}), flush=True)
    return 0


def run_support(args):
    """Rooflines of the per-step support routines: mo_energy's pair-potential
    kernel against the FP64 issue peak at the headline config (13 FP64-pipe instructions per unordered
    pair: 3 DADD, 3 DMUL, 6 DFMA, 1 DSETP = 18 flop + 1 compare); mo_hill and the h2dh/dh2h pair against HBM at nb = 2^24
    (mode 0: 32 B in + 8 B out per body; a conversion: 24 B psum pass + 48 B shift pass).  One JSON line."""
    import torch
    from paper_2601_19654_b200 import mopal as M
    from paper_2601_19654_b200 import workloads as W
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    hbm = float(peaks.get("hbm_gbs", 6550.0))

    def timed(m, fn, n):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(m.stream)
        for _ in range(n):
            fn()
        e1.record(m.stream); torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    w = W.make_config(args.config)
    m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=16)
    peak_burst, _, peak_sust = M.probe_fp64_peak(160, with_mean=True)
    ms_en = timed(m, m.energy, 20)
    upairs = w.nb * (w.nb - 1) / 2
    en = {"workload": w.name, "ms": ms_en, "unordered_pairs_per_s": upairs / (ms_en * 1e-3),
          "roofline": {"bound": "alu", "kernel": "energy_pair_kernel", "achieved": 18.0 * upairs / (ms_en * 1e-3) / 1e12,
                       "peak": peak_sust, "unit": "TFLOP/s", "frac": 18.0 * upairs / (ms_en * 1e-3) / 1e12 / peak_sust,
                       "note": "whole mo_energy call (3 kernels + 56 B D2H + sync) over 18 executed flop per unordered pair"}}
    ms_h0 = timed(m, lambda: m.hill(3.0, 0), 200); ms_h1 = timed(m, lambda: m.hill(3.0, 1), 200)
    small = {"nb": w.nb, "hill_mode0_us": ms_h0 * 1e3, "hill_mode1_us": ms_h1 * 1e3,
             "dh2h_us": timed(m, m.dh2h, 200) * 1e3}
    m.close()
    nb = 1 << 24
    base = W.make_config(2)
    idx = np.arange(nb) % base.nb
    m = M.Mopal(np.full(nb, 1e-10), base.x[:, idx].copy(), base.v[:, idx].copy(), np.zeros(nb), m_star=base.m_star, G=base.G, cap=16)
    ms0 = timed(m, lambda: m.hill(3.0, 0), 20)
    ms1 = timed(m, lambda: m.hill(3.0, 1), 20)
    msc = timed(m, m.dh2h, 20)
    big = {"nb": nb,
           "hill_mode0": {"us": ms0 * 1e3, "GBps": 40.0 * nb / (ms0 * 1e-3) / 1e9, "frac": 40.0 * nb / (ms0 * 1e-3) / 1e9 / hbm},
           "hill_mode1": {"us": ms1 * 1e3, "GBps": (32.0 + 64.0) * nb / (ms1 * 1e-3) / 1e9,
                          "frac": (32.0 + 64.0) * nb / (ms1 * 1e-3) / 1e9 / hbm, "bytes_per_body": "psum pass 32 + hill pass 64"},
           "dh2h": {"us": msc * 1e3, "GBps": (32.0 + 48.0) * nb / (msc * 1e-3) / 1e9, "frac": (32.0 + 48.0) * nb / (msc * 1e-3) / 1e9 / hbm,
                    "bytes_per_body": "psum pass 32 (v, gm) + shift pass 48"}}
    m.close()
    print(json.dumps({"metric": "support_routines", "energy": en, "at_config": small, "hbm_bound": big,
                      "hbm_peak_GBps": hbm, "fp64_peak_sustained_TFLOPs": peak_sust}), flush=True)
    return 0


def run_resolve(args):
    """Cost of the on-device close-encounter resolution: mo_step with mo_set_resolve(1e-12)
    against the plain step, graph replay, at configs 0, 1 and 3; the Bulirsch-Stoer work of the last step (bodies,
    accepted steps and right-hand sides summed over the components) and the time per right-hand side it implies.
    The solve is a chain of dependent right-hand sides: latency-bound, no roofline fraction applies.  One JSON line."""
    import torch
    from paper_2601_19654_b200 import mopal as M
    from paper_2601_19654_b200 import workloads as W
    rows = []
    for cfg, nsteps in ((0, 500), (1, 200), (3, 20)):
        nsteps = min(nsteps, args.steps) if args.steps < 100 else nsteps      # --steps 3: a short run for profiling
        w = W.make_config(cfg)
        row = {"workload": w.name}
        for tag, tol in (("plain", 0.0), ("resolved", 1e-12)):
            m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G)
            m.set_resolve(tol)
            m.step(w.dt, 3)
            rhs = 0
            if tol > 0:                      # right-hand sides of the timed steps, counted on single steps of a twin run
                m2 = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G)
                m2.set_resolve(tol); m2.step(w.dt, 3)
                for _ in range(nsteps):
                    m2.step(w.dt, 1); rhs += m2.resolve_stats()["rhs"]
                m2.close()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(m.stream); st = m.step(w.dt, nsteps); e1.record(m.stream); torch.cuda.synchronize()
            row[tag + "_ms_per_step"] = e0.elapsed_time(e1) / nsteps
            if tol > 0:
                row["encounter_pairs_last_step"] = st.nce_last
                row["last_step"] = m.resolve_stats()
                row["rhs_per_step"] = rhs / nsteps
                extra_ms = row["resolved_ms_per_step"] - row["plain_ms_per_step"]
                row["us_per_rhs_longest_chain_bound"] = extra_ms * 1e3 / max(rhs / nsteps, 1)
            m.close()
        rows.append(row)
    print(json.dumps({"metric": "encounter_resolution_cost", "tol": 1e-12, "rows": rows,
                      "note": "us_per_rhs divides by ALL right-hand sides of a step although components run concurrently: "
                              "it is a lower bound on the latency of one right-hand side of the slowest component"}), flush=True)
    return 0


def run_step_sweep(args):
    """Step time (CUDA-graph replay of 1000 steps, CUDA events) of the cfg1 disk recipe at small and middle sizes
    through each launch path the library can take, selected with its MO_* environment switches (read at
    mo_create): the evidence behind the default thresholds in choose_geometry().  One JSON line."""
    import torch
    from paper_2601_19654_b200 import mopal as M
    from paper_2601_19654_b200 import workloads as W
    keys = ("MO_SMALL", "MO_SMALL_MAX", "MO_PSM", "MO_PSM_MAX", "MO_OVERLAP_MIN", "MO_OVERLAP")
    paths = {"default": {},
             "single_cta_front_end+lane_split_pair": {"MO_SMALL_MAX": "1024", "MO_PSM_MAX": "8191"},
             "lane_split_pair+overlap": {"MO_SMALL": "0", "MO_PSM_MAX": "8191", "MO_OVERLAP_MIN": "1"},
             "lane_split_pair": {"MO_SMALL": "0", "MO_PSM_MAX": "8191", "MO_OVERLAP": "0"},
             "tiled_pair+overlap": {"MO_SMALL": "0", "MO_PSM": "0", "MO_OVERLAP_MIN": "1"},
             "tiled_pair (round 1d)": {"MO_SMALL": "0", "MO_PSM": "0", "MO_OVERLAP": "0"}}
    saved = {k: os.environ.get(k) for k in keys}
    rows = []
    for N in [64, 128, 256, 384, 512, 768, 1000, 1536, 2048, 3072, 4096, 8192]:
        w = W.make_config(0) if N == 256 else W.make_config(1) if N == 4096 else W.shrink(1, N)
        row = {"N": N}
        for tag, env in paths.items():
            if tag.startswith("single_cta") and w.nb > 1024:
                continue
            for k in keys:
                os.environ.pop(k, None)
            os.environ.update(env)
            m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G)
            m.step(w.dt, 5)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(m.stream); m.step(w.dt, 1000); e1.record(m.stream); torch.cuda.synchronize()
            row[tag] = round(e0.elapsed_time(e1), 1)          # ms per 1000 steps = us per step
            if tag == "default":
                row["default_pair_kernel"] = m.pair_kernel_name()
            m.close()
        rows.append(row)
    for k, v in saved.items():
        os.environ.pop(k, None)
        if v is not None:
            os.environ[k] = v
    print(json.dumps({"metric": "us_per_step_by_launch_path", "workload": "cfg1 recipe at N (cfg0 at 256)", "rows": rows}), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (3 = N=65,536 headline)")
    ap.add_argument("--bigsmall", default="", metavar="N,NBIG",
                    help="big x all workload (SURVEY.md 8(f) row 1): N objects, NBIG gravity sources, e.g. 1000000,100")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of CPU work for the cpu_baseline sample")
    ap.add_argument("--drift-sweep", action="store_true", help="time mo_drift alone against the HBM roofline and exit")
    ap.add_argument("--support", action="store_true", help="time mo_energy / mo_hill / mo_dh2h against their rooflines and exit")
    ap.add_argument("--step-sweep", action="store_true", help="step time at small / middle N through every launch path and exit")
    ap.add_argument("--resolve", action="store_true", help="cost of the on-device close-encounter resolution and exit")
    args = ap.parse_args()
    if args.resolve:
        return run_resolve(args)
    if args.step_sweep:
        return run_step_sweep(args)
    if args.support:
        return run_support(args)
    if args.drift_sweep:
        return run_drift_sweep(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
