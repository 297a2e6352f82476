#!/usr/bin/env python
"""bench.py - BASELINE.json's metric on BASELINE.json's headline config.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one pass of the whole hot path (kick, jump, snapshot,
Kepler drift, encounter boxes + pair list, jump, O(N^2) K-weighted pair accelerations, kick)
= one ``mo_step`` over the N=65,536 planetesimal disk (config 3, seed 4; synthetic, recipe
in DESIGN.md).  ``value`` = ordered FP64 pair interactions per second, nb*(nb-1) per step,
with all state resident in HBM; ``e2e`` = the same through ``mo_step_host`` with pinned HOST
buffers (x, v, rcrit up; x, v, pair list, stats down inside the timed region).

The same JSON line carries what north_star asks for beside the headline (rank 0, N = 1 only; each
takes milliseconds to seconds): ``per_config`` (the other four BASELINE.json configs: ms/step, pairs/s,
pair-kernel roofline fractions), ``bigsmall`` (the paper's production regime, N = 1e6 x nbig = 100),
``drift`` (mo_drift alone at nb = 2^24 against the measured HBM bandwidth), ``resolve`` (cost of the
on-device close-encounter solve at the headline config) and ``cpu_baseline`` (the plain-double build
of the oracle on the box's host cores: one thread and all cores, as BASELINE.md plans).

One JSON line on stdout (rank 0).  Under torchrun every rank runs an independent replica
(DESIGN.md section 1 row e: replicas by default; ``--sharded`` times the step of row f4, the pair sum split over the ranks,
instead), timing is the max over ranks, ``value`` the total over ranks.

``--impl reference`` times the CPU oracle (test infrastructure, as it stands; plain-double build, all
host cores) on the same step - a deliberately slow baseline.
"""
from __future__ import annotations

import argparse
import json
import os
import platform
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
# executed FP64 flops per ORDERED pair: the two-sided kernel issues 3 DADD + 6 DMUL + 11 DFMA = 31 flop per
# unordered pair (pair_sym.cuh; the ncu dadd/dmul/dfma counters in profiles/ show the same 3 : 6 : 11 mix);
# the one-sided kernels (pair_accel, pair_big, pair_small) 3 DADD + 5 DMUL + 8 DFMA per ordered pair
EXECUTED_FLOP_PER_PAIR = {"pair_sym_kernel": 15.5, "pair_accel_kernel": 24.0, "pair_big_kernel": 24.0, "pair_small_kernel": 24.0}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the ncu --set full captures
# summarised under profiles/ (the file names its captures); keyed by workload name
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "dram_traffic.json")


def _traffic(workload_name, kernel):
    try:
        t = json.load(open(TRAFFIC_JSON)).get(workload_name, {}).get(kernel)
        return None if t is None else float(t["dram_bytes_read"]) + float(t["dram_bytes_write"])
    except (OSError, ValueError, KeyError):
        return None


def _measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        return {}


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


def _cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return platform.processor() or "unknown"


def oracle_step_time(w, budget_s: float, kind: str = "f64", threads: int = 0, nbig=None):
    """Seconds of ONE hybrid step of workload w by the oracle build `kind` on `threads` host threads (0 = all).
    The whole step (oracle.step: kick, jump, copy, drift, boxes + pair test, jump, pair sum, kick) is run when
    a calibration says it fits the budget; otherwise a bounded sample - R evenly spaced rows of the pair sum
    (each the full ascending-j loop), a strided row sample of the encounter pass, the full O(N) drift -
    scaled up.  Returns (seconds per step, description, threads used)."""
    import oracle
    cores = _host_cores()
    nthr = oracle.set_threads(threads if threads > 0 else cores, kind)
    gm, mu = w.G * w.mass, w.G * w.m_star
    nb = w.nb
    name = {"f64": "plain double", "ld": "x87 long double"}[kind]
    # calibrate on a few rows
    rows = np.unique(np.linspace(0, nb - 1, min(nb, 4 * nthr)).astype(np.int32))
    t0 = time.perf_counter(); oracle.accel_rows(gm, w.x, w.rcrit, rows, kind=kind, nbig=nbig); t1 = time.perf_counter()
    per_row = (t1 - t0) / len(rows)
    if per_row * nb * 1.6 <= budget_s:       # pair sum + encounter pass (about half of it) fit: the real thing
        a0 = np.zeros_like(w.x)
        t0 = time.perf_counter()
        oracle.step(mu, gm, w.rcrit, w.dt, w.x, w.v, a0, cap=1 << 20, kind=kind, nbig=nbig)
        sec = time.perf_counter() - t0
        return sec, f"one full hybrid step (oracle.step, build '{kind}' = {name}, {nthr} thread(s)): {sec:.3f} s", nthr
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
    what = (f"one hybrid step ESTIMATED from {len(rows)} of {nb} pair-sum rows ({t_acc:.2f} s), encounter rows "
            f"i%{stride}==0 ({t_enc:.2f} s) and the full drift ({t_drift:.3f} s); build '{kind}' = {name}, {nthr} thread(s)")
    return est, what, nthr


def cpu_baseline(w, nbig, budget_s: float, with_configs: bool):
    """BASELINE.md's CPU-baseline plan: the plain-double build of the oracle on this box's host cores, (i) one thread,
    (ii) all cores; the long-double parity build (all cores) as a third figure."""
    pairs = _pairs_per_step(w, nbig)
    sec_all, what_all, nthr = oracle_step_time(w, 0.5 * budget_s, "f64", 0, nbig)
    sec_one, what_one, _ = oracle_step_time(w, 0.3 * budget_s, "f64", 1, nbig)
    sec_ld, what_ld, _ = oracle_step_time(w, 0.2 * budget_s, "ld", 0, nbig)
    out = {"value": pairs / sec_all, "unit": UNIT, "cores": nthr, "kind": "oracle", "build": "f64",
           "sample": what_all, "ms_per_step": sec_all * 1e3, "nproc": _host_cores(), "cpu_model": _cpu_model(),
           "single_thread": {"value": pairs / sec_one, "unit": UNIT, "cores": 1, "ms_per_step": sec_one * 1e3, "sample": what_one},
           "long_double_parity_build": {"value": pairs / sec_ld, "unit": UNIT, "cores": nthr, "ms_per_step": sec_ld * 1e3,
                                        "sample": what_ld}}
    if with_configs:
        from paper_2601_19654_b200 import workloads as W
        rows = {}
        for cfg in range(5):
            wc = W.make_config(cfg)
            if wc.name == w.name:
                continue
            pc = _pairs_per_step(wc, None)
            sa, wa, _ = oracle_step_time(wc, 6.0, "f64", 0)
            so, wo, _ = oracle_step_time(wc, 3.0, "f64", 1)
            rows[wc.name] = {"all_cores": {"value": pc / sa, "ms_per_step": sa * 1e3, "sample": wa},
                             "single_thread": {"value": pc / so, "ms_per_step": so * 1e3, "sample": wo}}
        out["per_config"] = rows
    return out


def run_reference(args):
    rank, _, world = _dist_env()
    if rank != 0:
        return 0
    w, nbig = _workload(args)
    pairs = _pairs_per_step(w, nbig)
    budget = max(2.0, min(20.0, 150.0 / max(args.steps + args.warmup, 1)))
    est = []
    what, nthr = "", 0
    for k in range(args.warmup + args.steps):
        e, what, nthr = oracle_step_time(w, budget, "f64", 0, nbig)
        if k >= args.warmup:
            est.append(e)
    sec = sum(est) / len(est)
    val = pairs / sec
    one, what_one, _ = oracle_step_time(w, min(budget, 8.0), "f64", 1, nbig)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nb": w.nb, "nbig": w.nb if nbig is None else nbig, "dt_days": w.dt, "seed": w.seed},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": nthr, "kind": "oracle", "build": "f64", "sample": what,
                             "nproc": _host_cores(), "cpu_model": _cpu_model(),
                             "single_thread": {"value": pairs / one, "unit": UNIT, "cores": 1, "ms_per_step": one * 1e3, "sample": what_one}},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------- GPU leg
def _time_steps(torch, m, w, K, flush, barrier=None):
    """K single mo_step calls, each bracketed by CUDA events on the context's stream, L2 flushed (untimed) before
    each; the pair kernel's own duration from the library's events.  Returns (total ms, pair kernel ms, launches, n)."""
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    m.set_kernel_timing(True)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    n0 = m.launch_count()
    for k in range(K):
        flush.zero_()                       # untimed: evicts the state from L2
        ev[k][0].record(m.stream)
        m.step(w.dt, 1, sync=False)
        ev[k][1].record(m.stream)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    n_launch = m.launch_count() - n0
    pair_ms, n_pair = m.pair_kernel_ms()
    m.set_kernel_timing(False)
    return sum(a.elapsed_time(b) for a, b in ev), pair_ms, n_launch, n_pair


def _pair_roofline(kname, pairs, pair_ms, peak_sust):
    alg = FLOP_PER_PAIR * pairs / (pair_ms * 1e-3) / 1e12
    exe = EXECUTED_FLOP_PER_PAIR[kname] * pairs / (pair_ms * 1e-3) / 1e12
    return alg, exe


def side_config(torch, M, w, nbig, flush, peak_sust, steps_single=5, steps_graph=20, resolve_tol=0.0):
    """One workload beside the headline: ms/step (single steps, L2 flushed, and CUDA-graph replay of a run),
    pairs/s and the pair kernel's roofline fractions."""
    pairs = _pairs_per_step(w, nbig)
    m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=1 << 20)
    if nbig is not None:
        m.set_nbig(nbig)
    if resolve_tol > 0:
        m.set_resolve(resolve_tol)
    kname = m.pair_kernel_name()
    m.step(w.dt, 3, sync=True)
    total_ms, pair_ms, n_launch, n_pair = _time_steps(torch, m, w, steps_single, flush)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m.step(w.dt, 2, sync=True)                                      # builds the graph
    e0.record(m.stream); st = m.step(w.dt, steps_graph, sync=False); e1.record(m.stream); torch.cuda.synchronize()
    g_ms = e0.elapsed_time(e1) / steps_graph
    st = m.stats()
    alg, exe = _pair_roofline(kname, pairs, pair_ms, peak_sust) if pair_ms > 0 else (0.0, 0.0)   # (no kernel time in the resolving step: gated launches)
    out = {"workload": w.name, "N": w.N, "nbig": w.nb if nbig is None else nbig, "ms_per_step": total_ms / steps_single,
           "ms_per_step_graph_replay": g_ms, "pairs_per_s": pairs / (total_ms / steps_single * 1e-3),
           "pairs_per_s_graph_replay": pairs / (g_ms * 1e-3), "pair_kernel": kname, "pair_kernel_ms": pair_ms,
           "frac": alg / peak_sust, "frac_executed": exe / peak_sust, "gpu_launches_per_step": n_launch / steps_single,
           "encounter_pairs_last_step": st.nce_last, "geometry": m.pair_geometry(),
           "traffic": _traffic(w.name, kname)}
    if resolve_tol > 0:
        out["resolve_last_step"] = m.resolve_stats()
        out["resolve_fail_total"] = st.resolve_fail
    m.close()
    del m
    torch.cuda.empty_cache()
    return out


def side_drift(torch, M, W, hbm):
    """HBM roofline of the O(N) Kepler-drift kernel (north_star: 'achieved HBM GB/s for the drift kernel'): mo_drift
    alone at nb = 2^24, where the 96 B/body (x, v read and written) really come from HBM."""
    base = W.make_config(2)
    nb = 1 << 24
    idx = np.arange(nb) % base.nb                     # tile the 16,383-body disk (orbits only matter here)
    m = M.Mopal(np.full(nb, 1e-10), base.x[:, idx].copy(), base.v[:, idx].copy(), np.zeros(nb), m_star=base.m_star, G=base.G, cap=16)
    for _ in range(3):
        m.drift(base.dt)
    n_it = 20
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(m.stream)
    for _ in range(n_it):
        m.drift(base.dt)
    e1.record(m.stream); torch.cuda.synchronize()
    us = e0.elapsed_time(e1) * 1e3 / n_it
    st = m.stats()
    m.close(); del m
    torch.cuda.empty_cache()
    gbs = 96.0 * nb / (us * 1e-6) / 1e9
    return {"kernel": "drift_kernel", "nb": nb, "us_per_launch": us, "algorithmic_bytes_per_body": 96,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm,
                         "traffic": _traffic("drift_nb16777216", "drift_kernel")},
            "bodies_per_s": nb / (us * 1e-6), "drift_fail": st.drift_fail, "max_newton": st.max_newton}


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

    if args.side_only:
        # one of the side measurements alone (short runs for ncu: profiles/README.md names the commands)
        peak = M.probe_fp64_peak(20, with_mean=True)[2]
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{dev}")
        hbm = float(_measured_peaks().get("hbm_gbs", 6550.0))
        name = args.side_only
        if name == "drift":
            out = side_drift(torch, M, W, hbm)
        elif name == "bigsmall":
            out = side_config(torch, M, W.make_bigsmall(1_000_000, 100), 100, flush, peak, 3, 3)
        elif name == "bigsmall_resolve":
            out = side_config(torch, M, W.make_bigsmall(1_000_000, 100), 100, flush, peak, 3, 3, resolve_tol=1e-12)
        elif name == "resolve":
            out = side_config(torch, M, W.make_config(args.config), None, flush, peak, 3, 3, resolve_tol=1e-12)
        else:
            out = side_config(torch, M, W.make_config(int(name[3:])), None, flush, peak, 3, 3)
        print(json.dumps({"side_only": name, **out}), flush=True)
        return 0
    w, nbig = _workload(args)
    nb, pairs = w.nb, _pairs_per_step(w, nbig)
    K, Wm = args.steps, max(args.warmup, 3)
    cap = 1 << 20
    m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=cap, device=f"cuda:{dev}")
    if nbig is not None:
        m.set_nbig(nbig)
    kname = m.pair_kernel_name()
    two_sided = kname == "pair_sym_kernel"
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
    sampler = ClockSampler(dev)
    sampler.start()
    t_s = time.perf_counter()
    while sampler.p is not None and sampler.count() == 0 and time.perf_counter() - t_s < 2.0:
        m.step(w.dt, 1, sync=True)          # nvidia-smi takes ~0.1 s to start: keep the GPU on the same work until it samples
    n_idle = sampler.count()
    st0 = m.stats()
    t_wall0 = time.perf_counter()
    total_ms, pair_ms, n_launch, n_pair = _time_steps(torch, m, w, K, flush, barrier)
    t_wall = time.perf_counter() - t_wall0
    st1 = m.stats()
    # a timed region shorter than a few sampling periods (20 ms): untimed repeats of the same step until 3 samples exist
    t_s = time.perf_counter()
    while sampler.p is not None and sampler.count() < n_idle + 3 and time.perf_counter() - t_s < 1.0:
        m.step(w.dt, 1, sync=True)
    clocks = sampler.stop()
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
    m.close()
    del m

    if rank == 0:
        achieved, executed = _pair_roofline(kname, pairs, pair_ms_max, peak_sust)
        nsm = torch.cuda.get_device_properties(dev).multi_processor_count
        sm_max = clocks.get("sm_max_mhz") or 1965.0
        nominal = nsm * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
        exf = EXECUTED_FLOP_PER_PAIR[kname]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": total_ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nb": nb, "nbig": nb if nbig is None else nbig, "dt_days": w.dt, "seed": w.seed,
                       "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (path does not shard)",
                       "l2": f"flushed (256 MiB memset) between timed steps; the {88 * nb / 1e6:.1f} MB state is otherwise L2-resident",
                       "pair_kernel_geometry": geo, "encounter_pairs_last_step": st1.nce_last},
            # hardware fraction first: FP64 flops the kernel really issues / peak; "effective" = the algorithmic 26 flop per
            # ordered pair of SURVEY.md 8(d), which a kernel that evaluates each unordered pair once can push past 100 %
            "pct_fp64_peak": {"of_measured_sustained": 100 * executed / peak_sust, "of_measured_burst": 100 * executed / peak_burst,
                              "of_nominal": 100 * executed / nominal, "executed_flop_per_ordered_pair": exf,
                              "effective_algorithmic": {"flop_per_pair": FLOP_PER_PAIR, "of_measured_sustained": 100 * achieved / peak_sust,
                                                        "of_nominal": 100 * achieved / nominal}},
            "roofline": {"bound": "alu", "kernel": kname, "achieved": achieved, "peak": peak_sust,
                         "unit": "TFLOP/s", "frac": achieved / peak_sust,
                         "traffic": _traffic(w.name, kname),
                         "note": (f"achieved = the contract's ALGORITHMIC figure: 26 flop per ordered pair (SURVEY.md 8(d)) x nb(nb-1) / kernel "
                                  f"time; the hardware figure is achieved_executed / frac_executed = the {exf} FP64 flop per ordered "
                                  "pair the kernel really issues" + (" (it evaluates each unordered pair once - Newton III - so frac can "
                                  "exceed 1)" if two_sided else "")),
                         "achieved_executed": executed, "frac_executed": executed / peak_sust,
                         "peak_source": "mo_probe_fp64_peak: register-resident DFMA loop on this GPU, 160 launches back to "
                                        "back (sustained); MEASURED_PEAKS.json has no FP64 figure",
                         "peak_burst": peak_burst, "peak_nominal": nominal, "kernel_ms": pair_ms_max, "kernel_launches_timed": n_pair,
                         "kernel_share_of_step": pair_ms_max * n_pair / total_ms_max,
                         "pairs_per_s_kernel": pairs / (pair_ms_max * 1e-3)},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": Ke, "ms_per_step": e2e_ms_max / Ke,
                    "api": "mo_step_host (pinned host x, v, rcrit in; x, v, pairs, stats out)",
                    "note": "a is carried on the device between calls (a_is_current): the first call's extra mo_accel is in the untimed warm-up"},
            "gpu_launches": n_launch,
            "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons", "samples", "power_w_max")},
            "wall_s_timed_region": t_wall,
        }
        if world == 1 and not args.no_side:
            def guarded(fn):
                try:
                    return fn()
                except Exception as e:      # a side line must never cost the headline
                    torch.cuda.empty_cache()
                    return {"error": f"{type(e).__name__}: {e}"}
            hbm = float(_measured_peaks().get("hbm_gbs", 6550.0))
            per = {}
            if not args.bigsmall:
                for cfg in range(5):
                    if cfg != args.config:
                        wc = W.make_config(cfg)
                        per[wc.name] = guarded(lambda: side_config(torch, M, wc, None, flush, peak_sust,
                                                                   steps_graph=100 if cfg < 2 else 10))
                line["per_config"] = per
                line["bigsmall"] = guarded(lambda: side_config(torch, M, W.make_bigsmall(1_000_000, 100), 100, flush, peak_sust))
                line["resolve"] = guarded(lambda: dict(side_config(torch, M, w, None, flush, peak_sust, resolve_tol=1e-12), tol=1e-12,
                                                       note="the headline step with mo_set_resolve(1e-12): the Bulirsch-Stoer "
                                                            "solve of every encounter component inside every step"))
                line["bigsmall_resolve"] = guarded(lambda: dict(side_config(torch, M, W.make_bigsmall(1_000_000, 100), 100, flush, peak_sust,
                                                                            resolve_tol=1e-12), tol=1e-12))
            line["drift"] = guarded(lambda: side_drift(torch, M, W, hbm))
            line["drift"]["peak_source"] = "MEASURED_PEAKS.json hbm_gbs" if _measured_peaks() else "fallback 6550 GB/s"
        if not args.no_cpu and world == 1:
            line["cpu_baseline"] = cpu_baseline(w, nbig, args.cpu_budget, with_configs=not args.bigsmall and not args.no_side)
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_sharded(args):
    """Row f4: ONE system whose O(N^2) pair sum is split over the ranks (strong scaling) - every rank holds the whole
    state, one all-reduce of a (3*ld doubles, NCCL) per step.  Only ever exercised at world 1 on this pool (one GPU per
    call); the driver's own scaling runs use the default replicas."""
    import torch
    rank, local_rank, world = _dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --sharded: no CUDA device")
    dev = local_rank % torch.cuda.device_count()
    torch.cuda.set_device(dev)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", dev))
    from paper_2601_19654_b200 import mopal as M
    from paper_2601_19654_b200.sharded import ShardedMopal
    w, nbig = _workload(args)
    pairs = _pairs_per_step(w, nbig)
    m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=1 << 20, device=f"cuda:{dev}")
    if nbig is not None:
        m.set_nbig(nbig)
    sm = ShardedMopal(m, dist, rank, world)
    K, Wm = args.steps, max(args.warmup, 3)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=m.device)
    sm.step(w.dt, Wm)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    for k in range(K):
        flush.zero_()
        ev[k][0].record(m.stream); sm.step(w.dt, 1, sync=False); ev[k][1].record(m.stream)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    (total_ms_max,) = reduce_max_over_ranks([total_ms], dist, m.device)
    st = m.stats()
    units = m.shard_units()
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": pairs * K / (total_ms_max * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": total_ms_max / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nb": w.nb, "nbig": w.nb if nbig is None else nbig, "dt_days": w.dt, "seed": w.seed,
                       "parallelism": f"pair sum sharded over {world} rank(s): work units {units[0]}, rank 0 takes [{units[1]}, {units[2]}); "
                                      "one all-reduce of a per step; O(N) stages and the encounter pass replicated",
                       "l2": "flushed (256 MiB memset) between timed steps"},
            "allreduces": sm.allreduces, "allreduce_bytes_per_step": 3 * m.ld * 8 if world > 1 else 0,
            "encounter_pairs_last_step": st.nce_last, "gpu_launches": None}), flush=True)
    m.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
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
    ap.add_argument("--sharded", action="store_true", help="row f4: one system, the pair sum split over the ranks (strong scaling)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-side", action="store_true", help="skip per_config / bigsmall / resolve / drift (profiling runs)")
    ap.add_argument("--side-only", default="", metavar="NAME",
                    help="run one side measurement alone: drift, resolve, bigsmall, bigsmall_resolve, cfg0..cfg4 (profiling runs)")
    ap.add_argument("--cpu-budget", type=float, default=20.0, help="seconds of CPU work for the headline cpu_baseline sample")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sharded:
        return run_sharded(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
