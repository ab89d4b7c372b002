#!/usr/bin/env python
"""bench.py -- PDF evaluations/s (points x flavours, fp64) on B200, BASELINE.json's metric.

A step = one pdf_xfxq2 call over the whole batch of config 3 (NNPDF-shaped grid, 1e8 in-range
points log-uniform in x and Q^2, all 11 flavours), inputs resident in HBM.
`e2e` = the same through pdf_xfxq2_host with pinned HOST buffers (copies inside the timed
region).  `--impl reference` times the CPU oracle on a bounded sample of the same workload.
Multi-GPU (torchrun): every rank evaluates its own 1e8-point shard, no collective on the data
path (points are independent) -> weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2009_06635_b200 import sharding, workloads as W  # noqa: E402

METRIC = "pdf_evaluations_per_sec"
UNIT = "evaluations/s"
N_FULL = 100_000_000


def ncu_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum of one k_xfxq2_smem launch on the config-3 batch, per
    point, read from profiles/r3_traffic.json -- the file the `ncu --set full` capture of that launch is
    turned into (command in profiles/r3_traffic.md).  None if the file is missing: a stale literal in
    this source would not notice a regression, a missing capture is visible."""
    p = os.path.join(ROOT, "profiles", "r3_traffic.json")
    try:
        with open(p) as f:
            t = json.load(f)
        return (float(t["dram_bytes_read"]) + float(t["dram_bytes_write"])) / float(t["points"]), \
            f"profiles/r3_traffic.json ({t.get('source', 'ncu --set full')}; scaled by points)"
    except (OSError, ValueError, KeyError):
        return None, "profiles/r3_traffic.json missing"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs.  NVML is
    initialised in the constructor, so the first sample lands inside even a 60 ms timed region."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self._nv = self._h = None
        try:
            import pynvml as nv
            nv.nvmlInit()
            self._nv, self._h = nv, nv.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(self._h, nv.NVML_CLOCK_SM)
            self._names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
                           nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                           nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
                           nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap"}
        except Exception as exc:  # NVML missing: report, do not fail the bench
            self.reasons.add(f"nvml_unavailable:{type(exc).__name__}")

    def _sample(self):
        nv = self._nv
        self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
        r = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
        for bit, name in self._names.items():
            if r & bit:
                self.reasons.add(name)

    def run(self):
        if self._nv is None:
            return
        try:
            while not self._stop_evt.is_set():
                self._sample()
                time.sleep(0.002)
        except Exception as exc:
            self.reasons.add(f"nvml_error:{type(exc).__name__}")

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def cpu_baseline(grid, x, q2, pids, target_s=12.0):
    """The oracle as it stands, on the first points of the same batch (bounded sample): once with all
    host cores (the reported value) and once with one thread.  The oracle takes its
    coordinate logarithms in binary128 (reading R-ln): slower than a libm-log oracle
    would be, and stated as such."""
    import oracle
    og = oracle.OraclePdfGrid.from_spec(grid)
    cores = oracle.threads()
    m = min(len(x), 200_000)
    t = time.perf_counter()
    og.xfxq2(pids, x[:m], q2[:m])
    rate = m / (time.perf_counter() - t)
    m = int(min(len(x), max(m, rate * target_s)))
    t = time.perf_counter()
    og.xfxq2(pids, x[:m], q2[:m])
    dt = time.perf_counter() - t
    m1 = max(20_000, int(m / cores / 3))          # ~4 s on one thread
    oracle.set_threads(1)
    t = time.perf_counter()
    og.xfxq2(pids, x[:m1], q2[:m1])
    dt1 = time.perf_counter() - t
    oracle.set_threads(cores)
    return {"value": m * len(pids) / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {m} points of the config-3 batch x {len(pids)} flavours, {dt:.1f} s",
            "value_1_thread": m1 * len(pids) / dt1, "sample_1_thread": f"first {m1} points, {dt1:.1f} s",
            "note": "oracle ln = binary128 logq rounded once (reading R-ln): slower than a libm-log oracle"}


def cpu_baseline_other_configs(grid, target_s=2.0):
    """The oracle as it stands on the first points of configs 1, 2, 4 and 5 ("on the first
    min(N, 1e7) points of each of the five configs", one thread and all cores) -- bounded to about
    `target_s` seconds per config and thread count so that the default run stays within minutes; the
    sample is stated.  Evaluations (points x flavours) per second."""
    import oracle
    cores = oracle.threads()
    p11 = list(W.PIDS_11)
    g1 = W.grid_config1()
    x1, x2, qe = W.queries_mc_events(grid, 10_000_000)
    cases = {
        "config1_1e4x3": (oracle.OraclePdfGrid.from_spec(g1), list(W.PIDS_3), 10_000) + W.queries_in_range(g1, 10_000, 1),
        "config2_1e6x11": (oracle.OraclePdfGrid.from_spec(grid), p11, 1_000_000) + W.queries_in_range(grid, 1_000_000, 2),
        "config4_mix_1e7x11": (oracle.OraclePdfGrid.from_spec(grid), p11, 10_000_000) + W.queries_extrapolation_mix(grid, 10_000_000),
        "config5_1e7_events": (oracle.OraclePdfGrid.from_spec(grid), p11, 10_000_000, x1, qe),
    }
    res = {}
    for name, (og, pids, n_full, x, q2) in cases.items():
        e = {"unit": UNIT, "kind": "oracle", "cores": cores}
        for threads, key in ((cores, "value"), (1, "value_1_thread")):
            oracle.set_threads(threads)
            m = min(n_full, 20_000)
            t = time.perf_counter(); og.xfxq2(pids, x[:m], q2[:m]); rate = m / (time.perf_counter() - t)
            m = int(min(n_full, max(m, rate * target_s)))
            t = time.perf_counter(); og.xfxq2(pids, x[:m], q2[:m]); dt = time.perf_counter() - t
            e[key] = m * len(pids) / dt
            e["sample" if threads != 1 else "sample_1_thread"] = f"first {m} of {n_full} points x {len(pids)} flavours, {dt:.1f} s"
        oracle.set_threads(cores)
        res[name] = e
    res["config5_1e7_events"]["note"] = "the x1 leg of the events (the x2 leg and alpha_s cost the oracle the same per point / far less)"
    return res


def parity_population(torch, out_d, grid, x_h, q2_h, pids, chunk=10_000_000):
    """--parity: EVERY output of the timed batch against the oracle ("parity is
    checked on all points", config 3 in 1e7-point chunks): max eq.-1 difference,
    outputs breaking the 1e-12 / 1e-15 rule, outputs that needed the conditioning clause."""
    import oracle
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity_util import check_parity_population
    og = oracle.OraclePdfGrid.from_spec(grid)
    t = time.perf_counter()
    st = check_parity_population(lambda a, b: out_d[:, a:b].cpu().numpy(), og, pids, x_h, q2_h, chunk=chunk,
                                 max_clause_frac=2e-3, what="bench --parity, config 3 all points")
    st["seconds"] = time.perf_counter() - t
    st["rule"] = "|d| <= 1e-12 |ref|, or |d| <= 1e-15 where |ref| < 1e-3; clause |d| <= 1e-12 S (DESIGN.md 5)"
    return st


def run_reference(args):
    """--impl reference: the CPU oracle on the box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    grid = W.grid_nnpdf_shaped()
    pids = list(W.PIDS_11)
    m = args.ref_points
    x, q2 = W.queries_in_range(grid, m, 3)
    og = oracle.OraclePdfGrid.from_spec(grid)
    for _ in range(args.warmup):
        og.xfxq2(pids, x[: m // 10], q2[: m // 10])
    t = time.perf_counter()
    for _ in range(args.steps):
        og.xfxq2(pids, x, q2)
    dt = (time.perf_counter() - t) / args.steps
    val = m * len(pids) / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config3: NNPDF-shaped grid 100x(7+14+23+20)x11, in-range log-uniform points, 11 flavours",
                       "points_per_step": m, "note": "each step is a bounded sample of the 1e8-point batch"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle",
                             "sample": f"{m} points x 11 flavours per step"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# Algorithmic FP64-pipe instruction counts per point, frozen in SURVEY.md 8(d) (FMA = 1):
#   in range W(F) = 2*28 + 32 + 16 + 16 F;  rules A / B ~ 120 + 120 F;  rule C ~ 136 + 110 F
def w_in(F):
    return 2 * 28 + 32 + 16 + 16 * F


def w_ab(F):
    return 120 + 120 * F


def w_c(F):
    return 136 + 110 * F


def w_config4(F):
    """Mix of reading Q14: 70 % in range, 20 % rule A, 5 % Q above / 5 % Q below the grid with x
    log-uniform on [1e-12, 1], i.e. a quarter of each in the corner (the Q^2 rule on two rule-A values)."""
    return 0.70 * w_in(F) + 0.20 * w_ab(F) + 0.0375 * w_ab(F) + 0.0125 * 2 * w_ab(F) + 0.0375 * w_c(F) + 0.0125 * (w_c(F) + w_ab(F))


def roofline_entry(ms, n_points, bytes_per_point, w_per_point, hbm_gbs, fma_per_s):
    """Fractions of the two contract bounds and of the slower one (north_star: "the roofline is the
    slower of two bounds")."""
    t = ms * 1e-3
    t_hbm, t_fp64 = bytes_per_point * n_points / (hbm_gbs * 1e9), w_per_point * n_points / fma_per_s
    return {"hbm_frac": t_hbm / t, "fp64_frac": t_fp64 / t, "bound": "hbm" if t_hbm >= t_fp64 else "fp64",
            "roofline_ms": max(t_hbm, t_fp64) * 1e3, "roofline_frac": max(t_hbm, t_fp64) / t,
            "fp64_ops_per_point": w_per_point, "bytes_per_point": bytes_per_point}


def timed_reps(torch, fn, reps=20, warm=3):
    """Median and best of `reps` CUDA-event timings of fn() on the current stream."""
    for _ in range(warm):
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for a, b in ev:
        a.record(); fn(); b.record()
    torch.cuda.synchronize()
    ts = sorted(a.elapsed_time(b) for a, b in ev)
    return {"ms": float(np.median(ts)), "ms_best": ts[0], "reps": reps}


def graph_replay_ms(torch, fn, per_graph=20, reps=10):
    """Device time of one fn() when `per_graph` of them are captured into ONE CUDA graph and replayed:
    what a launch-latency-sized call costs inside a captured loop (the calls allocate nothing and never
    synchronise, so they can be captured).  Median over `reps` replays, per call."""
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        fn()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        for _ in range(per_graph):
            fn()
    g.replay()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for a, b in ev:
        a.record(); g.replay(); b.record()
    torch.cuda.synchronize()
    return float(np.median([a.elapsed_time(b) for a, b in ev])) / per_graph


def bench_other_configs(torch, B, h, ha, grid, peak, fma_per_s, graph=True):
    """Configs 1, 2, 4 and 5 of BASELINE.json at their full sizes, device-resident, reported beside
    the metric (parity-test cases, not the headline): median and best of 20 CUDA-event timings, each
    with its fraction of the slower contract bound."""
    def dev(*arrs):
        return [torch.from_numpy(a).cuda() for a in arrs]

    def entry(t, n_points, F, bpp, w, **extra):
        e = dict(t)
        e["evaluations_per_s"] = n_points * F / (t["ms"] * 1e-3)
        e.update(roofline_entry(t["ms"], n_points, bpp, w, peak, fma_per_s))
        e.update(extra)
        return e

    res, p11 = {}, list(W.PIDS_11)
    g1 = W.grid_config1()
    h1 = B.load_pdf_spec(g1)
    x, q2 = dev(*W.queries_in_range(g1, 10_000, 1))
    o = torch.empty((3, 10_000), dtype=torch.float64, device="cuda")
    f1 = lambda: B.pdf_xfxq2(h1, list(W.PIDS_3), x, q2, o)
    gr = (lambda f: {"ms_in_cuda_graph": graph_replay_ms(torch, f)}) if graph else (lambda f: {})
    res["config1_1e4x3"] = entry(timed_reps(torch, f1), 10_000, 3, 40, w_in(3), note="launch-latency sized", **gr(f1))
    B.pdf_grid_free(h1)
    x, q2 = dev(*W.queries_in_range(grid, 1_000_000, 2))
    o = torch.empty((11, 1_000_000), dtype=torch.float64, device="cuda")
    f2 = lambda: B.pdf_xfxq2(h, p11, x, q2, o)
    res["config2_1e6x11"] = entry(timed_reps(torch, f2), 1_000_000, 11, 104, w_in(11), **gr(f2))
    n4 = 10_000_000
    x, q2 = dev(*W.queries_extrapolation_mix(grid, n4))
    o = torch.empty((11, n4), dtype=torch.float64, device="cuda")
    res["config4_mix_1e7x11"] = entry(timed_reps(torch, lambda: B.pdf_xfxq2(h, p11, x, q2, o)), n4, 11, 104, w_config4(11))
    res["config4_mix_1e7x1"] = entry(timed_reps(torch, lambda: B.pdf_xfxq2(h, [21], x, q2, o)), n4, 1, 24, w_config4(1))
    # the two output variants of SURVEY.md 8(f).4 on the same batch
    opm = torch.empty((n4, 11), dtype=torch.float64, device="cuda")
    o32 = torch.empty((11, n4), dtype=torch.float32, device="cuda")
    res["config4_mix_1e7x11_point_major"] = entry(timed_reps(torch, lambda: B.pdf_xfxq2_pm(h, p11, x, q2, opm), reps=10), n4, 11, 104, w_config4(11))
    res["config4_mix_1e7x11_fp32_out"] = entry(timed_reps(torch, lambda: B.pdf_xfxq2_f32(h, p11, x, q2, o32), reps=10), n4, 11, 60, w_config4(11))
    del opm, o32
    x1, x2, q2 = dev(*W.queries_mc_events(grid, n4))
    o2 = torch.empty((11, n4), dtype=torch.float64, device="cuda")
    oa = torch.empty(n4, dtype=torch.float64, device="cuda")

    def events():
        B.pdf_xfxq2(h, p11, x1, q2, o); B.pdf_xfxq2(h, p11, x2, q2, o2); B.alphas_q2(ha, q2, oa)
    t = timed_reps(torch, events)
    res["config5_1e7_events"] = entry(t, 2 * n4, 11, 104 + 8, w_in(11) + 24, events_per_s=n4 / (t["ms"] * 1e-3),
                                      calls="pdf_xfxq2(x1), pdf_xfxq2(x2), alphas_q2 on the shared Q^2 (per PDF point: 104 B + half of alpha_s' 16 B)")
    # the fused call (luminosity sum over 11 flavour pairs + alpha_s), one number per event out
    terms = [(q, -q, 1.0) for q in (1, 2, 3, 4, 5)] + [(-q, q, 1.0) for q in (1, 2, 3, 4, 5)] + [(21, 21, 0.25)]
    lum = torch.empty(n4, dtype=torch.float64, device="cuda")
    t = timed_reps(torch, lambda: B.pdf_lumi_events(h, terms, x1, x2, q2, lum, alphas=ha, alphas_out=oa))
    w_ev = 3 * 28 + 3 * 16 + 2 * (16 + 16 * 11) + 2 * 11 * 11 + 48   # 3 ln, 3 weight sets, 2 x (outer product + contraction), bilinear form, alpha_s
    e = dict(t)
    e.update(roofline_entry(t["ms"], n4, 24 + 16, w_ev, peak, fma_per_s))
    e.update({"events_per_s": n4 / (t["ms"] * 1e-3), "evaluations_per_s": 22 * n4 / (t["ms"] * 1e-3),
              "speedup_vs_three_launches": res["config5_1e7_events"]["ms"] / t["ms"],
              "calls": "pdf_lumi_events(x1, x2, Q^2) with alpha_s: 40 B per event of HBM traffic instead of 240 + 176 + the consumer's 176",
              "onchip_gather_bound_ms": 2 * 16 * 12 * 8 * n4 / (128 * 148 * 1.965e9) * 1e3})
    res["config5_fused_lumi"] = e
    return res


def bench_members(torch, B, local, n_rep, hbm_gbs=None, lds_bps=None, fma_per_s=None):
    """SURVEY.md 8(f).1 / PAPER.md:171-190, Table 2: all 13 flavours of N_rep members on a 2415-point
    x-grid, one pdf_xfxq2_members launch; reported beside the metric, not inside it."""
    g0 = W.grid_member(0)
    vals = W.member_values(n_rep)
    hs = B.pdf_set_load(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, vals, device=local)
    pids = list(W.PIDS_13)
    x, q2 = W.queries_fk_xgrid(g0)
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    out = torch.empty((n_rep, len(pids), len(x)), dtype=torch.float64, device="cuda")
    for _ in range(3):
        B.pdf_xfxq2_members(hs, 0, n_rep, pids, dx, dq, out)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(10):
        B.pdf_xfxq2_members(hs, 0, n_rep, pids, dx, dq, out)
    b.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b) / 10
    B.pdf_grid_free(hs)
    ev = n_rep * len(pids) * len(x)
    # Algorithmic traffic of the launch: all points sit at the grid's lowest scale, so a member's stencils
    # touch table rows 0..3 of the 64 (rows -1..2 of Q^2 interval 0 plus the head of row 3) in each of its
    # 4 flavour-group slices -- 4 rows x 100 knots x 32 B -- read once; the points are read once per job
    # (L2-resident after the first), the outputs written once.
    n_groups, rows_needed, row_bytes = 4, 4, 100 * 32
    bytes_alg = n_rep * n_groups * rows_needed * row_bytes + 16 * len(x) + 8 * ev
    t = ms * 1e-3
    roof = None
    if hbm_gbs and lds_bps and fma_per_s:
        # three bounds of one launch: HBM on the algorithmic bytes, the on-chip stencil gather (one 4-column
        # group = 128 B x 4 rows per point: 16 LDS.128; 4 groups hold 13 + 3 padding columns) and FP64
        # (per job and point: two weight sets from the cached t, tau ~ 40 FMA, 4 x 20 contraction)
        t_hbm = bytes_alg / (hbm_gbs * 1e9)
        gather_bytes = n_rep * n_groups * len(x) * 4 * 128
        t_gather = gather_bytes / lds_bps
        t_fp64 = n_rep * n_groups * len(x) * (40 + 80) / fma_per_s
        b = max((t_gather, "smem"), (t_hbm, "hbm"), (t_fp64, "alu"))
        roof = {"bound": b[1], "frac": b[0] / t, "roofline_ms": b[0] * 1e3, "hbm_frac": t_hbm / t, "smem_frac": t_gather / t,
                "fp64_frac": t_fp64 / t, "achieved": gather_bytes / t / 1e9, "peak": lds_bps / 1e9, "unit": "GB/s",
                "peak_source": "measured: pdfb_probe(PDFB_PROBE_LDS), conflict-free LDS.128",
                "note": "the launch moves 0.06 of a slice per job, so the stencil gather from shared memory, not HBM, bounds it"}
    paper = {10: 0.07, 50: 0.35, 100: 0.69, 200: 1.46, 300: 1.29, 400: 1.69}.get(n_rep)
    return {"n_rep": n_rep, "flavours": len(pids), "points": len(x), "ms": ms, "evaluations_per_s": ev / (ms * 1e-3),
            "algorithmic_bytes": bytes_alg, "algorithmic_gbs": bytes_alg / t / 1e9, "roofline": roof,
            "paper_pdfflow_gpu_s": paper, "paper_hardware": "system P1 (Titan V / RTX 2080 Ti), PAPER.md:179-188: context, another machine",
            "workload": "synthetic member tables on the NNPDF-shaped knots (workloads.member_values)"}


def run_gpu(args):
    import torch
    from paper_2009_06635_b200 import binding as B, build
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference "
                         "for the oracle baseline)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    B.lib()

    grid = W.grid_nnpdf_shaped()
    pids = list(W.PIDS_11)
    F = len(pids)
    n = args.points
    h = B.load_pdf_spec(grid, device=local)
    # every rank draws its own shard (seed offset by rank): weak scaling, no collective
    x_h, q2_h = W.queries_in_range(grid, n, sharding.rank_seed(3, rank))
    x_d, q2_d = torch.from_numpy(x_h).cuda(), torch.from_numpy(q2_h).cuda()
    out_d = torch.empty((F, n), dtype=torch.float64, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        B.pdf_xfxq2(h, pids, x_d, q2_d, out_d)

    sampler = ClockSampler(local)  # NVML initialised here, outside the timed region
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches0 = B.launch_count()
    barrier()
    t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
    t0.record()
    for k, (a, b) in enumerate(evs):
        a.record(); step(); b.record()
        if k == 0:
            sampler.start()  # the GPU is busy from here to t1: every sample is under load
    t1.record()
    barrier()
    launches = B.launch_count() - launches0
    clocks = sampler.stop()
    total_ms = t0.elapsed_time(t1)
    per_step = sorted(a.elapsed_time(b) for a, b in evs)
    kern_ms, kern_med, kern_best = float(np.mean(per_step)), float(np.median(per_step)), per_step[0]
    total_ms, kern_ms, kern_med, kern_best = sharding.reduce_max([total_ms, kern_ms, kern_med, kern_best], dist, "cuda")
    ms_per_step = total_ms / args.steps
    value = sharding.aggregate_throughput([n * F] * world, [ms_per_step])

    # ---- end to end: pinned host buffers through pdf_xfxq2_host, copies inside the timed region.
    # Every rank takes part (the value is the whole job's); the pinned buffers of all ranks together
    # stay at one config-3 batch (10.4 GB), whatever the rank count.
    e2e = None
    if not args.no_e2e:
        n_e, n_e_all = sharding.e2e_split(args.e2e_points, rank, world, n)
        xp = torch.from_numpy(x_h[:n_e]).pin_memory(); qp = torch.from_numpy(q2_h[:n_e]).pin_memory()
        op = torch.empty((F, n_e), dtype=torch.float64).pin_memory()
        B.pdf_xfxq2_host(h, pids, xp, qp, op)
        barrier()
        ks = max(1, min(args.steps, 3))
        tw = time.perf_counter()
        for _ in range(ks):
            B.pdf_xfxq2_host(h, pids, xp, qp, op)  # synchronous: returns when `out` is complete
        barrier()
        e_s = (time.perf_counter() - tw) / ks
        e_s = sharding.reduce_max_ms(e_s * 1e3, dist, "cuda") * 1e-3
        e2e = {"value": sharding.aggregate_throughput([n_e_all * F], [e_s * 1e3]), "unit": UNIT, "h2d_bytes_per_step": 16 * n_e_all,
               "d2h_bytes_per_step": 8 * F * n_e_all, "points_per_step": n_e_all, "ms_per_step": e_s * 1e3,
               "api": "pdf_xfxq2_host (pinned host buffers, 3-stage copy/compute pipeline)"}
        del xp, qp, op

    if rank != 0:
        B.pdf_grid_free(h)
        if dist is not None:
            dist.destroy_process_group()
        return
    # ---- alpha_s (row S8), reported beside the metric, not inside it
    aspec = W.make_alphas_grid()
    ha = B.load_alphas_spec(aspec, device=local)
    a_out = torch.empty(n, dtype=torch.float64, device="cuda")
    a_t = timed_reps(torch, lambda: B.alphas_q2(ha, q2_d, a_out))
    peak, peak_src = measured_peaks()
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    # measured denominators for the two bounds MEASURED_PEAKS.json does not carry (pdfb_probe)
    lds_bps, fma_ps = B.probe(B.PROBE_LDS, local), B.probe(B.PROBE_FP64, local)
    bytes_per_launch = (16 + 8 * F) * n
    achieved = bytes_per_launch / (kern_ms * 1e-3) / 1e9
    w_f = w_in(F)
    t_hbm, t_fp64, t_gather = bytes_per_launch / (peak * 1e9), w_f * n / fma_ps, 128.0 * F * n / lds_bps
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config3: NNPDF-shaped grid 100x(7+14+23+20)x11 PIDs, in-range points "
                                   "log-uniform in x and Q2, all 11 flavours, flavour-major output",
                       "points_per_gpu": n, "flavours": F, "l2_policy": "inputs+outputs per step "
                       f"({bytes_per_launch / 1e9:.2f} GB) exceed the 126 MB L2; no flush needed",
                       "grid_setup_ms": B.pdf_grid_setup_ms(h)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": (ncu_traffic()[0] * n / 1e9) if F == 11 and ncu_traffic()[0] else None, "traffic_unit": "GB per launch",
                         "traffic_source": ncu_traffic()[1],
                         "kernel": "k_xfxq2_smem" if B.pdf_grid_uses_smem_path(h) else "k_xfxq2_v0", "kernel_ms": kern_ms,
                         "kernel_ms_median": kern_med, "kernel_ms_best": kern_best,
                         "algorithmic_bytes_per_point": 16 + 8 * F, "peak_source": peak_src,
                         # the same launch against the other contract bound and against the bound the design
                         # actually runs into: every gathered table byte crosses the SM's
                         # 128 B/clk shared-memory pipe, 16 x 8 B x F per point, measured peak (pdfb_probe)
                         "fp64_frac": t_fp64 / (kern_ms * 1e-3), "slower_contract_bound": "hbm" if t_hbm >= t_fp64 else "fp64",
                         "bound_onchip_ms": t_gather * 1e3, "bound_onchip_frac": t_gather / (kern_ms * 1e-3),
                         "bound_onchip_as_roofline_frac": max(t_hbm, t_fp64) / t_gather,
                         "bound_onchip_note": "a per-point gather cannot run faster than bound_onchip_ms: at most "
                                              "bound_onchip_as_roofline_frac of the contract roofline (DESIGN.md 6)"},
            "onchip_gather": {"bound": "smem", "achieved": 128 * F * n / (kern_ms * 1e-3) / 1e9, "peak": lds_bps / 1e9,
                              "peak_nominal": sms * 128 * (clocks["sm_mhz"] or 1965.0) * 1e6 / 1e9, "unit": "GB/s",
                              "frac": t_gather / (kern_ms * 1e-3), "algorithmic_bytes_per_point": 128 * F,
                              "peak_source": "measured: pdfb_probe(PDFB_PROBE_LDS), conflict-free LDS.128",
                              "note": "context only; the contract roofline is `roofline` (HBM)"},
            "fp64": {"bound": "alu", "achieved": w_f * n / (kern_ms * 1e-3) / 1e12, "peak": fma_ps / 1e12,
                     "unit": "T FP64 op/s (FMA = 1)", "frac": t_fp64 / (kern_ms * 1e-3),
                     "algorithmic_ops_per_point": w_f, "peak_source": "measured: pdfb_probe(PDFB_PROBE_FP64), DFMA chains",
                     "note": "context only; HBM is the slower of the two contract bounds"},
            "alphas": {"points": n, "ms": a_t["ms"], "ms_best": a_t["ms_best"], "evaluations_per_s": n / (a_t["ms"] * 1e-3),
                       **roofline_entry(a_t["ms"], n, 16, 48, peak, fma_ps)}}
    if not args.no_other_configs:
        line["other_configs"] = bench_other_configs(torch, B, h, ha, grid, peak, fma_ps, graph=not args.no_graph)
    B.alphas_grid_free(ha)
    if not args.no_members:
        line["multi_member"] = bench_members(torch, B, local, args.members, peak, lds_bps, fma_ps)
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(grid, x_h, q2_h, pids)
        if not args.no_other_configs:
            for name, e in cpu_baseline_other_configs(grid).items():
                line["other_configs"][name]["cpu_baseline"] = e
    if args.parity:
        step()
        torch.cuda.synchronize()
        line["parity"] = parity_population(torch, out_d, grid, x_h, q2_h, pids)
    B.pdf_grid_free(h)
    if dist is not None:
        dist.destroy_process_group()
    print(json.dumps(line), flush=True)


def run_leg(args):
    """--leg NAME: one named workload, --warmup + --steps launches and nothing else -- the command the ncu
    captures under profiles/ were taken with (one kernel family per capture)."""
    import torch
    from paper_2009_06635_b200 import binding as B, build
    build.build()
    grid = W.grid_nnpdf_shaped()
    h = B.load_pdf_spec(grid)
    p11 = list(W.PIDS_11)
    dev = lambda *arrs: [torch.from_numpy(a).cuda() for a in arrs]
    n4 = 10_000_000
    if args.leg in ("config4", "config4_f1"):
        x, q2 = dev(*W.queries_extrapolation_mix(grid, n4))
        pids = p11 if args.leg == "config4" else [21]
        o = torch.empty((len(pids), n4), dtype=torch.float64, device="cuda")
        fn = lambda: B.pdf_xfxq2(h, pids, x, q2, o)
    elif args.leg == "lumi":
        x1, x2, q2 = dev(*W.queries_mc_events(grid, n4))
        terms = [(q, -q, 1.0) for q in (1, 2, 3, 4, 5)] + [(-q, q, 1.0) for q in (1, 2, 3, 4, 5)] + [(21, 21, 0.25)]
        lum = torch.empty(n4, dtype=torch.float64, device="cuda")
        fn = lambda: B.pdf_lumi_events(h, terms, x1, x2, q2, lum)
    elif args.leg == "alphas":
        ha = B.load_alphas_spec(W.make_alphas_grid())
        (q2,) = dev(W.queries_in_range(grid, args.points, 3)[1])
        o = torch.empty_like(q2)
        fn = lambda: B.alphas_q2(ha, q2, o)
    elif args.leg == "members":
        g0 = W.grid_member(0)
        hs = B.pdf_set_load(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, W.member_values(args.members))
        x, q2 = dev(*W.queries_fk_xgrid(g0))
        o = torch.empty((args.members, 13, len(x)), dtype=torch.float64, device="cuda")
        fn = lambda: B.pdf_xfxq2_members(hs, 0, args.members, list(W.PIDS_13), x, q2, o)
    else:
        raise SystemExit(f"unknown --leg {args.leg}")
    t = timed_reps(torch, fn, reps=args.steps, warm=max(args.warmup, 1))
    print(json.dumps({"leg": args.leg, **t}), flush=True)


def relaunch_ranks(args):
    """`python bench.py --gpus N` without torchrun: start the N ranks ourselves (one process per GPU,
    rendezvous on 127.0.0.1), with the same arguments."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--points", type=int, default=N_FULL, help="points per GPU (config 3: 1e8)")
    ap.add_argument("--e2e-points", type=int, default=N_FULL, help="points of the end-to-end leg, all ranks together")
    ap.add_argument("--ref-points", type=int, default=2_000_000, help="oracle sample per step")
    ap.add_argument("--parity", action="store_true", help="check every output of the batch against the oracle (~2 min)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-members", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="skip the CUDA-graph replay timings of configs 1 and 2 (the ncu launch list)")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--members", type=int, default=400, help="N_rep of the multi-member leg (Table 2)")
    ap.add_argument("--leg", default=None, help="profiling aid: run only config4 | config4_f1 | lumi | alphas | members")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.leg:
        run_leg(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_ranks(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
