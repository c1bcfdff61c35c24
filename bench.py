#!/usr/bin/env python
"""Benchmark of the TCR-NET hot path on B200 (contract: see DESIGN.md section 8).

A "step" is one pass of the whole hot path over one batch of synthetic input:
A1 pack -> A2 schedule -> A3/A4 distances with early exit -> A5 emission -> A6 sort/CSR/degrees.
Workload at N=1 GPU: BASELINE.json configs[3] ("cfg4": N = 800,000 CDR3-beta-shaped sequences,
l_max = 1), the configuration the metric is quoted on.

  value : N(N-1)/2 pairs decided per second, raw inputs already resident in HBM, device-timed.
  e2e   : the same through the C ABI with HOST buffers (tcrnet_load H2D + build + tcrnet_copy_csr
          D2H inside the timed region, wall clock between synchronisations).
  roofline : the distance kernel against the INT32 ALU-pipe peak.
  cpu_baseline : the oracle, as it stands, on this box's host cores, on a bounded sample.

`--impl reference` times the oracle alone (rank 0 only).  N > 1: one process per GPU, each rank
builds an independent repertoire of the same shape (replicas, no data-path collective): weak.
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

WORKLOAD = "cfg4"
ALU_LANES_PER_SM = 64          # INT32 ALU-pipe lanes per SM per clock on sm_100
# prefix-trie / text-chunk kernels (Myers column recurrence), DESIGN.md section 7
ALU_OPS_PER_COLUMN = 7         # LOP3 per pair and text column (distance.cu)
ALU_OPS_FIRST_COLUMN = 3       # the first column of a text needs only 3 (constant Pv, Mv = 0)
ALU_OPS_PER_TEST = 4           # 2 LOP3 + IADD3 + ISETP per pair and early-exit test
ALU_OPS_PER_PREFIX_TEST = 2    # LOP3 + ISETP per pair and DP cell read in a guided expansion (distance_trie.cu)
# segment join (segjoin.cu): what the method itself needs on the ALU pipe
JOIN_OPS_PER_PROBE = 25        # 5 plane slices x (SHF + AND + XOR) + the 64-bit xor-shifts of the mixing rounds
JOIN_OPS_PER_ENTRY = 16        # per directory entry read: segment-number compare (2), composition distance of the two
                               # signature words (13: SWAR subtract / sign / fold, its 2 multiplies and the POPC not
                               # counted), order compare (1)
JOIN_OPS_PER_CANDIDATE = 12    # widening the 5 text planes (2 x 5) + the filter's AND / compare
JOIN_OPS_PER_DIAGONAL = 11     # 5 funnel shifts + 5 LOP3 (a ^ b | acc) + 1 AND of the shifted-Hamming filter
JOIN_OPS_PER_LV_STATE = 12     # Landau-Vishkin: compare / select / max / min / shift per (edit level, diagonal)
ORACLE_SAMPLE_ROWS = 1024
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the ncu --set full captures
# summarised under profiles/ (regenerated with them; a workload / kernel that is not listed prints null)
NCU_DRAM_BYTES_PER_LAUNCH = {
    # (workload, kernel): bytes per step of that kernel / kernel pair - profiles/r2_join_ncu.txt
    ("cfg4", "k_join_probe"): 30_912_000 + 5_376,
    ("cfg3", "k_join_probe + k_join_verify"): 9_013_760 + 0 + 11_579_648 + 0,
    ("cfg5", "k_join_probe + k_join_verify"): 1_270_189_000 + 288_741_376 + 368_049_000 + 52_908_544,
}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """SM clock / throttle reasons during the timed region (B200_PROFILING.md recipe).  The timed region
    of this path is tens of milliseconds, far below nvidia-smi's shortest loop, so the sampler polls NVML
    in-process (the same counters nvidia-smi prints) every ~1 ms; nvidia-smi -lms is the fallback."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []      # (t, sm_mhz, set of reasons)
        self.sm_max = None
        self.stop_flag = False
        self.proc = None
        self.source = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and all(x.strip().isdigit() for x in vis.split(",")) else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nv = pynvml
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.source = "nvml"
            self.thread = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nv = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.source = "nvidia-smi"
            self.thread = threading.Thread(target=self._pump_smi, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _poll_nvml(self):
        nv = self.nv
        names = (("hw_slowdown", nv.nvmlClocksThrottleReasonHwSlowdown),
                 ("hw_thermal_slowdown", nv.nvmlClocksThrottleReasonHwThermalSlowdown),
                 ("sw_thermal_slowdown", nv.nvmlClocksThrottleReasonSwThermalSlowdown),
                 ("sw_power_cap", nv.nvmlClocksThrottleReasonSwPowerCap))
        while not self.stop_flag:
            try:
                clk = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.rows.append((time.perf_counter(), clk, {n for n, bit in names if mask & bit}))
            except Exception:
                pass
            time.sleep(0.001)

    def _pump_smi(self):
        for line in self.proc.stdout:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                clk, mx = float(f[0]), float(f[1])
            except ValueError:
                continue
            self.sm_max = mx
            reasons = {n for n, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"),
                                         f[3:7]) if v.lower().startswith("active")}
            self.rows.append((time.perf_counter(), clk, reasons))

    def stop(self, t0: float, t1: float) -> dict:
        if self.source is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": ["no clock source"]}
        time.sleep(0.05)
        self.stop_flag = True
        if self.proc is not None:
            self.proc.terminate()
        sm, reasons = [], set()
        for t, clk, rs in list(self.rows):
            if t0 <= t <= t1:
                sm.append(clk)
                reasons |= rs
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": self.sm_max,
                "samples": len(sm), "source": self.source, "reasons": sorted(reasons)}


def oracle_sample(d, l_max: int, rows: int, seed: int = 0, tier: int = 0, threads: int = 0):
    """The oracle on `rows` random rows against every other row (tier 0: full Wagner-Fischer table, no pruning;
    tier 1: length filter + the paper's row-minimum abort).  Returns (pairs/s, cells/s, threads, seconds, pairs)."""
    import oracle
    rng = np.random.default_rng(seed)
    sample = np.sort(rng.choice(d.n, size=min(rows, d.n), replace=False))
    t0 = time.perf_counter()
    _, used = oracle.edges(d.residues, d.lengths, l_max, rows=sample, all_partners=True, tier=tier, threads=threads)
    dt = time.perf_counter() - t0
    pairs = int(sample.size) * (d.n - 1)
    cells = float((d.lengths[sample].astype(np.int64) * (int(d.lengths.astype(np.int64).sum()))).sum()
                  - (d.lengths[sample].astype(np.int64) ** 2).sum())
    return pairs / dt, cells / dt, used, dt, pairs


def run_reference(args, rank: int) -> None:
    if rank != 0:
        return
    from cdr3_synth import CONFIGS, generate
    cfg = CONFIGS[WORKLOAD]
    d = generate(cfg)
    l_max = cfg.l_max[0]
    for _ in range(args.warmup):
        oracle_sample(d, l_max, 4)
    times, pairs, threads = [], 0, 0
    for k in range(args.steps):
        pps, cps, threads, dt, pairs = oracle_sample(d, l_max, ORACLE_SAMPLE_ROWS, seed=k)
        times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = pairs / (ms * 1e-3)
    sample = f"{ORACLE_SAMPLE_ROWS} random rows x all {d.n - 1} partners per step ({pairs} pairs), tier-0 full table"
    print(json.dumps({
        "impl": "reference", "metric": "levenshtein_pairs_per_s", "value": value, "unit": "pairs/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": f"{WORKLOAD}: N={cfg.n} synthetic CDR3b, l_max={l_max} (bounded sample per step)"},
        "cpu_baseline": {"value": value, "unit": "pairs/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def alu_ops_columns(work) -> float:
    """Algorithmic ALU lane-ops of the column-recurrence kernels (prefix trie / text chunks)."""
    return (ALU_OPS_PER_COLUMN * work["lane_columns_exec"] + ALU_OPS_PER_TEST * work["lane_tests_exec"]
            + ALU_OPS_PER_PREFIX_TEST * work["lane_prefix_tests_exec"]
            - (ALU_OPS_PER_COLUMN - ALU_OPS_FIRST_COLUMN) * work["lane_pairs_exec"] * (work["first_check"] > 0))


def alu_ops_join(work, l_max: int) -> float:
    """Algorithmic ALU lane-ops of the segment join (probe + verify kernels), from the counters of the instrumented
    instance: probes hashed, directory entries compared, candidates filtered (masks per diagonal of the band),
    survivors verified by Landau-Vishkin (l_max levels x the band's diagonals)."""
    cand = max(1, work["join_candidates"])
    nb_avg = work["join_diagonals"] / (cand + (work["join_survivors"] if l_max >= 2 else 0))
    verified = work["join_survivors"]
    ops = (JOIN_OPS_PER_PROBE * work["join_probes"] + JOIN_OPS_PER_ENTRY * work["join_entries"]
           + JOIN_OPS_PER_CANDIDATE * work["join_candidates"] + JOIN_OPS_PER_DIAGONAL * work["join_diagonals"]
           + verified * JOIN_OPS_PER_LV_STATE * max(1, l_max) * nb_avg)
    if l_max >= 2:  # the verify kernel widens the planes of every survivor again
        ops += JOIN_OPS_PER_CANDIDATE * verified
    return ops


def join_bytes(work, n_distinct: int, l_max: int, row_bytes: int) -> float:
    """Algorithmic bytes of the join: one directory pair per probe, every entry read, one plane row per candidate
    (and per survivor in the verify kernel, both rows), the pattern rows once per length difference."""
    b = 8.0 * work["join_probes"] + 8.0 * work["join_entries"] + row_bytes * work["join_candidates"]
    b += row_bytes * n_distinct * (l_max + 1)
    if l_max >= 2:
        b += (2 * row_bytes + 9 + 9) * work["join_survivors"]
    return b


def time_steps(net, step, flush, k, torch):
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
    stats = []
    for i in range(k):
        flush.fill_(i)
        ev[i][0].record()
        step()
        ev[i][1].record()
        stats.append(net.get_stats())
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in ev], stats


def run_widenings(args) -> None:
    """Wall-clock device timings (synchronised, best of 5) of the calls SURVEY 8(f) adds around the hot path."""
    import torch

    import paper_2112_06613_b200 as pkg
    from cdr3_synth import CONFIGS, generate
    cfg = CONFIGS[args.workload]
    l_max = cfg.l_max[0]
    d = generate(cfg)
    d_res, d_len = torch.from_numpy(d.residues).cuda(), torch.from_numpy(d.lengths).cuda()

    def best(f, k=5):
        f()
        ts = []
        for _ in range(k):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            f()
            torch.cuda.synchronize()
            ts.append(time.perf_counter() - t0)
        return 1e3 * min(ts)

    out = {"workload": args.workload, "n": d.n, "l_max": l_max, "unit": "ms (wall clock between synchronisations, best of 5)"}
    with pkg.TcrNet(0) as net:
        net.load(d_res, d_len)
        out["edges"] = net.build(l_max)
        # NEXT-1: observables on the CSR in HBM
        out["degree_histogram"] = best(lambda: (net.build(l_max), net.degree_histogram()))
        out["build_alone"] = best(lambda: net.build(l_max))
        out["degree_histogram"] -= out["build_alone"]
        out["neighbor_degree"] = best(lambda: (net.build(l_max), net.neighbor_degree())) - out["build_alone"]
        lab = {}
        def comp():
            net.build(l_max)
            lab["c"] = net.components()
        out["components"] = best(comp) - out["build_alone"]
        out["n_components"], out["lcc"] = lab["c"][2], lab["c"][3]
        rng = np.random.default_rng(0)
        rank = rng.permutation(d.n).astype(np.int32)
        steps = np.linspace(0, d.n, 21).astype(np.int64)
        out["percolation_21_steps"] = best(lambda: net.percolation(rank, steps), 3)
        # NEXT-3: labels of a build at l_max + 1, then the sweep down
        def sweep():
            net.build(l_max + 1)
            net.edge_distances()
            for t in range(l_max, -1, -1):
                net.restrict(t)
        out[f"build_l{l_max + 1}_labels_restrict_down_to_0"] = best(sweep, 3)
        out[f"build_l{l_max + 1}_alone"] = best(lambda: net.build(l_max + 1), 3)
        # 8(e): one shard through build_shard + assemble (what every rank of a sharded build does, world = 1)
        out["build_shard_plus_assemble"] = best(lambda: net.assemble(net.build_shard(l_max, 0, 1)))
    # NEXT-2: query x repertoire mode (first n_q rows are the queries), load + build
    for n_q in (177, 16663):
        if n_q >= d.n:
            continue
        with pkg.TcrNet(0) as net:
            net.set_option(pkg.OPT_N_QUERY, n_q)
            def step():
                net.load(d_res, d_len)
                return net.build(l_max)
            out[f"query_mode_nq{n_q}_load_build"] = best(step)
            out[f"query_mode_nq{n_q}_edges"] = step()
    print(json.dumps(out))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=WORKLOAD, help="cdr3_synth config name (bench line: cfg4)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the side measurements (prefix-trie path, collapse off, CASS-prefixed input, pipe probes)")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: ONE repertoire, every rank builds its shard of the work items, the edge keys are "
                         "all-gathered and every rank assembles the CSR (strong scaling); default: replicas (weak)")
    ap.add_argument("--widenings", action="store_true",
                    help="instead of the bench line: device timings of the SURVEY 8(f) rows on the workload (observables, "
                         "distance labels + threshold sweep, query x repertoire mode, one shard + assemble), one JSON line")
    ap.add_argument("--first-check", type=int, default=0)
    ap.add_argument("--text-chunk", type=int, default=0)
    ap.add_argument("--trie-chunk", type=int, default=0)
    ap.add_argument("--no-trie", action="store_true", help="text-chunk kernel only (every kept pair visited)")
    ap.add_argument("--segment-join", type=int, default=None, choices=[-1, 0, 1],
                    help="TCRNET_OPT_SEGMENT_JOIN (default: the library's)")
    ap.add_argument("--no-dedup", action="store_true", help="TCRNET_OPT_DEDUP = 0 (identical rows are not collapsed)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.widenings:
        if rank == 0:
            run_widenings(args)
        return

    import torch
    import torch.distributed as dist

    import paper_2112_06613_b200 as pkg
    from cdr3_synth import CONFIGS, generate

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sharded = args.sharded  # (N = 1: one shard - the same calls, no collective)
    cfg = CONFIGS[args.workload]
    l_max = cfg.l_max[0]
    # replicas: an independent repertoire per rank; sharded: the same repertoire on every rank
    d = generate(cfg, seed=cfg.seed + (0 if sharded else 1000 * rank))
    n = d.n
    pairs_all = n * (n - 1) // 2

    # raw inputs: pinned host copies (e2e) and device copies (value)
    h_res = torch.from_numpy(d.residues).pin_memory()
    h_len = torch.from_numpy(d.lengths).pin_memory()
    d_res, d_len = h_res.cuda(non_blocking=True), h_len.cuda(non_blocking=True)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    net = pkg.TcrNet(local_rank)
    if args.first_check:
        net.set_option(pkg.OPT_FIRST_CHECK, args.first_check)
    if args.text_chunk:
        net.set_option(pkg.OPT_TEXT_CHUNK, args.text_chunk)
    if args.trie_chunk:
        net.set_option(pkg.OPT_TRIE_CHUNK, args.trie_chunk)
    if args.no_trie:
        net.set_option(pkg.OPT_PREFIX_TRIE, 0)
    if args.segment_join is not None:
        net.set_option(pkg.OPT_SEGMENT_JOIN, args.segment_join)
    if args.no_dedup:
        net.set_option(pkg.OPT_DEDUP, 0)

    def step_device():
        net.load(d_res, d_len)
        if sharded:
            from paper_2112_06613_b200.parallel import build_distributed
            return build_distributed(net, l_max)
        return net.build(l_max)

    e2e_split = [0.0, 0.0, 0.0]

    def step_host():
        t0 = time.perf_counter()
        net.load(h_res.numpy(), h_len.numpy())
        t1 = time.perf_counter()
        if sharded:
            from paper_2112_06613_b200.parallel import build_distributed
            build_distributed(net, l_max)
        else:
            net.build(l_max)
        t2 = time.perf_counter()
        out = net.copy_csr(staged=True)  # page-locked result buffers owned by the binding
        t3 = time.perf_counter()
        for i, dt in enumerate((t1 - t0, t2 - t1, t3 - t2)):
            e2e_split[i] += dt
        return out

    # work accounting pass (instrumented kernel, outside every timed region)
    net.set_option(pkg.OPT_COUNT_WORK, 1)
    step_device()
    work = net.get_stats()
    net.set_option(pkg.OPT_COUNT_WORK, 0)

    for _ in range(max(args.warmup, 3) if args.warmup else 0):
        step_device()

    # ---- timed: K steps, device-resident inputs, CUDA events on the library's stream ----
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    stats = []
    barrier()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.fill_(k)  # L2 flush between timed iterations (not timed)
        ev[k][0].record()
        n_edges = step_device()
        ev[k][1].record()
        stats.append(net.get_stats())
    barrier()
    t_wall1 = time.perf_counter()
    ms_steps = [a.elapsed_time(b) for a, b in ev]
    ms_step = float(np.mean(ms_steps))
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None

    # ---- timed: end to end from host buffers through the C ABI ----
    for _ in range(2):
        step_host()
    barrier()
    e2e_split[:] = [0.0, 0.0, 0.0]
    e2e_times = []
    for k in range(args.steps):
        flush.fill_(k)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        rp, cl, dg = step_host()
        torch.cuda.synchronize()
        e2e_times.append(time.perf_counter() - t0)
    barrier()
    ms_e2e = 1e3 * float(np.mean(e2e_times))
    h2d = int(d.residues.nbytes + d.lengths.nbytes)
    d2h = int(rp.nbytes + cl.nbytes + dg.nbytes)

    # the split of the step by phase needs an event around every phase (TCRNET_OPT_TIMING = 2: 2-4 us each and the
    # end of the launch overlap there), so it is measured in three steps of its own outside the timed region
    net.set_option(pkg.OPT_TIMING, 2)
    step_device()
    ms_phase_steps, phase_stats = time_steps(net, step_device, flush, 3, torch)
    net.set_option(pkg.OPT_TIMING, 1)
    barrier()

    if world > 1:
        t = torch.tensor([ms_step, ms_e2e], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_step, ms_e2e = float(t[0]), float(t[1])

    if rank == 0:
        peaks, peak_kind = _peaks()
        n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count
        ms_kernel = float(np.mean([s["ms_kernel"] for s in stats]))  # live, inside the timed region (TCRNET_OPT_TIMING = 1)
        mean = lambda key: float(np.mean([s[key] for s in phase_stats]))  # noqa: E731
        ms_dist, ms_sort, ms_csr, ms_load, ms_index = (mean(k) for k in (
            "ms_distance", "ms_sort", "ms_csr", "ms_load", "ms_index"))
        peak = n_sm * ALU_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12
        join = work["join_mode"] > 0 and work["work_items_join"] == work["work_items"]
        if join:
            alu_ops = alu_ops_join(work, l_max)
            kernel = "k_join_probe" + (" + k_join_verify" if l_max >= 2 else "")
        else:
            alu_ops = alu_ops_columns(work)
            kernel = "k_distance_trie" if work["work_items_trie"] else "k_distance"
        achieved = alu_ops / (ms_kernel * 1e-3) / 1e12
        jobs = 1 if sharded else world  # networks built per step
        out = {
            "metric": "levenshtein_pairs_per_s", "value": jobs * pairs_all / (ms_step * 1e-3), "unit": "pairs/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
            "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "int32",
            "data": "synthetic",
            "config": {
                "workload": f"{args.workload}: N={n} synthetic CDR3b" +
                            (f" (BASELINE.json configs[{cfg.index - 1}])" if cfg.index <= 5 else " (stress input)") +
                            f", l_max={l_max}",
                "n": n, "l_max": l_max, "edges": int(n_edges), "l2": "flushed between timed steps (256 MiB write)",
                "parallelism": ("sharded work items + all-gather of edge keys" if sharded else "replicas") if world > 1
                               else "single GPU",
                "path": "segment join (pigeonhole index, shifted-Hamming filter, Landau-Vishkin verification)" if join
                        else "length-bucket pairs through the prefix trie / text chunks (Myers column recurrence)",
            },
            "clocks": clocks,
            "e2e": {"value": jobs * pairs_all / (ms_e2e * 1e-3), "unit": "pairs/s", "ms_per_step": ms_e2e,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_load_build_copy": [1e3 * x / args.steps for x in e2e_split]},
            "gpu_launches": int(sum(s["launches_load"] + s["launches_build"] for s in stats)),
            "roofline": {
                "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TIOP/s (INT32 ALU-pipe lane-ops)",
                "frac": achieved / peak, "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get((args.workload, kernel)),
                "kernel": kernel, "kernel_ms": ms_kernel, "kernel_share_of_step": ms_kernel / ms_step,
                "peak_source": f"{n_sm} SMs x {ALU_LANES_PER_SM} lanes x {peaks['sm_max_mhz']} MHz ({peak_kind} sm_max_mhz)",
                "alu_ops_per_launch": alu_ops,
                # also against the issue-slot ceiling (4 schedulers x 32 lanes per SM and clock)
                "issue_ceiling": 2 * peak, "frac_of_issue_ceiling": achieved / (2 * peak),
            },
            "detail": {
                "pairs_kept": work["pairs_kept"], "cells_kept": work["cells_kept"], "cells_all": work["cells_all"],
                "n_distinct": work["n_distinct"],
                "pairs_per_s_evaluated": work["pairs_kept"] / (ms_kernel * 1e-3),
                "gcups_evaluated": work["cells_kept"] / (ms_kernel * 1e-3) / 1e9,
                "gcups_effective": work["cells_all"] / (ms_step * 1e-3) / 1e9,
                "ms_pack": ms_load, "ms_distance": ms_dist, "ms_distance_kernel": ms_kernel, "ms_index": ms_index,
                "ms_sort": ms_sort, "ms_csr": ms_csr, "ms_step_with_phase_events": float(np.mean(ms_phase_steps)),
                "launches_per_step": stats[-1]["launches_load"] + stats[-1]["launches_build"],
                "work_items": work["work_items"], "work_items_trie": work["work_items_trie"],
                "work_items_join": work["work_items_join"], "join_mode": work["join_mode"],
                "join_probes": work["join_probes"], "join_entries": work["join_entries"],
                "join_candidates": work["join_candidates"], "join_survivors": work["join_survivors"],
                "join_diagonals": work["join_diagonals"], "join_index_entries": work["join_index_entries"],
                "lane_columns_exec": work["lane_columns_exec"], "lane_tests_exec": work["lane_tests_exec"],
                "lane_prefix_tests_exec": work["lane_prefix_tests_exec"],
                "columns_executed_fraction": work["lane_columns_exec"] / max(1, work["columns_kept"]),
                "ms_steps": ms_steps,
            },
        }
        if join:
            row_bytes = 64 if work["max_len"] > 32 else 32
            jb = join_bytes(work, work["n_distinct"], l_max, row_bytes)
            out["roofline"]["memory_view"] = {
                "algorithmic_bytes": jb, "gb_per_s": jb / (ms_kernel * 1e-3) / 1e9,
                "frac_of_hbm_peak": jb / (ms_kernel * 1e-3) / 1e9 / peaks["hbm_gbs"],
                "note": "random 32-byte sector reads of L2-resident tables; the HBM copy peak is the contract's denominator",
            }
        # the emission / CSR passes against the HBM peak (algorithmic bytes of DESIGN.md section 7:
        # A6 bucket scatter 8 + 8 B, rank 8 + 4 B per edge, 12 B per node and the scan's 4 + 8 B per node)
        e_cnt = int(n_edges)
        csr_bytes = e_cnt * 28 + n * 24
        out["hbm_passes"] = {
            "csr_algorithmic_bytes": csr_bytes, "csr_ms": ms_csr,
            "csr_gb_per_s": csr_bytes / (ms_csr * 1e-3) / 1e9 if ms_csr > 0 else None,
            "csr_frac_of_hbm_peak": (csr_bytes / (ms_csr * 1e-3) / 1e9) / peaks["hbm_gbs"] if ms_csr > 0 else None,
            "note": "L2-resident, launch- and latency-bound at this size (6 launches, 20-50 us each)",
        }
        if not args.no_extras and world == 1:
            extras = {}
            # (a) the length-bucket path of round 1 (every length-compatible pair through the prefix trie): its own
            #     roofline line, measured outside the timed region
            def side(opts, data=None, k=3, lm=None):
                with pkg.TcrNet(local_rank) as other:
                    for o, v in opts.items():
                        other.set_option(o, v)
                    r_d, l_d = (d_res, d_len) if data is None else data

                    def one():
                        other.load(r_d, l_d)
                        other.build(l_max if lm is None else lm)
                    other.set_option(pkg.OPT_COUNT_WORK, 1)
                    one()
                    w = other.get_stats()
                    other.set_option(pkg.OPT_COUNT_WORK, 0)
                    one()
                    ms, st = time_steps(other, one, flush, k, torch)
                return float(np.mean(ms)), w, st
            if join and l_max <= 4 and n <= 1_000_000:
                ms_t, w_t, st_t = side({pkg.OPT_SEGMENT_JOIN: 0})
                k_ms = float(np.mean([s["ms_kernel"] for s in st_t]))
                ach = alu_ops_columns(w_t) / (k_ms * 1e-3) / 1e12
                out["roofline_trie_path"] = {
                    "bound": "alu", "kernel": "k_distance_trie", "kernel_ms": k_ms, "ms_per_step": ms_t,
                    "achieved": ach, "peak": peak, "frac": ach / peak, "alu_ops_per_launch": alu_ops_columns(w_t),
                    "columns_executed_fraction": w_t["lane_columns_exec"] / max(1, w_t["columns_kept"]),
                    "gcups_evaluated": w_t["cells_kept"] / (k_ms * 1e-3) / 1e9,
                    "note": "TCRNET_OPT_SEGMENT_JOIN = 0: not the timed path; kept for comparison with round 1",
                }
            # (b) how much of the step is the data: identical rows not collapsed; conserved CASS... / ...EQYF ends
            ms_nd, _, _ = side({pkg.OPT_DEDUP: 0})
            extras["ms_step_dedup_off"] = ms_nd
            if args.workload == "cfg4":
                dc = generate("cfg4_cass")
                data = (torch.from_numpy(dc.residues).cuda(), torch.from_numpy(dc.lengths).cuda())
                ms_c, w_c, st_c = side({}, data)
                extras["ms_step_cass_prefix_input"] = ms_c
                extras["cass_prefix_input"] = {"edges": int(st_c[-1]["n_edges"]), "n_distinct": int(w_c["n_distinct"]),
                                               "join_candidates": int(w_c["join_candidates"]),
                                               "ms_distance_kernel": float(np.mean([s["ms_kernel"] for s in st_c]))}
                # ... and at l_max = 2, where the segment cuts follow the residue statistics of the load
                ms_c2, w_c2, st_c2 = side({}, data, lm=2)
                extras["cass_prefix_input_l_max_2"] = {
                    "ms_step": ms_c2, "edges": int(st_c2[-1]["n_edges"]),
                    "join_entries": int(w_c2["join_entries"]), "join_candidates": int(w_c2["join_candidates"]),
                    "join_adapted_lengths": int(w_c2["join_adapted_lengths"]),
                    "ms_distance_kernel": float(np.mean([s["ms_kernel"] for s in st_c2]))}
                del data
                # ... and the same repertoire as a table of DISTINCT sequences (the usual form of real data): nothing
                # to collapse; after the first such load the library pauses the attempt (TCRNET_OPT_DEDUP)
                off = np.concatenate([[0], np.cumsum(d.lengths.astype(np.int64))])
                first = {}
                for i in range(n):
                    first.setdefault(d.residues[off[i]:off[i + 1]].tobytes(), i)
                keep = np.fromiter(sorted(first.values()), dtype=np.int64)
                u_res = np.concatenate([d.residues[off[i]:off[i + 1]] for i in keep])
                data = (torch.from_numpy(u_res).cuda(), torch.from_numpy(np.ascontiguousarray(d.lengths[keep])).cuda())
                ms_u, w_u, st_u = side({}, data)
                extras["distinct_rows_input"] = {"n": int(keep.size), "ms_step": ms_u, "edges": int(st_u[-1]["n_edges"]),
                                                 "pairs_per_s": keep.size * (keep.size - 1) / 2 / (ms_u * 1e-3)}
                del data
            out["detail"].update(extras)
            probes = {}
            for kind, name in ((0, "lop3"), (2, "imad"), (3, "lop3_imad_mix"), (5, "myers_step")):
                ops, mhz = net.probe_int32(kind)
                probes[name] = {"tera_per_s": ops / 1e12, "sm_mhz": mhz}
            out["roofline"]["measured_pipe_peaks"] = probes
        if not args.no_cpu_baseline and world == 1:
            all_cores = os.cpu_count() or 1
            pps, cps, threads, dt, pairs = oracle_sample(d, l_max, ORACLE_SAMPLE_ROWS, threads=all_cores)
            out["cpu_baseline"] = {
                "value": pps, "unit": "pairs/s", "cores": threads, "kind": "oracle", "gcups": cps / 1e9,
                "sample": f"{ORACLE_SAMPLE_ROWS} random rows x all {n - 1} partners ({pairs} pairs, {dt:.1f} s), tier-0 full table",
            }
            # the paper's CPU comparison is ONE core; tier 1 = the paper's own abort + length filter
            p1, _, t1, dt1, pr1 = oracle_sample(d, l_max, 64, tier=0, threads=1)
            p2, _, t2, dt2, pr2 = oracle_sample(d, l_max, 4 * ORACLE_SAMPLE_ROWS, tier=1, threads=all_cores)
            p3, _, t3, dt3, pr3 = oracle_sample(d, l_max, 128, tier=1, threads=1)
            out["cpu_baseline"]["also"] = {
                "tier0_1core": {"value": p1, "cores": t1, "sample": f"64 rows x all partners ({pr1} pairs, {dt1:.1f} s)"},
                "tier1_all_cores": {"value": p2, "cores": t2, "sample": f"{4 * ORACLE_SAMPLE_ROWS} rows x all partners ({pr2} pairs, {dt2:.1f} s), length filter + row-minimum abort"},
                "tier1_1core": {"value": p3, "cores": t3, "sample": f"128 rows x all partners ({pr3} pairs, {dt3:.1f} s)"},
            }
        print(json.dumps(out))
    net.destroy()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
