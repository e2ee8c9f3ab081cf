#!/usr/bin/env python
"""bench.py -- times the two-vector Four-Russians fold on B200 and prints ONE JSON line.

Workload at N=1: BASELINE.json's headline configuration, configs[2] = "single sequence n=6000,
i.i.d. uniform {A,C,G,U}, seed 2, q=8" (the paper's largest length; the metric "fold time at
n=6000 (s) and cell-k-updates/s" is quoted on it).  A step = one whole fold through the C ABI
(rna4r_fold: encode, plan, persistent wavefront fill with fused vector packing, score) with the
sequence already resident in HBM; rna4r_prepare (the one-time R-table build, step a2) is timed
separately and reported as `prepare_ms`.  `e2e` is the same fold through rna4r_fold_host with
pinned HOST buffers, host<->device copies inside the timed region.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-cpu] [--no-also]

N>1 (torchrun): the single fold does not shard (every cell needs its whole row and column,
PAPER.md:223) -- "replicas only": each rank folds its own replica, value = N*W / max-rank time.

--impl reference: the oracle (oracle/, plain eq. (1), 1 thread) timed as it stands on a bounded
sample of the same workload (the first 2000 bases of the same sequence).
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

import workloads  # noqa: E402

Q = 8
CFG = "cfg3"
WORKLOAD = "cfg3: single RNA sequence n=6000, i.i.d. uniform {A,C,G,U}, seed 2, q=8, score only (BASELINE.json configs[2])"


def nussinov_updates(n: int) -> int:
    """W(n) = n(n^2-1)/6 Nussinov-equivalent cell-k-updates (inner-loop steps of eq. (1))."""
    return n * (n * n - 1) // 6


def algorithmic_lookups(n: int, q: int) -> int:
    """L = sum_d (n-d) floor(d/q): table lookups of the two-vector fill."""
    d = np.arange(1, n, dtype=np.int64)
    return int(((n - d) * (d // q)).sum())


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.01):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.sm_max = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, nm in names.items():
                    if mask & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        return {
            "sm_mhz": float(np.median(self.samples)) if self.samples else None,
            "sm_max_mhz": self.sm_max,
            "reasons": sorted(self.reasons),
            "samples": len(self.samples),
        }


def cpu_baselines(seq: bytes, q: int):
    """Oracle as it stands, host cores, bounded sample; plus the serial two-vector build."""
    import oracle
    n_s = 3000
    t0 = time.perf_counter()
    sc = oracle.nussinov(seq[:n_s])
    dt = time.perf_counter() - t0
    base = {
        "value": nussinov_updates(n_s) / dt, "unit": "cell-k-updates/s", "cores": 1, "kind": "oracle",
        "sample": f"plain eq.(1) oracle (oracle_nussinov, int32, 1 thread) on the first {n_s} bases of the same sequence: {dt:.2f} s, D(1,{n_s})={sc}",
    }
    t0 = time.perf_counter()
    tv = oracle.two_vector_serial(seq, q)
    dt2 = time.perf_counter() - t0
    extra = {
        "two_vector_serial": {
            "value": nussinov_updates(len(seq)) / dt2, "unit": "cell-k-updates/s", "cores": 1, "seconds": dt2,
            "sample": f"Algorithm 1 (PAPER.md:125-187), q={q}, whole n={len(seq)} fold, 1 thread; paper: ~57 s desktop / ~15 s server (PAPER.md:13)",
            "score": tv["score"],
        }
    }
    # the paper's speed-up table (Nussinov seconds and the speed-ups of two-vector, partially
    # memoised, completely memoised, FG) on this host, on the same 3000-base sample as the oracle above
    tab = {"n": n_s, "nussinov_s": dt, "paper_row_n3000": {"nussinov_s": 62.5, "two_vector": 8.8, "partially_memoized": 8.3,
                                                            "completely_memoized": 6.4, "frid_gusfield": 3.4, "cite": "PAPER.md:320"}}
    for name, qq, fn in (("two_vector", q, lambda: oracle.two_vector_serial(seq[:n_s], q)),
                         ("partially_memoized", q, lambda: oracle.serial_variant(seq[:n_s], q, "partially_memoized")),
                         ("completely_memoized", q, lambda: oracle.serial_variant(seq[:n_s], q, "completely_memoized")),
                         ("frid_gusfield", 3, lambda: oracle.serial_variant(seq[:n_s], 3, "frid_gusfield"))):
        t0 = time.perf_counter()
        rr = fn()
        dtv = time.perf_counter() - t0
        assert rr["score"] == sc
        tab[name] = {"q": qq, "seconds": dtv, "speedup_vs_nussinov": dt / dtv}
    extra["serial_speedup_table"] = tab
    return base, extra


def run_reference(args, rank: int):
    """--impl reference: the oracle timed as it stands on a bounded sample per step."""
    if rank != 0:
        return
    import oracle
    seq = workloads.single_config(CFG)
    n_s = 2000
    sample = seq[:n_s]
    for _ in range(args.warmup):
        oracle.nussinov(sample)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.nussinov(sample)
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    val = nussinov_updates(n_s) / dt
    desc = f"plain eq.(1) oracle (oracle_nussinov, 1 thread) on the first {n_s} bases of the cfg3 sequence, one fold per step"
    print(json.dumps({
        "impl": "reference", "metric": "cell_k_updates_per_s", "value": val, "unit": "cell-k-updates/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "q": Q, "n": 6000},
        "cpu_baseline": {"value": val, "unit": "cell-k-updates/s", "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": "cell-k-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-also", action="store_true", help="skip the extra workloads (cfg2, cfg4 batch, cfg5)")
    ap.add_argument("--profile", action="store_true", help="short run for ncu: no e2e leg, no tail loop, no extras")
    ap.add_argument("--engine", default="auto", choices=["auto", "tiled", "diag"],
                    help="auto (what a user gets): single folds on the tiled engine, batches of short sequences on the "
                         "CTA-per-sequence shared-memory engine")
    ap.add_argument("--cfg", default="cfg3", choices=["cfg2", "cfg3", "cfg4", "cfg5"],
                    help="workload (profiling aid; the headline and the default is cfg3; cfg4 = the batch, device-timed only)")
    ap.add_argument("--q", type=int, default=8, help="vector length q (profiling aid; the headline is q = 8)")
    args = ap.parse_args()
    global CFG, WORKLOAD, Q
    Q = args.q
    if args.cfg == "cfg4":
        return profile_batch(args)
    if args.cfg != CFG:
        CFG = args.cfg
        WORKLOAD = f"{CFG}: single RNA sequence n={workloads.SINGLE_CONFIGS[CFG]['n']}, i.i.d. uniform {{A,C,G,U}}, q=8, score only"
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import paper_1307_7820_b200 as pkg

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    args.warmup = max(args.warmup, 3)
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    peaks = measured_peaks()
    seq = workloads.single_config(CFG)
    n = len(seq)
    W_updates = nussinov_updates(n)
    L_lookups = algorithmic_lookups(n, Q)

    # one-time preprocessing (step a2), timed separately
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    r = pkg.Rna4r(Q, local_rank, {"auto": pkg.ENGINE_AUTO, "tiled": pkg.ENGINE_TILED, "diag": pkg.ENGINE_DIAG}[args.engine])
    torch.cuda.synchronize()
    prepare_ms = (time.perf_counter() - t0) * 1e3
    r.enable_kernel_timing(True)

    seq_dev = torch.from_numpy(np.frombuffer(seq, dtype=np.uint8).copy()).cuda()
    score_dev = torch.zeros(1, dtype=torch.int32, device="cuda")
    ws = r.workspace(r.workspace_bytes_host(np.array([n], dtype=np.int32)))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()

    def one_fold():
        r.fold(seq_dev, n, score_out=score_dev, workspace=ws, stream=stream)

    for _ in range(args.warmup):
        flush.fill_(1)
        one_fold()
    torch.cuda.synchronize()
    score = int(score_dev.item())

    # ---- timed region: K folds, each bracketed by CUDA events on the launching stream; L2 flushed between
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    fill_ms = []
    launches = 0
    for k in range(args.steps):
        flush.fill_(k & 0xFF)
        ev[k][0].record(stream)
        one_fold()
        ev[k][1].record(stream)
        launches += r.last_launch_count()
        fill_ms.append(r.last_fill_kernel_ms())       # waits for this fold's dominant kernel
    barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    # keep the GPU busy a little longer so the sampler sees clocks under load even for short runs
    t_end = time.perf_counter() + (0.0 if args.profile else 0.25)
    while time.perf_counter() < t_end:
        one_fold()
    torch.cuda.synchronize()
    clocks = sampler.stop()

    if dist is not None:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    value = world * W_updates / (ms_per_step * 1e-3)

    # ---- e2e: host buffers through rna4r_fold_host, copies inside the timed region (wall clock, synchronous call)
    seq_pinned = torch.from_numpy(np.frombuffer(seq, dtype=np.uint8).copy()).pin_memory()
    score_pinned = torch.zeros(1, dtype=torch.int32).pin_memory()
    for _ in range(0 if args.profile else 3):
        r.fold_host(seq_pinned, workspace=ws, stream=stream, score_host=score_pinned)
    barrier()
    t0 = time.perf_counter()
    for _ in range(1 if args.profile else args.steps):
        sc_e2e, _ = r.fold_host(seq_pinned, workspace=ws, stream=stream, score_host=score_pinned)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / (1 if args.profile else args.steps)
    if dist is not None:
        t = torch.tensor([e2e_s], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    assert sc_e2e == score

    # ---- N > 1: the workload that shards: cfg4, sequences dealt longest-first round-robin to the ranks,
    # each rank folds its shard through rna4r_fold_batch_host, no data-path collective (scores gathered host-side)
    sharded = None
    if world > 1:
        sharded = sharded_batch(pkg, torch, dist, r, rank, world, barrier, args.steps)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the persistent fill kernel)
    fill_avg_ms = float(np.mean(fill_ms))
    sm_count = torch.cuda.get_device_properties(local_rank).multi_processor_count
    peak_lookups = sm_count * 32 * peaks["sm_max_mhz"] * 1e6          # one 32-lane shared-memory wavefront / SM / clk
    ach_lookups = L_lookups / (fill_avg_ms * 1e-3)
    alg_bytes = n + 4                                                  # read n bases, write one int32 score
    roofline = {
        "bound": "smem", "kernel": f"tiled::fill_kernel<{Q}>" if args.engine != "diag" else "diag_fill_kernel (all diagonals)",
        "achieved": ach_lookups / 1e9, "peak": peak_lookups / 1e9, "unit": "Glookup/s",
        "frac": ach_lookups / peak_lookups,
        "traffic": None,
        "per_unit": "1 table lookup = one 1-byte shared-memory gather (replaces q=8 inner-loop steps); "
                    f"units per launch L = sum_d (n-d) floor(d/q) = {L_lookups}",
        "peak_source": f"{sm_count} SMs x 32 lanes x {peaks['sm_max_mhz']:.0f} MHz (max SM clock, MEASURED_PEAKS.json: {peaks['source']})",
        "kernel_ms": fill_avg_ms, "kernel_share_of_step": fill_avg_ms / ms_per_step,
        "hbm": {"algorithmic_bytes": alg_bytes, "achieved_gbs": alg_bytes / (fill_avg_ms * 1e-3) / 1e9,
                "peak_gbs": peaks["hbm_gbs"], "frac": alg_bytes / (fill_avg_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                "note": "not the binding roofline: the fold reads n bytes and writes 4"},
    }
    # DRAM traffic of the same kernel, per launch: an ncu counter cannot be read inside an un-profiled run, so this
    # is the committed value of the latest `ncu --set full` capture (profiles/traffic.json names the capture)
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath) and CFG == "cfg3" and Q == 8 and args.engine != "diag":
        try:
            with open(tpath) as f:
                tj = json.load(f)
            roofline["traffic"] = tj.get("cfg3_fill_kernel_dram_bytes")
            roofline["traffic_source"] = "static: " + str(tj.get("source")) + " (not measured by this run)"
        except Exception:
            pass
    # measured ceiling of the lookup sequence itself (rna4r_microbench_lookups): what the SM sustains for the bare
    # 4-instruction lookup, and for the bulk product's inner loop, conflict-free on every SM
    if not args.profile and args.engine != "diag" and Q == 8:
        try:
            ceil = {}
            for name, variant in (("pure_4_instr_lookup", 0), ("bulk_product_inner_loop", 1)):
                best = 0.0
                for _ in range(3):
                    ms, nl = r.microbench_lookups(variant, 4000 if variant == 0 else 500)
                    best = max(best, nl / (ms * 1e-3))
                ceil[name] = {"glookups_per_s": best / 1e9, "frac_of_formula_peak": best / peak_lookups}
            roofline["measured_ceiling"] = ceil
            roofline["frac_of_measured_ceiling"] = ach_lookups / (ceil["pure_4_instr_lookup"]["glookups_per_s"] * 1e9)
        except Exception as e:       # profiling aid only
            roofline["measured_ceiling"] = {"error": str(e)}

    out = {
        "metric": "cell_k_updates_per_s", "value": value, "unit": "cell-k-updates/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "fold_time_s": ms_per_step * 1e-3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "n": n, "q": Q, "engine": {1: "tiled", 2: "diag", 3: "smem"}[r.engine], "score": score,
                   "l2": "flushed between steps (256 MB write)", "prepare": "rna4r_prepare timed separately (prepare_ms)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "prepare_ms": prepare_ms,
        "clocks": clocks,
        "e2e": {"value": world * W_updates / e2e_s, "unit": "cell-k-updates/s", "seconds_per_fold": e2e_s,
                "h2d_bytes_per_step": n, "d2h_bytes_per_step": 4},
        "gpu_launches": launches,
        "roofline": roofline,
        "paper_context": {"tesla_c2070_s": 2.50, "geforce_gtx550ti_s": 4.97, "cite": "PAPER.md:345"},
    }

    if sharded is not None:
        out["batch_sharded"] = sharded
    if args.profile:
        args.no_also = args.no_cpu = True
    if not args.no_also and world == 1:
        out["also"] = also_workloads(pkg, torch, r, flush)
        for v in out["also"].values():      # the same shared-memory-gather roofline for the throughput-bound configs
            if "lookups" in v and v.get("fill_kernel_ms"):
                v["smem_roofline_frac"] = v["lookups"] / (v["fill_kernel_ms"] * 1e-3) / peak_lookups
    if not args.no_cpu and world == 1:
        base, extra = cpu_baselines(seq, Q)
        out["cpu_baseline"] = base
        out["cpu_baselines_extra"] = extra
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def profile_batch(args):
    """--cfg cfg4: the batch of config 4 through rna4r_fold_batch (AUTO: the SMEM engine), device-timed; for ncu."""
    import torch
    import paper_1307_7820_b200 as pkg
    r = pkg.Rna4r(Q, 0, {"auto": pkg.ENGINE_AUTO, "tiled": pkg.ENGINE_TILED, "diag": pkg.ENGINE_DIAG}[args.engine])
    r.enable_kernel_timing(True)
    seqs, lens = workloads.gc_rich_batch()
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    fd, od = torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda()
    ws = torch.empty(r.workspace_bytes_batch(lens32), dtype=torch.uint8, device="cuda")
    sc = torch.empty(len(lens32), dtype=torch.int32, device="cuda")
    ms = []
    for _ in range(max(args.warmup, 1) + args.steps):
        r.fold_batch(fd, od, lens32, scores_out=sc, workspace=ws)
        ms.append(r.last_fill_kernel_ms())
    ltot = int(sum(algorithmic_lookups(int(x), Q) for x in lens32))
    k = float(np.median(ms[max(args.warmup, 1):]))
    print(json.dumps({"workload": "cfg4: 1024 sequences, lengths U[300,700], one rna4r_fold_batch call", "q": Q,
                      "launches_per_call": r.last_launch_count(), "kernel_ms": k, "lookups": ltot,
                      "smem_roofline_frac": ltot / (k * 1e-3) / (148 * 32 * 1.965e9), "sum_scores": int(sc.sum().item())}))


def sharded_batch(pkg, torch, dist, r, rank, world, barrier, steps):
    """cfg4 sharded by sequence over the ranks (paper_1307_7820_b200/shard.py); value = sum W / max-rank time."""
    from paper_1307_7820_b200 import shard
    seqs, lens = workloads.gc_rich_batch()
    idx = shard.shard_indices(lens, world, rank)
    mine = [seqs[i] for i in idx]
    flat, _, lens32 = workloads.pack_batch(mine)
    pinned = torch.from_numpy(flat).pin_memory()
    out_p = torch.zeros(len(lens32), dtype=torch.int32).pin_memory()
    ws = torch.empty(r.workspace_bytes_host(lens32), dtype=torch.uint8, device="cuda")
    for _ in range(3):
        r.fold_batch_host(pinned, lens32, workspace=ws, scores_host=out_p)
    barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        sc = r.fold_batch_host(pinned, lens32, workspace=ws, scores_host=out_p)
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / steps
    t = torch.tensor([dt], device="cuda", dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    tot = torch.tensor([float(sc.sum())], device="cuda", dtype=torch.float64)
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    wtot = int(sum(nussinov_updates(int(x)) for x in lens))
    return {"workload": "cfg4: 1024 sequences, lengths U[300,700], sharded by sequence (longest first, round robin), "
                        "rna4r_fold_batch_host per rank, no collective on the data path",
            "value": wtot / float(t.item()), "unit": "cell-k-updates/s", "seconds_per_batch_max_rank": float(t.item()),
            "sum_scores": int(tot.item()), "scaling": "strong"}


def also_workloads(pkg, torch, r8, flush):
    """Device-timed numbers for the other configs (parity cases; context beside the headline)."""
    res = {}

    def time_call(fn, reps):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            flush.fill_(3)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts))

    # cfg2
    s = workloads.single_config("cfg2")
    d = torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda()
    ms = time_call(lambda: r8.fold(d), 10)
    res["cfg2_n2000_q8"] = {"ms": ms, "cell_k_updates_per_s": nussinov_updates(len(s)) / (ms * 1e-3)}
    # cfg3 with the full int16 table written (72 MB, step a8) and one traceback over it
    s3 = workloads.single_config("cfg3")
    d3 = torch.from_numpy(np.frombuffer(s3, dtype=np.uint8).copy()).cuda()
    tab3 = torch.empty((len(s3), len(s3)), dtype=torch.int16, device="cuda")
    ms_tab = time_call(lambda: r8.fold(d3, table_dtype=pkg.TABLE_INT16, table_out=tab3), 5)
    out_tb = {}

    def tb():
        out_tb["r"] = r8.traceback(d3, tab3)

    ms_tb = time_call(tb, 5)
    res["cfg3_n6000_q8_with_table"] = {"ms": ms_tab, "table_bytes": int(tab3.numel()) * 2,
                                        "traceback_ms": ms_tb, "traceback_pairs": int(out_tb["r"][1].item())}
    del tab3
    # q sweep at n = 6000 (the paper saw the serial gains saturate at q = 8-9)
    sweep = {}
    for q in (4, 5, 6, 7, 8, 9, 10, 11):
        rq = r8 if q == 8 else pkg.Rna4r(q, 0)
        sweep[str(q)] = time_call(lambda: rq.fold(d3), 5)
        if q != 8:
            rq.close()
    res["q_sweep_n6000_ms"] = sweep
    # the comparison engines at n = 6000, q = 8: the paper's section 4 kernel (one launch per cell
    # diagonal), its section 5.3 q x q tile kernel (one launch per tile diagonal), and a DPX max-plus kernel without R
    cmp_ms = {"tiled": sweep["8"]}
    for name, eng in (("diag_paper_section4", pkg.ENGINE_DIAG), ("paper_tile_section5_3", pkg.ENGINE_PAPER_TILE),
                      ("maxplus_dpx_no_table", pkg.ENGINE_MAXPLUS)):
        rc = pkg.Rna4r(8, 0, eng)
        cmp_ms[name] = time_call(lambda: rc.fold(d3), 2)
        rc.close()
    res["engines_n6000_q8_ms"] = cmp_ms
    # cfg4 batch
    seqs, lens = workloads.gc_rich_batch()
    flat, offsets, lens32 = workloads.pack_batch(seqs)
    fd, od = torch.from_numpy(flat).cuda(), torch.from_numpy(offsets).cuda()
    wsb = torch.empty(r8.workspace_bytes_batch(lens32), dtype=torch.uint8, device="cuda")
    sc = torch.empty(len(lens32), dtype=torch.int32, device="cuda")
    ms = time_call(lambda: r8.fold_batch(fd, od, lens32, scores_out=sc, workspace=wsb), 10)
    wtot = int(sum(nussinov_updates(int(x)) for x in lens32))
    ltot = int(sum(algorithmic_lookups(int(x), 8) for x in lens32))
    res["cfg4_batch1024_q8"] = {"ms": ms, "cell_k_updates_per_s": wtot / (ms * 1e-3), "fill_kernel_ms": r8.last_fill_kernel_ms(),
                               "lookups": ltot, "sum_scores": int(sc.sum().item()),
                               "engine": "smem (one CTA per sequence, one launch)" if r8.last_launch_count() == 1 else "tiled",
                               "kernel": "smemseq::seq_kernel<8,false,24>" if r8.last_launch_count() == 1 else "tiled::fill_kernel<8>"}
    # the same batch forced onto the long-sequence (tiled) engine: what the batch cost before the SMEM engine existed
    if r8.last_launch_count() == 1:
        rt = pkg.Rna4r(8, 0, pkg.ENGINE_TILED)
        res["cfg4_batch1024_q8"]["tiled_engine_ms"] = time_call(lambda: rt.fold_batch(fd, od, lens32, scores_out=sc, workspace=wsb), 5)
        rt.close()
    del wsb
    # the same batch end to end: pinned host buffers through rna4r_fold_batch_host, copies inside the timed region
    pinned = torch.from_numpy(flat).pin_memory()
    out_p = torch.zeros(len(lens32), dtype=torch.int32).pin_memory()
    wsh = torch.empty(r8.workspace_bytes_host(lens32), dtype=torch.uint8, device="cuda")
    for _ in range(3):
        r8.fold_batch_host(pinned, lens32, workspace=wsh, scores_host=out_p)
    t0 = time.perf_counter()
    for _ in range(10):
        r8.fold_batch_host(pinned, lens32, workspace=wsh, scores_host=out_p)
    e2e_s = (time.perf_counter() - t0) / 10
    res["cfg4_batch1024_q8"]["e2e"] = {"value": wtot / e2e_s, "unit": "cell-k-updates/s", "seconds_per_batch": e2e_s,
                                        "h2d_bytes_per_step": int(flat.size + 4 * len(lens32)), "d2h_bytes_per_step": int(4 * len(lens32)),
                                        "sum_scores": int(out_p.sum().item())}
    del wsh
    # cfg5
    s = workloads.single_config("cfg5")
    d = torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda()
    for q in (8, 10, 11):                      # q = 10 is BASELINE.json's second cfg5 point; q = 11 the last q of the tiled engine
        rr = r8 if q == 8 else pkg.Rna4r(q, 0)
        rr.enable_kernel_timing(True)
        ms = time_call(lambda: rr.fold(d), 3)
        res[f"cfg5_n16384_q{q}"] = {"ms": ms, "cell_k_updates_per_s": nussinov_updates(len(s)) / (ms * 1e-3),
                                    "fill_kernel_ms": rr.last_fill_kernel_ms(), "lookups": algorithmic_lookups(len(s), q)}
        if q != 8:
            rr.close()
    # cfg6: n = 32768 (beyond BASELINE.json's configs), score only
    s = workloads.single_config("cfg6")
    d = torch.from_numpy(np.frombuffer(s, dtype=np.uint8).copy()).cuda()
    ms = time_call(lambda: r8.fold(d), 2)
    res["cfg6_n32768_q8"] = {"ms": ms, "cell_k_updates_per_s": nussinov_updates(len(s)) / (ms * 1e-3),
                             "fill_kernel_ms": r8.last_fill_kernel_ms(), "lookups": algorithmic_lookups(len(s), 8)}
    return res


if __name__ == "__main__":
    main()
