#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on BASELINE.json's headline workload.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

A "step" is one pass of the whole hot path (DESIGN.md rows a0..a9: link costs, distances,
holdings/wants bitmaps, the event loop with candidate bitmap / pick / conflict resolve /
free-time advance, and the emitter) over one synthetic problem: by default config 4, the
8x8x8-torus 512-NPU All-to-All with 261,632 chunks (`configs[3]` of BASELINE.json, the
workload `metric` is quoted on).  Metric: link-chunk matches per second = transfers of the
synthesized schedule / synthesis time; synthesis seconds are reported beside it.

  value   inputs (topology + normalised conditions) resident in HBM, schedule left in HBM;
          timed per step with CUDA events on the launching stream, L2 flushed between steps.
  e2e     the same through pccl_synthesize with HOST buffers: normalise, host->device copies,
          all kernels, device->host copy of the schedule (streamed out in pieces on a copy
          stream while the event loop is still running), all inside the timed region.
  roofline  the event-loop kernel k_loop: bitmap bytes it requested / its CUDA-event time,
          against MEASURED_PEAKS.json's HBM copy bandwidth.
  cpu_baseline  the oracle, as it stands, one thread, on this box's host cores.

N > 1 (torchrun): replicas only -- every rank synthesizes the same problem with its own seed
(rank r uses seed r), no data-path collective; value = all ranks' matches / max-over-ranks time.
`--impl reference` times the CPU oracle (there is no reference implementation to install:
/root/reference holds only the paper's text).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "link-chunk matches/s, 512-NPU All-to-All synthesis"
UNIT = "matches/s"
KERNELS_PER_STEP_COPY = 8   # k_link_cost, k_distances, k_have, k_wants, k_sum_u32, k_loop_init, k_count_init, k_loop1


def workload(cfg: int, seed: int):
    import workloads as wl
    return wl.CONFIGS[cfg](seed)


def config_dict(p, cfg, extra=None):
    d = {"workload": f"config{cfg}:{p.name}", "n_npus": int(p.n_npus), "n_links": int(len(p.links)),
         "n_chunks": int(p.n_chunks), "chunk_bytes": int(p.chunk_bytes), "seed": int(p.seed),
         "l2": "flushed between timed steps (256 MiB write)"}
    if extra:
        d.update(extra)
    return d


# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.stop, self.th = index, [], threading.Event(), None

    def _run_nvml(self):
        import pynvml
        pynvml.nvmlInit()
        h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
        mx = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
        get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
        bits = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40}
        while not self.stop.is_set():
            sm = pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)
            r = int(get_reasons(h))
            row = [str(sm), str(mx), "0"] + [("Active" if r & bits[n] else "Not Active")
                                            for n in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")]
            self.rows.append(row)
            self.stop.wait(0.002)

    def _run(self):
        try:
            self._run_nvml()          # NVML: a sample every ~2 ms (the timed region is ~50 ms long)
            return
        except Exception:
            pass
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                for line in out.strip().splitlines():
                    self.rows.append([x.strip() for x in line.split(",")])
            except Exception:
                pass
            self.stop.wait(0.1)

    def __enter__(self):
        self.th = threading.Thread(target=self._run, daemon=True)
        self.th.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.th.join(timeout=10)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def lower_bound_ps(p):
    """Bandwidth lower bound of the collective time for COPY problems on homogeneous links (DESIGN.md
    "Lower bound"; harness arithmetic, not part of the method): max of the ingress bound
    max_v ceil(chunks v must receive / indeg v), the egress bound likewise, and the work bound
    ceil(sum over (chunk, dest) of hop distance / L) for single-dest chunks, times the link cost."""
    import numpy as np
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import shortest_path
    links = p.links
    if len(np.unique(links["alpha_ps"])) != 1 or len(np.unique(links["bytes_per_ps"])) != 1:
        return None
    w = int(links["alpha_ps"][0]) + -(-int(p.chunk_bytes) // int(links["bytes_per_ps"][0]))
    n = p.n_npus
    src_of = np.full(p.n_chunks, -1, dtype=np.int64)
    cnt = np.bincount(p.pre["chunk"], minlength=p.n_chunks)
    if cnt.max() != 1:
        return None                                    # reductions: not bounded here
    src_of[p.pre["chunk"]] = p.pre["npu"]
    need = p.post[src_of[p.post["chunk"]] != p.post["npu"]]          # (dest, chunk) that must be delivered
    indeg = np.bincount(links["dst"], minlength=n)
    outdeg = np.bincount(links["src"], minlength=n)
    need_in = np.bincount(need["npu"], minlength=n)
    has_dest = np.zeros(p.n_chunks, dtype=bool)
    has_dest[need["chunk"]] = True
    need_out = np.bincount(src_of[has_dest], minlength=n)
    with np.errstate(divide="ignore", invalid="ignore"):
        ingress = int(np.nanmax(np.where(need_in > 0, np.ceil(need_in / np.maximum(indeg, 1)), 0)))
        egress = int(np.nanmax(np.where(need_out > 0, np.ceil(need_out / np.maximum(outdeg, 1)), 0)))
    bound = max(ingress, egress)
    per_chunk = np.bincount(need["chunk"], minlength=p.n_chunks)
    if per_chunk.max() == 1:                            # single-dest chunks: every hop of a shortest path is a transfer
        g = csr_matrix((np.ones(len(links)), (links["src"], links["dst"])), shape=(n, n))
        hops = shortest_path(g, method="D", unweighted=True)
        total = int(hops[src_of[need["chunk"]], need["npu"]].sum())
        bound = max(bound, -(-total // len(links)))
    return bound * w


def time_oracle(p, budget_s: float, max_runs: int):
    """Oracle wall times (its own steady-clock seconds) for up to max_runs runs within budget_s."""
    import oracle
    secs, m = [], 0
    t0 = time.perf_counter()
    for _ in range(max_runs):
        r = oracle.synthesize(*p.args())
        secs.append(r.seconds)
        m = len(r.transfers)
        if time.perf_counter() - t0 + secs[-1] > budget_s:
            break
    return secs, m


# ---------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    p = workload(args.config, 0)
    import oracle
    oracle.build()
    warm, _ = time_oracle(p, 60.0, max(0, min(args.warmup, 1)))   # the oracle has no warm-up effects worth more
    secs, m = time_oracle(p, 200.0, args.steps)
    k = len(secs)
    tot = sum(secs)
    val = m * k / tot
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": k, "warmup": len(warm), "ms_per_step": 1e3 * tot / k, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": config_dict(p, args.config, {"note": "CPU oracle (oracle/pccl_oracle.cpp), 1 thread, "
                                                   "whole workload per step; steps capped by a 200 s budget"}),
            "synthesis_s": tot / k,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "sample": f"the whole config{args.config} problem, {k} run(s)", "host_cores": os.cpu_count()},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2606_07019_b200 as pk
    pk.use_torch(local)

    seed = rank                      # replicas: same problem, one seed per rank
    p = workload(args.config, seed)
    topo = pk.Topology(p.n_npus, p.links)
    prob = pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)
    prob.upload()                    # inputs resident in HBM before the timed region
    flags = pk.PCCL_FLAG_KEEP_ON_DEVICE | pk.PCCL_FLAG_TIME_LOOP
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def one_step():
        flush.zero_()                # evict L2 (126 MB) between steps; outside the events
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        s = prob.synthesize(seed, flags)
        e1.record()
        e1.synchronize()
        return s, e0.elapsed_time(e1)

    for _ in range(args.warmup):
        s, _ = one_step()
        s.close()
    barrier()
    step_ms, loop_ms, stats, M, T = [], [], None, 0, 0
    wall0 = time.perf_counter()
    with ClockSampler(local) as clk:
        for _ in range(args.steps):
            s, ms = one_step()
            step_ms.append(ms)
            stats = s.stats
            loop_ms.append(stats["loop_ms"])
            M, T = s.size, s.time_ps
            s.close()
        barrier()
    wall = time.perf_counter() - wall0
    tot_ms = sum(step_ms)
    if world > 1:
        t = torch.tensor([tot_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        m = torch.tensor([M * args.steps], dtype=torch.float64, device="cuda")
        dist.all_reduce(m, op=dist.ReduceOp.SUM)
        tot_ms_max, matches_all = float(t.item()), float(m.item())
    else:
        tot_ms_max, matches_all = tot_ms, float(M * args.steps)
    value = matches_all / (tot_ms_max * 1e-3)

    # ---- e2e: host buffers through pccl_synthesize, copies inside the timed region ----------
    def one_e2e():
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        s = pk.synthesize(*p.args())
        tr_ptr = pk.lib.pccl_schedule_transfers(s.handle)   # already on the host (eager download)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        assert tr_ptr or s.size == 0
        n = s.size
        s.close()
        return dt, n
    for _ in range(min(args.warmup, 3)):
        one_e2e()
    barrier()
    e2e_s = [one_e2e()[0] for _ in range(args.steps)]
    barrier()
    e2e_tot = sum(e2e_s)
    if world > 1:
        t = torch.tensor([e2e_tot], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_tot = float(t.item())
    e2e_val = matches_all / e2e_tot
    h2d = p.links.nbytes + p.group.nbytes + p.pre.nbytes + p.post.nbytes
    d2h = M * 32

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (k_loop) ------------------------------------------------
    peaks, peak_src = None, "fallback (B200_PROFILING.md: 6650 GB/s)"
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peaks = json.load(f)
        peak, peak_src = float(peaks["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        peak = 6650.0
    loop_avg_ms = sum(loop_ms) / len(loop_ms)
    alg_bytes = stats["rows_scanned"] * stats["row_bytes"]     # bitmap rows the kernel requested x padded row bytes
    achieved = alg_bytes / (loop_avg_ms * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "k_loop_traffic.txt")   # from the committed ncu --set full capture
    if os.path.exists(tpath):
        for ln in open(tpath):
            f = ln.split()
            if len(f) == 2 and f[0] == f"config{args.config}":
                traffic = int(f[1])
    req_bytes = stats["bytes_requested"]
    roofline = {"bound": "hbm", "kernel": "k_loop1 (one-barrier event loop, kept counts)", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": loop_avg_ms,
                "kernel_share_of_step": loop_avg_ms / (tot_ms / args.steps),
                "frac_of_8TBps_nominal": achieved / 8000.0,
                "requested_bytes_per_launch": req_bytes,
                "requested_gbs": req_bytes / (loop_avg_ms * 1e-3) / 1e9,
                "note": "algorithmic bytes = SURVEY 8(d): padded row bytes x (destinations + in-links swept), counted "
                        "by the kernel (rows_scanned x row_bytes): what a per-event recount of every free link would "
                        "read. The default kernel keeps the per-segment candidate counts current instead (arrivals "
                        "add, claims subtract) and requests only requested_bytes, so achieved can exceed the HBM "
                        "peak and the loop is bound by grid barriers and dependent L2 round trips, not bandwidth. "
                        "two_barrier_kept_counts, rescan_sector_list and dense_sweep below are the two-barrier loop "
                        "k_loop with kept counts and recounting at every event (PCCL_FLAG_TWO_BARRIERS / _RESCAN / "
                        "_DENSE_SWEEP); dense_sweep is the plain memory-bound bitmap scan. At config 4 both bitmaps (2 x 16.8 MB) sit in the 126 MB L2, so DRAM traffic is far "
                        "below all of these figures"}
    # the two-barrier loop (k_loop) with kept counts, and recounting candidates at every event, timed the same way
    for key, fl in (("two_barrier_kept_counts", pk.PCCL_FLAG_TWO_BARRIERS), ("rescan_sector_list", pk.PCCL_FLAG_RESCAN),
                    ("dense_sweep", pk.PCCL_FLAG_DENSE_SWEEP)):
        ms_v, stv = [], None
        for i in range(2 + min(args.steps, 5)):
            flush.zero_()
            sv = prob.synthesize(seed, flags | fl)
            stv = sv.stats
            sv.close()
            if i >= 2:
                ms_v.append(stv["loop_ms"])
        mv = sum(ms_v) / len(ms_v)
        algv = stv["rows_scanned"] * stv["row_bytes"]
        roofline[key] = {"kernel_ms": mv, "requested_bytes_per_launch": stv["bytes_requested"],
                         "requested_gbs": stv["bytes_requested"] / (mv * 1e-3) / 1e9,
                         "algorithmic_bytes_per_launch": algv, "achieved": algv / (mv * 1e-3) / 1e9, "unit": "GB/s",
                         "frac": algv / (mv * 1e-3) / 1e9 / peak}
    # ---- the dynamic relay rule (Q18) on the same problem: schedule quality vs cost ----
    dynamic = None
    if not args.no_other_configs:
        ms_d, sd = [], None
        for i in range(3):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sd = prob.synthesize(seed, flags | pk.PCCL_FLAG_DYNAMIC_RELAY)
            e1.record()
            e1.synchronize()
            if i >= 1:
                ms_d.append(e0.elapsed_time(e1))
            dM, dT, dst = sd.size, sd.time_ps, sd.stats
            sd.close()
        dynamic = {"synthesis_ms": sum(ms_d) / len(ms_d), "loop_ms": dst["loop_ms"], "transfers": dM,
                   "events": dst["events"], "schedule_time_ps": dT,
                   "schedule_time_vs_thin_tree": dT / T if T else None,
                   "initial_wants": dst["wants_total"],
                   "counting": "kept counts + per-chunk holder lists (the rule's default)"}
        # the same rule recounting by the dense sweep and dropping every stale wants bit at once (cross-check mode)
        sd = prob.synthesize(seed, flags | pk.PCCL_FLAG_DYNAMIC_RELAY | pk.PCCL_FLAG_DENSE_SWEEP)
        assert (sd.size, sd.time_ps) == (dM, dT)
        dynamic["dense_sweep_loop_ms"] = sd.stats["loop_ms"]
        sd.close()

    # ---- the paper's own per-condition synthesizer (PCCL_FLAG_BFS; Q19-Q22) on the same problem
    bfs = None
    if not args.no_other_configs:
        ms_b = []
        for i in range(3):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sb = prob.synthesize(seed, flags | pk.PCCL_FLAG_BFS)
            e1.record()
            e1.synchronize()
            if i >= 1:
                ms_b.append(e0.elapsed_time(e1))
            bM, bT, bst = sb.size, sb.time_ps, sb.stats
            sb.close()
        bms = sum(ms_b) / len(ms_b)
        bfs = {"synthesis_ms": bms, "loop_ms": bst["loop_ms"], "conditions": bst["events"], "transfers": bM,
               "conditions_per_s": bst["events"] / (bms * 1e-3), "searches": bst["rows_scanned"],
               "link_relaxations": bst["links_scanned"], "commit_rounds": bst["slow_picks"], "window": bst["grid_blocks"],
               "schedule_time_ps": bT, "schedule_time_vs_matching": bT / T if T else None,
               "schedule_time_over_lower_bound": (bT / lower_bound_ps(p)) if lower_bound_ps(p) else None,
               "bound": "latency: ~10 dependent sweeps per search, one L2 round trip or more each; see DESIGN.md"}

    # ---- the other BASELINE.json configs, same path, resident inputs (context; parity is in tests/) ---
    per_config = {}
    if not args.no_other_configs:
        for cfg in (1, 2, 3, 5):
            if cfg == args.config:
                continue
            pc = workload(cfg, 0)
            tc = pk.Topology(pc.n_npus, pc.links)
            prc = pk.Problem(tc, pc.group, pc.n_chunks, pc.pre, pc.post, pc.chunk_bytes)
            prc.upload()
            ms_l, sc = [], None
            for i in range(4):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                sc = prc.synthesize(0, flags)
                e1.record()
                e1.synchronize()
                if i >= 1:
                    ms_l.append((e0.elapsed_time(e1), sc.stats))
                mc, tcps = sc.size, sc.time_ps
                sc.close()
            ms_c, stc = sorted(ms_l, key=lambda x: x[0])[len(ms_l) // 2]   # the median run and ITS loop time
            algb = stc["rows_scanned"] * stc["row_bytes"]
            per_config[f"config{cfg}"] = {
                "workload": pc.name, "synthesis_ms": ms_c, "loop_ms": stc["loop_ms"], "transfers": mc,
                "matches_per_s": mc / (ms_c * 1e-3), "events": stc["events"], "schedule_time_ps": tcps,
                "algorithmic_gbs": algb / (stc["loop_ms"] * 1e-3) / 1e9 if stc["loop_ms"] else None,
                "frac_of_measured_hbm": (algb / (stc["loop_ms"] * 1e-3) / 1e9 / peak) if stc["loop_ms"] else None,
                "requested_bytes": stc["bytes_requested"],
                "schedule_time_over_lower_bound": (tcps / lower_bound_ps(pc)) if lower_bound_ps(pc) else None,
                "roofline_note": "rows of 128 B: launch/sync-bound, roofline n/a" if stc["row_bytes"] <= 256 else "bitmap scan"}
            if stc["row_bytes"] > 256:   # a real bitmap scan: the two recount modes beside the default
                for key, fl in (("rescan_sector_list", pk.PCCL_FLAG_RESCAN), ("dense_sweep", pk.PCCL_FLAG_DENSE_SWEEP)):
                    flush.zero_()
                    sv = prc.synthesize(0, flags | fl)
                    stv = sv.stats
                    sv.close()
                    algv = stv["rows_scanned"] * stv["row_bytes"]
                    per_config[f"config{cfg}"][key] = {
                        "loop_ms": stv["loop_ms"], "requested_bytes": stv["bytes_requested"],
                        "algorithmic_gbs": algv / (stv["loop_ms"] * 1e-3) / 1e9,
                        "frac_of_measured_hbm": algv / (stv["loop_ms"] * 1e-3) / 1e9 / peak}
            prc.close()
            tc.close()

    # ---- cpu baseline: the oracle on this box's host cores ----------------------------------------
    cpu = None
    if not args.no_cpu_baseline:
        p0 = workload(args.config, seed)
        secs, m = time_oracle(p0, 30.0, 1)
        cpu = {"value": m / secs[0], "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"the whole config{args.config} problem once ({secs[0]:.2f} s, single thread)",
               "host_cores": os.cpu_count(), "seconds": secs[0]}

    lb = lower_bound_ps(p)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tot_ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": config_dict(p, args.config, {"parallelism": "replicas" if world > 1 else "single"}),
            "synthesis_s": tot_ms_max / args.steps * 1e-3,
            "transfers": M, "events": stats["events"], "schedule_time_ps": T,
            "schedule_time_over_lower_bound": (T / lb) if lb else None,
            "phases_ms": {"setup": stats["setup_ms"], "loop": loop_avg_ms, "emit": stats["emit_ms"]},
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": 1e3 * e2e_tot / args.steps},
            "gpu_launches": KERNELS_PER_STEP_COPY * args.steps,
            "roofline": roofline, "cpu_baseline": cpu, "clocks": clk.summary(), "per_config": per_config, "dynamic_relay": dynamic, "paper_bfs": bfs,
            "paper_context": "PCCL reports 11.68 min for 512-NPU All-to-All synthesis, hardware not stated "
                             "(PAPER.md:9, :388); a different procedure, context only",
            "wall_s_timed_region": wall}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_fig12(args):
    """Context run shaped like the paper's Fig. 12: All-to-All on 64 NPUs (8x8 mesh and
    4x4x4 torus), 128 KiB chunks, 1..64 chunks per (source, destination) pair, i.e. 8..512 MiB per NPU.  The
    paper reports 1.83 min for the 512 MiB point on its (unstated) host with its BFS procedure."""
    import numpy as np
    import torch
    import paper_2606_07019_b200 as pk
    import workloads as wl
    pk.use_torch(0)
    rows = []
    for name, dims, wrap in (("mesh8x8", (8, 8), False), ("torus4x4x4", (4, 4, 4), True)):
        links = wl.grid_links(dims, wrap=wrap)
        members = np.arange(64, dtype=np.uint32)
        topo = pk.Topology(64, links)
        for k in (1, 2, 4, 8, 16, 32, 64):
            nc, pre, post = wl.all_to_all(members, np.full((64, 64), k))
            prob = pk.Problem(topo, members, nc, pre, post, 128 << 10)
            prob.upload()
            ms = []
            for i in range(4):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                s = prob.synthesize(0, pk.PCCL_FLAG_KEEP_ON_DEVICE)
                e1.record()
                e1.synchronize()
                if i:
                    ms.append(e0.elapsed_time(e1))
                m, t, ev = s.size, s.time_ps, s.stats["events"]
                s.close()
            msb = []
            for i in range(2):   # the paper's own procedure (PCCL_FLAG_BFS) on the same problem
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                sb = prob.synthesize(0, pk.PCCL_FLAG_KEEP_ON_DEVICE | pk.PCCL_FLAG_BFS)
                e1.record()
                e1.synchronize()
                msb.append(e0.elapsed_time(e1))
                mb, tb, rb = sb.size, sb.time_ps, sb.stats["slow_picks"]
                sb.close()
            rows.append({"topology": name, "chunks_per_pair": k, "mib_per_npu": k * 64 * 128 // 1024, "chunks": nc,
                         "transfers": m, "events": ev, "synthesis_ms": sorted(ms)[1], "schedule_time_ps": t,
                         "bfs_synthesis_ms": min(msb), "bfs_transfers": mb, "bfs_rounds": rb, "bfs_schedule_time_ps": tb})
            prob.close()
        topo.close()
    print(json.dumps({"experiment": "fig12-shaped chunks-per-NPU sweep (context)", "rows": rows}), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--fig12", action="store_true", help="chunks-per-NPU sweep shaped like the paper's Fig. 12")
    args = ap.parse_args()
    if args.fig12:
        return run_fig12(args)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
