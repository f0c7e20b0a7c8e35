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
  roofline  the dominant kernel, the barrier-free event loop k_loop2: bytes it REQUESTED / its
          own CUDA-event time against MEASURED_PEAKS.json's HBM copy bandwidth -- it is latency
          bound and says so; the memory-bound form of the same work (the streaming candidate
          sweep, rows staged by TMA bulk copies) is timed beside it against the HBM peak and
          against the L2 / HBM read ceilings measured in the same run (pccl_device_read_bandwidth).
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


def workload(cfg: int, seed: int):
    import workloads as wl
    return wl.CONFIGS[cfg](seed)


def workload_big():
    """config 5's recipe on a 28x28 torus with every node in the group: 1.13 M chunks, bitmaps of 2 x 160 MB -- a working
    set the 126 MB L2 cannot hold, for the HBM-bound measurement of the candidate sweep"""
    import workloads as wl
    return wl.config5(0, dims=(28, 28), group_size=784)


def config_dict(p, cfg):
    """the workload, identical on the `ours` and `reference` arms"""
    return {"workload": f"config{cfg}:{p.name}", "n_npus": int(p.n_npus), "n_links": int(len(p.links)),
            "n_chunks": int(p.n_chunks), "chunk_bytes": int(p.chunk_bytes), "seed": int(p.seed)}


# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.stop, self.th = index, [], threading.Event(), None

    def _init_nvml(self):
        """NVML is initialised by the caller's thread BEFORE the timed region starts (nvmlInit alone can take longer than
        the whole region), so the sampling thread only reads."""
        import pynvml
        pynvml.nvmlInit()
        h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
        mx = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
        get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
        pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)      # fail here, not in the thread
        int(get_reasons(h))
        self.nvml = (pynvml, h, mx, get_reasons)

    def _sample_nvml(self):
        pynvml, h, mx, get_reasons = self.nvml
        bits = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40}
        sm = pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)
        r = int(get_reasons(h))
        self.rows.append([str(sm), str(mx), "0"] + [("Active" if r & bits[n] else "Not Active")
                                                    for n in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")])

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                              "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
        for line in out.strip().splitlines():
            self.rows.append([x.strip() for x in line.split(",")])

    def _run(self):
        # NVML: a sample every ~2 ms (the timed region is some tens of ms long); nvidia-smi (~100 ms a call) otherwise
        while True:
            try:
                if self.nvml is not None:
                    self._sample_nvml()
                else:
                    self._sample_smi()
            except Exception:
                pass
            if self.stop.wait(0.002 if self.nvml is not None else 0.1):
                return

    def __enter__(self):
        self.nvml = None
        try:
            self._init_nvml()
        except Exception:
            self.nvml = None
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


def _machines_bound(k: int, costs) -> int:
    """least T such that k transfers fit on parallel links with per-transfer costs `costs` (each link carries one chunk
    at a time): sum_i floor(T / w_i) >= k."""
    if k <= 0:
        return 0
    costs = [int(c) for c in costs]
    if not costs:
        return 0
    lo, hi = 0, k * min(costs)
    while lo < hi:
        mid = (lo + hi) // 2
        if sum(mid // c for c in costs) >= k:
            hi = mid
        else:
            lo = mid + 1
    return lo


def _copy_bound(n, src_l, dst_l, w, cond_src, dests_of):
    """bandwidth lower bound of a COPY phase (harness arithmetic, not part of the method): every chunk a node must
    receive enters over one of its in-links and every chunk with a dest elsewhere leaves its source over one of the
    source's out-links -- the exact parallel-links bound above (alpha-beta costs), i.e. bytes over the
    node's summed link bandwidth rounded to whole transfers; on homogeneous links with single-dest chunks also the work
    bound ceil(sum of hop distances / L) * w."""
    import numpy as np
    need_in = np.zeros(n, dtype=np.int64)
    need_out = np.zeros(n, dtype=np.int64)
    for c, ds in dests_of.items():
        if ds:
            need_out[cond_src[c]] += 1
            for d in ds:
                need_in[d] += 1
    in_costs = [[] for _ in range(n)]
    out_costs = [[] for _ in range(n)]
    for s_, d_, c_ in zip(src_l, dst_l, w):
        out_costs[int(s_)].append(int(c_))
        in_costs[int(d_)].append(int(c_))
    bound = 0
    for v in range(n):
        bound = max(bound, _machines_bound(int(need_in[v]), in_costs[v]), _machines_bound(int(need_out[v]), out_costs[v]))
    # the same argument across a cut: nodes joined by links cheaper than the dearest class form clusters (the pods of
    # config 3); a chunk sourced outside a cluster with a dest inside must cross one of the links into it, and vice versa
    wmax = max((int(c) for c in w), default=0)
    parent = list(range(n))

    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x
    for s_, d_, c_ in zip(src_l, dst_l, w):
        if int(c_) < wmax:
            parent[find(int(s_))] = find(int(d_))
    comp = [find(v) for v in range(n)]
    if len(set(comp)) < n:
        cut_in, cut_out, k_in, k_out = {}, {}, {}, {}
        for s_, d_, c_ in zip(src_l, dst_l, w):
            a, b = comp[int(s_)], comp[int(d_)]
            if a != b:
                cut_out.setdefault(a, []).append(int(c_))
                cut_in.setdefault(b, []).append(int(c_))
        for c, ds in dests_of.items():
            a = comp[cond_src[c]]
            outside = {comp[d] for d in ds} - {a}
            if outside:
                k_out[a] = k_out.get(a, 0) + 1
            for b in outside:
                k_in[b] = k_in.get(b, 0) + 1
        for b, k in k_in.items():
            bound = max(bound, _machines_bound(k, cut_in.get(b, [])))
        for a, k in k_out.items():
            bound = max(bound, _machines_bound(k, cut_out.get(a, [])))
    # no chunk arrives before its shortest alpha-beta path allows
    if len(w):
        from scipy.sparse import csr_matrix
        from scipy.sparse.csgraph import dijkstra
        best = {}
        for s_, d_, c_ in zip(src_l, dst_l, w):
            k = (int(s_), int(d_))
            best[k] = min(best.get(k, 1 << 62), int(c_))
        rows, cols = zip(*best.keys())
        g = csr_matrix((np.array(list(best.values()), dtype=np.float64), (rows, cols)), shape=(n, n))
        srcs = sorted({cond_src[c] for c, ds in dests_of.items() if ds})
        if srcs:
            dist = dijkstra(g, directed=True, indices=srcs)
            row = {s_: i for i, s_ in enumerate(srcs)}
            far = max(dist[row[cond_src[c]], d] for c, ds in dests_of.items() for d in ds)
            if np.isfinite(far):
                bound = max(bound, int(far))
    if len(set(int(x) for x in w)) == 1 and all(len(ds) <= 1 for ds in dests_of.values()) and len(w):
        from scipy.sparse import csr_matrix
        from scipy.sparse.csgraph import shortest_path
        g = csr_matrix((np.ones(len(w)), (src_l, dst_l)), shape=(n, n))
        hops = shortest_path(g, method="D", unweighted=True)
        total = int(sum(hops[cond_src[c], ds[0]] for c, ds in dests_of.items() if ds))
        bound = max(bound, -(-total // len(w)) * int(w[0]))
    return bound


def lower_bound_ps(p):
    """Bandwidth lower bound of the synthesized collective time for any of the three modes.
    A reduction is bounded through its reversed broadcast on the transposed links; an all-reduce, which
    this build composes sequentially (T = T_reduce + T_copy), by the sum of its two phases' bounds."""
    import numpy as np
    links = p.links
    w = [int(a) + -(-int(p.chunk_bytes) // int(b)) for a, b in zip(links["alpha_ps"], links["bytes_per_ps"])]
    n, C = p.n_npus, p.n_chunks
    pre = [set() for _ in range(C)]
    post = [set() for _ in range(C)]
    for r in p.pre:
        pre[int(r["chunk"])].add(int(r["npu"]))
    for r in p.post:
        post[int(r["chunk"])].add(int(r["npu"]))
    fwd = (links["src"], links["dst"])
    rev = (links["dst"], links["src"])
    if all(len(x) == 1 for x in pre):                                   # copy
        src = {c: next(iter(pre[c])) for c in range(C)}
        return _copy_bound(n, *fwd, w, src, {c: sorted(post[c] - {src[c]}) for c in range(C)})
    if all(len(pre[c]) > 1 and len(post[c]) == 1 for c in range(C)):    # reduce / reduce-scatter
        root = {c: next(iter(post[c])) for c in range(C)}
        return _copy_bound(n, *rev, w, root, {c: sorted(pre[c] - {root[c]}) for c in range(C)})
    if all(len(pre[c]) > 1 and len(post[c]) > 1 for c in range(C)):     # all-reduce: roots as in DESIGN.md step R
        root = {}
        for c in range(C):
            inter = sorted(pre[c] & post[c]) or sorted(post[c])
            root[c] = inter[c % len(inter)]
        b1 = _copy_bound(n, *rev, w, root, {c: sorted(pre[c] - {root[c]}) for c in range(C)})
        b2 = _copy_bound(n, *fwd, w, root, {c: sorted(post[c] - {root[c]}) for c in range(C)})
        return b1 + b2
    return None


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
            "config": config_dict(p, args.config),
            "note": "CPU oracle (oracle/pccl_oracle.cpp), 1 thread, whole workload per step; steps capped by a 200 s budget",
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
    launches0 = pk.launch_count()
    with ClockSampler(local) as clk:
        for _ in range(args.steps):
            s, ms = one_step()
            step_ms.append(ms)
            stats = s.stats
            loop_ms.append(stats["loop_ms"])
            M, T = s.size, s.time_ps
            s.close()
        barrier()
    launches_timed = pk.launch_count() - launches0      # the library counts every kernel launch where it issues it
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

    # ---- roofline of the dominant kernel: the barrier-free event loop k_loop2 --------------------------------
    peak_src = "fallback (B200_PROFILING.md: 6650 GB/s)"
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peak = float(json.load(f)["hbm_gbs"])
        peak_src = "measured (MEASURED_PEAKS.json hbm_gbs: copy, read + write bytes)"
    except Exception:
        peak = 6650.0
    # ceilings of the level that serves a bitmap sweep, measured in this run with the library's own read kernel
    # (128-bit ld.global.cg, the sweeps' access pattern): a 96 MiB buffer stays in the 126 MB L2, a 4 GiB one does not
    l2_read = pk.read_bandwidth_gbs(96 << 20, 30)
    hbm_read = pk.read_bandwidth_gbs(4 << 30, 5)
    loop_avg_ms = sum(loop_ms) / len(loop_ms)
    req_bytes = stats["bytes_requested"]
    achieved = req_bytes / (loop_avg_ms * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "k_loop_traffic.txt")   # dram__bytes_read + write per launch, from the committed ncu --set full capture
    if os.path.exists(tpath):
        for ln in open(tpath):
            f = ln.split()
            if len(f) >= 2 and f[0] == f"config{args.config}":
                traffic = int(f[1])
    dense_eq = stats["events"] * (p.n_npus + len(p.links)) * stats["row_bytes"]
    roofline = {"bound": "latency", "kernel": "k_loop2 (barrier-free event loop: one warp per destination, claim logs)",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "peak_source": peak_src, "kernel_ms": loop_avg_ms,
                "kernel_share_of_step": loop_avg_ms / (tot_ms / args.steps),
                "requested_bytes_per_launch": req_bytes,
                "frac_of_8TBps_nominal": achieved / 8000.0,
                "us_per_event": 1e3 * loop_avg_ms / max(1, stats["events"]),
                "measured_ceilings_gbs": {"l2_read_96MiB": l2_read, "hbm_read_4GiB": hbm_read, "hbm_copy": peak},
                "dense_equivalent": {"bytes_per_launch": dense_eq, "gbs": dense_eq / (loop_avg_ms * 1e-3) / 1e9,
                                     "meaning": "SURVEY 8(d)'s upper envelope, events x (N + L) x row bytes: what a recount of every "
                                                "link at every event would read; NOT traffic of this kernel and not a roofline fraction"},
                "note": "achieved = bytes the kernel requested (headers, log entries, translation words; counted by the kernel) / "
                        "its own CUDA-event time. The loop keeps every destination's candidate sets in shared memory and touches "
                        "no bitmap, so it is bound by dependent L2 round trips between neighbouring destinations (two per event) "
                        "and single-warp instruction latency, not by bandwidth. memory_bound_form is the same a5 work as a "
                        "streaming kernel; barrier_loops are the lockstep loops that recount or keep counts per event."}
    # ---- the memory-bound form: the streaming candidate sweep (row a5) alone, TMA-staged and per-lane loads ------
    sweeps = {}
    big = None
    if not args.no_other_configs:
        big = workload_big()
    for name, pw in ((f"config{args.config}", p), ("config5", workload(5, 0) if args.config != 5 and not args.no_other_configs else None),
                     ("torus28x28_alltoallv_784 (bitmaps 2 x 160 MB > L2)", big)):
        if pw is None:
            continue
        tw = pk.Topology(pw.n_npus, pw.links)
        prw = pk.Problem(tw, pw.group, pw.n_chunks, pw.pre, pw.post, pw.chunk_bytes)
        entry = {"chunks": int(pw.n_chunks), "bitmap_bytes_both": None}
        for key, fl in (("tma_bulk_staging", 0), ("per_lane_128bit_loads", pk.PCCL_FLAG_LSU_SWEEP)):
            ms, nbytes, tot = prw.candidate_sweep(0, 0, fl, iters=20)
            gbs = nbytes / (ms * 1e-3) / 1e9
            entry[key] = {"kernel_ms": ms, "algorithmic_bytes_per_launch": nbytes, "achieved": gbs, "unit": "GB/s",
                          "frac_of_measured_hbm_copy": gbs / peak, "frac_of_measured_l2_read": gbs / l2_read,
                          "frac_of_measured_hbm_read": gbs / hbm_read}
        row_b = ((pw.n_chunks + 63) // 64 + 15) // 16 * 16 * 8
        entry["bitmap_bytes_both"] = 2 * pw.n_npus * row_b
        entry["served_by"] = "L2" if entry["bitmap_bytes_both"] < (100 << 20) else "HBM (+ L2 reuse of have rows read by several links)"
        sweeps[name] = entry
        prw.close()
        tw.close()
    roofline["memory_bound_form"] = {"kernel": "k_count_sweep (candidate bitmap of every link, (N + L) rows per launch)",
                                     "bound": "hbm", "per_workload": sweeps}
    # ---- the lockstep loops on the same problem, timed the same way (loop kernel alone) ------------------------
    barrier = {}
    for key, fl in (("one_barrier_kept_counts", pk.PCCL_FLAG_BARRIER_LOOP), ("two_barrier_kept_counts", pk.PCCL_FLAG_TWO_BARRIERS),
                    ("rescan_sector_list", pk.PCCL_FLAG_RESCAN), ("dense_sweep", pk.PCCL_FLAG_DENSE_SWEEP)):
        ms_v, stv = [], None
        for i in range(2 + min(args.steps, 5)):
            flush.zero_()
            sv = prob.synthesize(seed, flags | fl)
            stv = sv.stats
            sv.close()
            if i >= 2:
                ms_v.append(stv["loop_ms"])
        mv = sum(ms_v) / len(ms_v)
        rq = stv["bytes_requested"] / (mv * 1e-3) / 1e9
        barrier[key] = {"kernel_ms": mv, "requested_bytes_per_launch": stv["bytes_requested"], "requested_gbs": rq,
                        "frac_of_measured_hbm_copy": rq / peak, "frac_of_measured_l2_read": rq / l2_read,
                        "us_per_event": 1e3 * mv / max(1, stv["events"])}
    roofline["barrier_loops"] = barrier
    lb = lower_bound_ps(p)
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
                   "schedule_time_over_lower_bound": (dT / lb) if lb else None,
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
               "schedule_time_over_lower_bound": (bT / lb) if lb else None,
               "bound": "latency: ~10 dependent sweeps per search, one L2 round trip or more each; see DESIGN.md"}

    # ---- NEXT-4 variants: the c.dist-priority pick on the same problem; the pipelined All-Reduce on config 2 (BFS mode) ----
    variants = None
    if not args.no_other_configs:
        ms_v = []
        for i in range(3):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sv = prob.synthesize(seed, flags | pk.PCCL_FLAG_DIST_PICK)
            e1.record()
            e1.synchronize()
            if i >= 1:
                ms_v.append(e0.elapsed_time(e1))
            vT, vst = sv.time_ps, sv.stats
            sv.close()
        variants = {"dist_pick": {"synthesis_ms": sum(ms_v) / len(ms_v), "loop_kernel_ms": vst["loop_ms"], "schedule_time_ps": vT,
                                  "schedule_time_vs_uniform_pick": vT / T if T else None,
                                  "schedule_time_over_lower_bound": (vT / lb) if lb else None}}
        p2 = workload(2, 0)
        t2 = pk.Topology(p2.n_npus, p2.links)
        pr2 = pk.Problem(t2, p2.group, p2.n_chunks, p2.pre, p2.post, p2.chunk_bytes)
        sq = pr2.synthesize(0, flags | pk.PCCL_FLAG_BFS)
        pl = pr2.synthesize(0, flags | pk.PCCL_FLAG_BFS | pk.PCCL_FLAG_PIPELINE)
        variants["pipelined_allreduce_config2_bfs"] = {"sequential_T_ps": sq.time_ps, "pipelined_T_ps": pl.time_ps,
                                                       "ratio": pl.time_ps / sq.time_ps, "reduce_phase_T_ps": pl.stats["time_phase1_ps"]}
        sq.close(); pl.close(); pr2.close(); t2.close()

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
            lbc = lower_bound_ps(pc)
            per_config[f"config{cfg}"] = {
                "workload": pc.name, "synthesis_ms": ms_c, "loop_kernel_ms": stc["loop_ms"], "transfers": mc,
                "matches_per_s": mc / (ms_c * 1e-3), "events": stc["events"], "schedule_time_ps": tcps,
                "us_per_event": 1e3 * stc["loop_ms"] / max(1, stc["events"]),
                "requested_bytes": stc["bytes_requested"],
                "requested_gbs": stc["bytes_requested"] / (stc["loop_ms"] * 1e-3) / 1e9 if stc["loop_ms"] else None,
                "lower_bound_ps": lbc, "schedule_time_over_lower_bound": (tcps / lbc) if lbc else None,
                "bound": "latency (dependent L2 round trips between neighbouring destinations)"}
            if stc["row_bytes"] > 256:   # a real bitmap scan: the lockstep loops beside the default
                for key, fl in (("one_barrier_kept_counts", pk.PCCL_FLAG_BARRIER_LOOP), ("rescan_sector_list", pk.PCCL_FLAG_RESCAN),
                                ("dense_sweep", pk.PCCL_FLAG_DENSE_SWEEP)):
                    flush.zero_()
                    sv = prc.synthesize(0, flags | fl)
                    stv = sv.stats
                    sv.close()
                    rq = stv["bytes_requested"] / (stv["loop_ms"] * 1e-3) / 1e9
                    per_config[f"config{cfg}"][key] = {
                        "loop_kernel_ms": stv["loop_ms"], "requested_bytes": stv["bytes_requested"], "requested_gbs": rq,
                        "frac_of_measured_hbm_copy": rq / peak, "frac_of_measured_l2_read": rq / l2_read}
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

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tot_ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": config_dict(p, args.config), "parallelism": "replicas" if world > 1 else "single",
            "l2": "flushed between timed steps (256 MiB write)",
            "synthesis_s": tot_ms_max / args.steps * 1e-3,
            "transfers": M, "events": stats["events"], "schedule_time_ps": T,
            "schedule_time_over_lower_bound": (T / lb) if lb else None,
            "lower_bound_ps": lb,
            "phases_ms": {"setup": stats["setup_ms"], "loop_kernel": loop_avg_ms, "emit": stats["emit_ms"]},
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": 1e3 * e2e_tot / args.steps},
            "gpu_launches": launches_timed,
            "roofline": roofline, "cpu_baseline": cpu, "clocks": clk.summary(), "per_config": per_config, "dynamic_relay": dynamic, "paper_bfs": bfs, "variants": variants,
            "paper_context": "PCCL reports 11.68 min for 512-NPU All-to-All synthesis, hardware not stated "
                             "(PAPER.md:9, :388); a different procedure, context only",
            "wall_s_timed_region": wall}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


CASES = {"default": 0, "barrier_loop": "BARRIER_LOOP", "two_barriers": "TWO_BARRIERS", "rescan": "RESCAN", "dense_sweep": "DENSE_SWEEP",
         "dynamic": "DYNAMIC_RELAY", "dynamic_dense": "DYNAMIC_RELAY|DENSE_SWEEP", "bfs": "BFS", "sweep_tma": None, "sweep_lsu": None}


def run_case(args):
    """One named form of the path on one workload, a few times -- the command the ncu captures under profiles/ use
    (`--config 6` = the 28x28 all-member workload whose bitmaps do not fit in L2).  Prints one JSON line."""
    import torch
    import paper_2606_07019_b200 as pk
    pk.use_torch(0)
    p = workload_big() if args.config == 6 else workload(args.config, 0)
    topo = pk.Topology(p.n_npus, p.links)
    prob = pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)
    prob.upload()
    out = {"case": args.case, "config": config_dict(p, args.config)}
    if args.case in ("sweep_tma", "sweep_lsu"):
        ms, nbytes, tot = prob.candidate_sweep(0, 0, pk.PCCL_FLAG_LSU_SWEEP if args.case == "sweep_lsu" else 0, iters=max(1, args.steps))
        out.update({"kernel_ms": ms, "algorithmic_bytes_per_launch": nbytes, "gbs": nbytes / (ms * 1e-3) / 1e9, "candidates": int(tot.sum())})
    else:
        flags = pk.PCCL_FLAG_KEEP_ON_DEVICE | pk.PCCL_FLAG_TIME_LOOP
        for name in (CASES[args.case].split("|") if CASES[args.case] else []):
            flags |= getattr(pk, "PCCL_FLAG_" + name)
        for _ in range(max(1, args.steps)):
            s = prob.synthesize(0, flags)
            st = s.stats
            out.update({"loop_kernel_ms": st["loop_ms"], "setup_ms": st["setup_ms"], "emit_ms": st["emit_ms"], "transfers": s.size,
                        "events": st["events"], "schedule_time_ps": s.time_ps, "requested_bytes": st["bytes_requested"]})
            s.close()
    torch.cuda.synchronize()
    print(json.dumps(out), flush=True)
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
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5, 6])
    ap.add_argument("--case", default=None, choices=sorted(CASES), help="run one named form of the path (for ncu captures)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--fig12", action="store_true", help="chunks-per-NPU sweep shaped like the paper's Fig. 12")
    args = ap.parse_args()
    if args.fig12:
        return run_fig12(args)
    if args.case:
        return run_case(args)
    if args.config == 6:
        raise SystemExit("--config 6 (the larger-than-L2 workload) is for --case runs only")
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
