"""Parity of the CUDA path (through the C-ABI of include/pccl.h) against the CPU oracle.

Bar: everything on this path is integer work, so every comparison is
bit-exact -- identical records (chunk, src, dst, link, t_start_ps, t_end_ps) in identical
canonical order, identical schedule time, identical event count.  On top of parity the
independent checker (oracle/checker.py) validates the CUDA schedule against what the paper
fixes (link exclusivity, causality, postconditions, relay-only non-members).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
import workloads as wl  # noqa: E402
from oracle import checker  # noqa: E402


@pytest.fixture(scope="module")
def pk():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_07019_b200 as pk
    pk.use_torch(0)
    return pk


def gpu_run(pk, p, flags=0):
    return pk.synthesize(*p.args()) if flags == 0 else _problem_run(pk, p, flags)


def _problem_run(pk, p, flags):
    topo = pk.Topology(p.n_npus, p.links)
    prob = pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)
    return prob.synthesize(p.seed, flags)


def assert_same(p, s, o):
    tr = s.transfers
    assert s.size == len(o.transfers), f"{p.name}: {s.size} transfers vs oracle {len(o.transfers)}"
    assert s.time_ps == o.time_ps, f"{p.name}: T {s.time_ps} vs oracle {o.time_ps}"
    for f in ("t_start_ps", "link", "chunk", "src", "dst", "t_end_ps"):
        if not np.array_equal(tr[f], o.transfers[f]):
            i = int(np.nonzero(tr[f] != o.transfers[f])[0][0])
            raise AssertionError(f"{p.name}: field {f} differs first at record {i}: "
                                 f"cuda {tr[i]} vs oracle {o.transfers[i]}")
    st = s.stats
    assert st["events"] == o.events
    assert st["wants_total"] == o.wants_total
    assert st["mode"] == o.mode
    assert st["time_phase1_ps"] == o.time_phase1_ps


# ------------------------------------------------------------------------------ single rows
def test_a6_philox_device_matches_known_answers_and_oracle(pk, golden_dir):
    import os
    rows = []
    with open(os.path.join(golden_dir, "philox_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            rows.append([int(x, 16) for x in line.split()])
    for v in rows:   # the published vectors, evaluated on the GPU
        out = pk.device_philox([v[0:4]], v[4:6])
        assert [int(x) for x in out[0]] == v[6:10]
    rng = np.random.default_rng(7)
    ctr = rng.integers(0, 2 ** 32, size=(1000, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=2, dtype=np.uint64).astype(np.uint32)
    out = pk.device_philox(ctr, key)
    for i in range(0, 1000, 37):
        assert tuple(int(x) for x in out[i]) == oracle.philox4x32_10(ctr[i], key)


def test_a0_link_costs(pk):
    rng = np.random.default_rng(3)
    links = np.zeros(500, dtype=wl.LINK_DT)
    links["src"] = rng.integers(0, 40, 500)
    links["dst"] = (links["src"] + 1 + rng.integers(0, 39, 500)) % 40
    links["alpha_ps"] = rng.integers(0, 10 ** 6, 500)
    links["bytes_per_ps"] = rng.integers(1, 1000, 500)
    topo = pk.Topology(40, links)
    for cb in (1, 63, 64, 1 << 20, (1 << 20) + 1, 10 ** 12 + 7):
        got = topo.link_costs(cb)
        want = [oracle.link_cost(int(l["alpha_ps"]), int(l["bytes_per_ps"]), cb) for l in links]
        assert got.tolist() == want


@pytest.mark.parametrize("maker", [wl.config1, wl.config2, wl.config3, wl.config5_small])
def test_a1_distances(pk, maker):
    p = maker(0)
    topo = pk.Topology(p.n_npus, p.links)
    tl = p.links.copy()
    tl["src"], tl["dst"] = p.links["dst"], p.links["src"]
    for s in (0, 1, p.n_npus // 2, p.n_npus - 1):
        assert np.array_equal(topo.distances(p.chunk_bytes, s), oracle.distances(p.n_npus, p.links, p.chunk_bytes, s))
        assert np.array_equal(topo.distances(p.chunk_bytes, s, transposed=True),
                              oracle.distances(p.n_npus, tl, p.chunk_bytes, s))


def test_a1_distances_unreachable_is_inf(pk):
    links = np.array([(0, 1, 5, 1), (1, 2, 5, 1)], dtype=wl.LINK_DT)   # 3 unreachable, 0 not reachable from 2
    topo = pk.Topology(4, links)
    d = topo.distances(10, 0)
    assert d.tolist() == [0, 15, 30, 2 ** 64 - 1]
    assert np.array_equal(d, oracle.distances(4, links, 10, 0))


def _copy_conditions(p):
    """COPY-mode problem -> (cond_src, dest_off, dests) for oracle.wants."""
    C = p.n_chunks
    src = np.zeros(C, dtype=np.uint32)
    src[p.pre["chunk"]] = p.pre["npu"]
    order = np.lexsort((p.post["npu"], p.post["chunk"]))
    pc, pn = p.post["chunk"][order], p.post["npu"][order]
    keep = pn != src[pc]
    pc, pn = pc[keep], pn[keep]
    off = np.zeros(C + 1, dtype=np.uint64)
    np.add.at(off, pc.astype(np.int64) + 1, 1)
    return src, np.cumsum(off).astype(np.uint64), pn.astype(np.uint32)


@pytest.mark.parametrize("maker", [wl.config1, wl.config4_small, wl.config5_small, wl.two_groups_mesh3x3])
@pytest.mark.parametrize("seed", [0, 3])
def test_a2_wants_bitmap(pk, maker, seed):
    p = maker(seed)
    src, off, dests = _copy_conditions(p)
    want = oracle.wants(p.n_npus, p.links, p.n_chunks, src, off, dests, p.chunk_bytes, seed)
    topo = pk.Topology(p.n_npus, p.links)
    prob = pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)
    got = prob.wants(0, seed)
    assert len(got) == len(want)
    assert np.array_equal(got["npu"], want["npu"]) and np.array_equal(got["chunk"], want["chunk"])


@pytest.mark.parametrize("maker", [wl.config1, wl.config4_small, wl.config5_small, wl.two_groups_mesh3x3,
                                   lambda s: wl.ring_all_gather(8, True, s, chunks_per_npu=1040, chunk_bytes=4096),
                                   lambda s: wl.full_mesh_problem(40, "allgather", seed=s)],
                         ids=lambda m: getattr(m, "__name__", "case"))
def test_a5_candidate_sweep(pk, maker):
    """Row a5 alone: |have[src_l] & wants[dst_l]| of every link at t = 0 from the streaming sweep kernel (rows staged by
    bulk asynchronous copies, and the per-lane-load form) against the oracle's wants relation intersected with the
    initial holdings -- rows of 1, 2, 130 and 4088 words, 39 in-links per destination (five sweeps of 8)."""
    p = maker(2)
    src, off, dests = _copy_conditions(p)
    want = oracle.wants(p.n_npus, p.links, p.n_chunks, src, off, dests, p.chunk_bytes, p.seed)
    wanted = set(zip(want["npu"].tolist(), want["chunk"].tolist()))
    by_src = {}
    for c, s_ in enumerate(src.tolist()):
        by_src.setdefault(s_, []).append(c)
    expect = np.array([sum((int(l["dst"]), c) in wanted for c in by_src.get(int(l["src"]), [])) for l in p.links], dtype=np.uint32)
    topo = pk.Topology(p.n_npus, p.links)
    prob = pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)
    for fl in (0, pk.PCCL_FLAG_LSU_SWEEP):
        ms, nbytes, tot = prob.candidate_sweep(0, p.seed, fl, iters=2)
        assert np.array_equal(tot, expect), fl
        assert ms > 0 and nbytes >= (len(p.links) + 1) * 128


# ------------------------------------------------------------------------------ whole path
SMALL = [wl.config1, wl.config2, wl.config3, wl.config4_small, wl.config5_small, wl.two_groups_mesh3x3]


@pytest.mark.parametrize("maker", SMALL, ids=lambda m: m.__name__)
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_schedule_bit_exact_small_configs(pk, maker, seed):
    p = maker(seed)
    o = oracle.synthesize(*p.args())
    s = gpu_run(pk, p)
    assert_same(p, s, o)
    checker.check_schedule(p, s.transfers)


@pytest.mark.parametrize("maker", [wl.config1, wl.config3, wl.config4_small], ids=lambda m: m.__name__)
def test_idle_skip_does_not_change_the_schedule(pk, maker):
    p = maker(1)
    o = oracle.synthesize(*p.args())
    a = gpu_run(pk, p, pk.PCCL_FLAG_NO_IDLE_SKIP)
    b = gpu_run(pk, p, pk.PCCL_FLAG_KEEP_ON_DEVICE | pk.PCCL_FLAG_TIME_LOOP)
    assert_same(p, a, o)
    assert_same(p, b, o)
    assert a.stats["rows_scanned"] >= b.stats["rows_scanned"]


@pytest.mark.parametrize("n,bidir", [(2, False), (5, False), (8, True), (9, True)])
def test_ring_all_gather_closed_form(pk, n, bidir, golden_dir):
    p = wl.ring_all_gather(n, bidir, seed=1)
    s = gpu_run(pk, p)
    w = 520_972   # tests/golden/closed_forms.txt
    steps = (n - 1) if not bidir else -(-(n - 1) // 2)
    assert s.time_ps == steps * w
    assert s.size == n * (n - 1)
    assert_same(p, s, oracle.synthesize(*p.args()))


def test_many_chunks_per_link_and_ragged_rows(pk):
    """rows of 1, 2 and 130 words (ragged tail inside a 64-word segment and across segments),
    several chunks per NPU so in-links of one destination overlap (the serial re-pick path)."""
    for cpn, n in ((1, 6), (20, 7), (1040, 8)):
        p = wl.ring_all_gather(n, True, seed=5, chunks_per_npu=cpn, chunk_bytes=4096)
        o = oracle.synthesize(*p.args())
        s = gpu_run(pk, p)
        assert_same(p, s, o)


def test_high_indegree_destination(pk):
    """a full mesh of 40 nodes: 39 in-links per destination -> several sweeps of 8 in-links and
    two 32-link windows are not needed, but 5 sweeps are; all-gather makes them overlap."""
    p = wl.full_mesh_problem(40, "allgather", seed=2)
    assert_same(p, gpu_run(pk, p), oracle.synthesize(*p.args()))
    p = wl.full_mesh_problem(40, "alltoall", seed=2)
    assert_same(p, gpu_run(pk, p), oracle.synthesize(*p.args()))


def test_star_switch_with_70_inlinks(pk):
    """one switch node with 70 in-links (three 32-link windows), all-to-all among the leaves."""
    n = 70
    links = [(i, n, 1000, 7) for i in range(n)] + [(n, i, 1000, 7) for i in range(n)]
    links = np.array(links, dtype=wl.LINK_DT)
    members = np.arange(n, dtype=np.uint32)
    nc, pre, post = wl.all_to_all(members)
    p = wl.Problem("star70_alltoall", n + 1, links, members, nc, pre, post, 1000, 11)
    o = oracle.synthesize(*p.args())
    s = gpu_run(pk, p)
    assert_same(p, s, o)
    checker.check_schedule(p, s.transfers)


def test_concurrent_calls_from_two_threads(pk):
    """include/pccl.h: calls on distinct handles may come from different threads (the device entry points
    serialise themselves).  Two threads synthesize different problems back to back; every result must be the
    oracle's."""
    import threading
    probs = [wl.config4_small(0), wl.config2(1), wl.config5_small(2), wl.config3(0)]
    expect = [oracle.synthesize(*p.args()) for p in probs]
    errors = []

    def work(order):
        try:
            for _ in range(3):
                for i in order:
                    assert_same(probs[i], gpu_run(pk, probs[i]), expect[i])
        except BaseException as e:   # noqa: BLE001 - reported by the main thread
            errors.append(e)

    threads = [threading.Thread(target=work, args=(o,)) for o in ([0, 1, 2, 3], [3, 2, 1, 0])]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors[0]


def test_empty_and_trivial(pk):
    links = wl.ring_links(4, True)
    members = np.arange(4, dtype=np.uint32)
    # no chunks at all
    p = wl.Problem("nochunks", 4, links, members, 0, np.zeros(0, wl.PAIR_DT), np.zeros(0, wl.PAIR_DT), 64, 0)
    s = gpu_run(pk, p)
    assert s.size == 0 and s.time_ps == 0 and len(s.transfers) == 0
    # post == pre: nothing to move
    pre = np.array([(0, 0), (1, 1)], dtype=wl.PAIR_DT)
    p = wl.Problem("noop", 4, links, members, 2, pre, pre.copy(), 64, 0)
    o = oracle.synthesize(*p.args())
    s = gpu_run(pk, p)
    assert s.size == 0 == len(o.transfers) and s.time_ps == 0
    # no links, nothing to move
    p = wl.Problem("nolinks", 2, np.zeros(0, wl.LINK_DT), members[:2], 1, pre[:1], pre[:1].copy(), 64, 0)
    assert gpu_run(pk, p).size == 0


def test_error_codes(pk):
    links = np.array([(0, 1, 5, 1)], dtype=wl.LINK_DT)   # 1 cannot reach 0
    members = np.array([0, 1], dtype=np.uint32)
    pre = np.array([(1, 0)], dtype=wl.PAIR_DT)
    post = np.array([(0, 0)], dtype=wl.PAIR_DT)
    with pytest.raises(pk.PcclError) as e:
        pk.synthesize(2, links, members, 1, pre, post, 64, 0)
    assert e.value.code == pk.PCCL_ERR_UNREACHABLE
    with pytest.raises(oracle.OracleError) as eo:
        oracle.synthesize(2, links, members, 1, pre, post, 64, 0)
    assert eo.value.code == oracle.ERR_UNREACHABLE


@pytest.mark.slow
def test_config4_full_size_bit_exact(pk):
    """BASELINE.json configs[3] at full size (the bench workload): 512 NPUs, 261,632 chunks."""
    p = wl.config4(0)
    o = oracle.synthesize(*p.args())
    s = gpu_run(pk, p)
    assert s.size == 1_572_864 == o.wants_total     # sum of hop distances, closed form
    assert_same(p, s, o)
    checker.check_structure(p, s.transfers)
    assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_BARRIER_LOOP), o)


@pytest.mark.parametrize("maker", [wl.config1, wl.config2, wl.config3, wl.config4_small, wl.config5_small,
                                   wl.two_groups_mesh3x3], ids=lambda m: m.__name__)
def test_three_ways_to_the_candidate_counts_agree(pk, maker):
    """kept-current counts (default), per-event recount through the sector work list (RESCAN) and the
    plain dense row sweep (DENSE_SWEEP) must give the same schedule."""
    p = maker(2)
    o = oracle.synthesize(*p.args())
    k = gpu_run(pk, p, pk.PCCL_FLAG_KEEP_ON_DEVICE)
    r = gpu_run(pk, p, pk.PCCL_FLAG_RESCAN)
    d = gpu_run(pk, p, pk.PCCL_FLAG_DENSE_SWEEP)
    for s in (k, r, d):
        assert_same(p, s, o)
    assert d.stats["bytes_requested"] >= r.stats["bytes_requested"]


def test_rescan_modes_on_high_indegree_and_ragged_rows(pk):
    for flags in (pk.PCCL_FLAG_RESCAN, pk.PCCL_FLAG_DENSE_SWEEP):
        p = wl.full_mesh_problem(40, "allgather", seed=2)
        assert_same(p, gpu_run(pk, p, flags), oracle.synthesize(*p.args()))
        p = wl.ring_all_gather(8, True, seed=5, chunks_per_npu=1040, chunk_bytes=4096)
        assert_same(p, gpu_run(pk, p, flags), oracle.synthesize(*p.args()))


@pytest.mark.slow
def test_config5_full_size_bit_exact(pk):
    """BASELINE.json configs[4] at full size: 32x32 torus, 512-member group, Zipf All-to-Allv
    (483,889 chunks, 7.76 M transfers).  The oracle needs a few minutes on one core."""
    p = wl.config5(0)
    s = gpu_run(pk, p, pk.PCCL_FLAG_KEEP_ON_DEVICE)
    assert s.size == 7_761_800
    r = gpu_run(pk, p, pk.PCCL_FLAG_KEEP_ON_DEVICE | pk.PCCL_FLAG_RESCAN)
    b = gpu_run(pk, p, pk.PCCL_FLAG_KEEP_ON_DEVICE | pk.PCCL_FLAG_BARRIER_LOOP)
    o = oracle.synthesize(*p.args())
    assert_same(p, s, o)
    assert_same(p, r, o)
    assert_same(p, b, o)
    checker.check_structure(p, s.transfers)


# ------------------------------------------------------------------------------ dynamic relay rule (NEXT-1)
@pytest.mark.parametrize("maker", SMALL, ids=lambda m: m.__name__)
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_dynamic_relay_bit_exact_small_configs(pk, maker, seed):
    p = maker(seed)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_DYNAMIC)
    s = gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY)
    assert_same(p, s, o)
    checker.check_schedule(p, s.transfers)


def test_dynamic_relay_rings_mesh_star_and_ragged_rows(pk):
    cases = [wl.ring_all_gather(5, False, 1), wl.ring_all_gather(9, True, 2),
             wl.ring_all_gather(8, True, 5, chunks_per_npu=1040, chunk_bytes=4096),
             wl.full_mesh_problem(40, "allgather", seed=2), wl.full_mesh_problem(12, "alltoall", seed=4),
             wl.path_point_to_point(6, 0)]
    n = 70
    links = np.array([(i, n, 1000, 7) for i in range(n)] + [(n, i, 1000, 7) for i in range(n)], dtype=wl.LINK_DT)
    members = np.arange(n, dtype=np.uint32)
    nc, pre, post = wl.all_to_all(members)
    cases.append(wl.Problem("star70_alltoall", n + 1, links, members, nc, pre, post, 1000, 11))
    for p in cases:
        o = oracle.synthesize(*p.args(), relay=oracle.RELAY_DYNAMIC)
        assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY), o)


@pytest.mark.parametrize("maker", [wl.config2, wl.config3, wl.config4_small, wl.config5_small], ids=lambda m: m.__name__)
def test_dynamic_relay_three_counting_modes(pk, maker):
    p = maker(1)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_DYNAMIC)
    for fl in (0, pk.PCCL_FLAG_KEPT_COUNTS, pk.PCCL_FLAG_RESCAN, pk.PCCL_FLAG_DENSE_SWEEP):
        assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY | fl), o)


def test_dynamic_relay_holder_rows_overflow(pk):
    """The holder row of a chunk has 31 slots: past that a claim falls back to the scan over all
    nodes.  A 40-node path (one chunk, 39 arrivals: the switch happens mid-run, with stale bits around), rings with
    32 dests and 32+ arrivals per chunk, a mesh where every chunk has more than 32 dests."""
    mesh = wl.grid_links((7, 6), wrap=False)
    m42 = np.arange(42, dtype=np.uint32)
    nc, pre, post = wl.all_gather(m42, 2)
    cases = [wl.path_point_to_point(40, 0), wl.ring_all_gather(33, False, 3), wl.ring_all_gather(36, True, 1),
             wl.ring_all_gather(33, True, 2, chunks_per_npu=3, chunk_bytes=4096),
             wl.Problem("mesh7x6_allgather2", 42, mesh, m42, nc, pre, post, 1 << 16, 5)]
    for p in cases:
        o = oracle.synthesize(*p.args(), relay=oracle.RELAY_DYNAMIC)
        for fl in (0, pk.PCCL_FLAG_DENSE_SWEEP):
            assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY | fl), o)


def _golden(case):
    """line of tests/golden/oracle_schedules.txt (written by tests/golden/make_golden.py from oracle/ only)"""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_schedules.txt")
    for ln in open(path):
        f = ln.split()
        if f and f[0] == case:
            return {"seed": int(f[1]), "transfers": int(f[2]), "time_ps": int(f[3]), "events": int(f[4]),
                    "wants_total": int(f[5]), "sha256": f[6]}
    return None


def _assert_digest(s, g, name):
    import hashlib
    assert s.size == g["transfers"], f"{name}: {s.size} transfers vs oracle {g['transfers']}"
    assert s.time_ps == g["time_ps"], f"{name}: T {s.time_ps} vs oracle {g['time_ps']}"
    st = s.stats
    assert st["events"] == g["events"] and st["wants_total"] == g["wants_total"], name
    assert hashlib.sha256(s.transfers.tobytes()).hexdigest() == g["sha256"], f"{name}: records differ from the oracle's"


FULL_SIZE = [("cfg4:thin", 0), ("cfg4:thin", "BARRIER_LOOP"), ("cfg4:dynamic", "DYNAMIC_RELAY"),
             ("cfg4:dynamic", "DYNAMIC_RELAY|DENSE_SWEEP"), ("cfg4:bfs", "BFS"), ("cfg5:thin", 0),
             ("cfg5:thin", "DENSE_SWEEP"), ("cfg5:dynamic", "DYNAMIC_RELAY"), ("cfg5:bfs", "BFS")]


@pytest.mark.slow
@pytest.mark.parametrize("case,mode", FULL_SIZE, ids=lambda x: str(x))
def test_full_size_schedule_equals_the_oracles_digest(pk, case, mode):
    """BASELINE.json configs 4 and 5 at full size under every relay mode: the CUDA schedule's records, T, event count and
    initial wants against the digest of the ORACLE's run (the oracle needs 15 minutes for cfg4:dynamic, hours for
    cfg5:dynamic, so its results are stored: tests/golden/oracle_schedules.txt, written by make_golden.py from oracle/
    only).  The dynamic rule is checked in both of its forms (holder lists / all-nodes scan)."""
    g = _golden(case)
    if g is None:
        pytest.skip(f"no oracle digest for {case} in tests/golden/oracle_schedules.txt (run tests/golden/make_golden.py {case})")
    flags = pk.PCCL_FLAG_KEEP_ON_DEVICE
    for name in (mode.split("|") if mode else []):
        flags |= getattr(pk, "PCCL_FLAG_" + name)
    p = {"cfg4": wl.config4, "cfg5": wl.config5}[case.split(":")[0]](g["seed"])
    s = gpu_run(pk, p, flags)
    _assert_digest(s, g, f"{case} {mode}")
    checker.check_structure(p, s.transfers)


@pytest.mark.slow
@pytest.mark.parametrize("case,runs", [("cfg4:thin", 6), ("cfg5:thin", 3)], ids=lambda x: str(x))
def test_full_size_streamed_schedule_equals_the_oracles_digest(pk, case, runs):
    """The e2e path (pccl_synthesize, host buffers): the emitter ranks the claims in windows behind the global virtual
    time on a second stream WHILE the barrier-free loop runs, and the host copies the finished prefix out meanwhile.
    Where the windows fall depends on timing, the records must not: several runs, each against the oracle's digest."""
    g = _golden(case)
    if g is None:
        pytest.skip(f"no oracle digest for {case}")
    p = {"cfg4": wl.config4, "cfg5": wl.config5}[case.split(":")[0]](g["seed"])
    for i in range(runs):
        s = pk.synthesize(*p.args())
        _assert_digest(s, g, f"{case} streamed, run {i}")
        s.close()


def test_dynamic_relay_record_buffer_rerun(pk):
    """The dynamic rule's record buffer is sized from the static relay tree's transfer count; when it is short the run
    still finishes (records past the end are dropped, the count goes on) and the phase is rerun with the exact count.
    Forced here with a 100-record buffer on copy, reduce and all-reduce problems."""
    cases = [wl.config4_small(1), wl.config3(0), wl.config2(2)]
    pk.set_option(pk.PCCL_OPT_DYNAMIC_RECORDS, 100)
    try:
        for p in cases:
            o = oracle.synthesize(*p.args(), relay=oracle.RELAY_DYNAMIC)
            assert len(o.transfers) > 100
            assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY), o)
    finally:
        pk.set_option(pk.PCCL_OPT_DYNAMIC_RECORDS, 0)


def test_dynamic_relay_unreachable(pk):
    links = np.array([(0, 1, 5, 1)], dtype=wl.LINK_DT)
    members = np.array([0, 1], dtype=np.uint32)
    pre = np.array([(1, 0)], dtype=wl.PAIR_DT)
    post = np.array([(0, 0)], dtype=wl.PAIR_DT)
    topo = pk.Topology(2, links)
    prob = pk.Problem(topo, members, 1, pre, post, 64)
    with pytest.raises(pk.PcclError) as e:
        prob.synthesize(0, pk.PCCL_FLAG_DYNAMIC_RELAY)
    assert e.value.code == pk.PCCL_ERR_UNREACHABLE


@pytest.mark.slow
def test_dynamic_relay_6x6x6_torus_all_to_all(pk):
    """216 NPUs, 46,440 chunks (rows of 726 words: 12 segments with a ragged tail), 212 k transfers."""
    p = wl.config4(0, dims=(6, 6, 6))
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_DYNAMIC)
    s = gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY)
    assert_same(p, s, o)
    checker.check_structure(p, s.transfers)


# ------------------------------------------------------------------------------ scale / shape stress
def _torus_all_gather(dims, cpn, seed):
    n = int(np.prod(dims))
    m = np.arange(n, dtype=np.uint32)
    nc, pre, post = wl.all_gather(m, cpn)
    return wl.Problem(f"torus{'x'.join(map(str, dims))}_allgather{cpn}", n, wl.grid_links(dims, wrap=True), m, nc,
                      pre, post, 1 << 16, seed)


def _ring3000_a2a(seed):
    n = 3000
    mem = np.array([0, 400, 777, 1200, 1500, 2100, 2500, 2999], dtype=np.uint32)
    nc, pre, post = wl.all_to_all(mem, np.full((8, 8), 3))
    return wl.Problem("ring3000_a2a8", n, wl.ring_links(n, True), mem, nc, pre, post, 1 << 12, seed)


@pytest.mark.parametrize("relay", [0, 1])
def test_multi_dest_trees_at_scale(pk, relay):
    """144-NPU torus All-Gather, 288 chunks with 143 dests each: every sweep has overlapping in-links (the
    serial re-pick path), multi-dest relay trees, 41 k transfers."""
    p = _torus_all_gather((12, 12), 2, 7)
    o = oracle.synthesize(*p.args(), relay=relay)
    s = gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY if relay else 0)
    assert_same(p, s, o)
    checker.check_structure(p, s.transfers)


@pytest.mark.parametrize("relay", [0, 1])
def test_more_nodes_than_resident_ctas(pk, relay):
    """3000-node ring, 8 members: every CTA serves several destinations (the third and later from the
    uncached tables), 1,500 events, almost all nodes only relay."""
    p = _ring3000_a2a(3)
    o = oracle.synthesize(*p.args(), relay=relay)
    s = gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY if relay else 0)
    assert_same(p, s, o)
    checker.check_structure(p, s.transfers)


@pytest.mark.parametrize("relay", [0, 1])
def test_ten_thousand_nodes(pk, relay):
    """10,000-node ring, 4 members: the distance kernel's per-source table is 80 KB of shared memory (the
    opt-in size), there are more destinations than the one-barrier loop caches (it falls back to the
    two-barrier loop), 5,000 events."""
    n = 10000
    mem = np.array([0, 2500, 5000, 7500], dtype=np.uint32)
    nc, pre, post = wl.all_to_all(mem, np.full((4, 4), 2))
    p = wl.Problem("ring10000_a2a4", n, wl.ring_links(n, True), mem, nc, pre, post, 1 << 12, 5)
    o = oracle.synthesize(*p.args(), relay=relay)
    s = gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY if relay else 0)
    assert_same(p, s, o)
    checker.check_structure(p, s.transfers)


# ------------------------------------------------------------------------------ the two event loops
@pytest.mark.parametrize("maker", SMALL + [lambda s: wl.ring_all_gather(8, True, s, chunks_per_npu=1040, chunk_bytes=4096),
                                           lambda s: _torus_all_gather((12, 12), 2, s)],
                         ids=lambda m: getattr(m, "__name__", "case"))
def test_the_three_event_loops_agree(pk, maker):
    """the default is the barrier-free loop where it applies (<= 8 in-links per node, link costs within 16x; ASYNC
    forces it for any link costs); BARRIER_LOOP selects the one-barrier loop (or the two-barrier one where that
    does not apply), TWO_BARRIERS the two-barrier loop.  All must equal the oracle."""
    p = maker(3)
    o = oracle.synthesize(*p.args())
    assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_KEEP_ON_DEVICE), o)
    assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_ASYNC), o)
    assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_BARRIER_LOOP), o)
    assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_TWO_BARRIERS), o)


# ------------------------------------------------------------------------------ the paper's own synthesizer (BFS)
BFS_CASES = [wl.config1, wl.config2, wl.config3, wl.config4_small, wl.config5_small, wl.two_groups_mesh3x3,
             lambda s: wl.ring_all_gather(8, False, s), lambda s: wl.ring_all_gather(9, True, s, chunks_per_npu=3),
             lambda s: wl.path_point_to_point(6, s), lambda s: _torus_all_gather((12, 12), 2, s)]


@pytest.mark.parametrize("maker", BFS_CASES, ids=lambda m: getattr(m, "__name__", "case"))
@pytest.mark.parametrize("seed", [0, 1])
def test_bfs_mode_equals_oracle(pk, maker, seed):
    """PCCL_FLAG_BFS (Alg. 1-3 + section 4.6, windowed optimistic search) against the strictly sequential oracle:
    identical records, T, condition count, transfer count."""
    p = maker(seed)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS)
    s = gpu_run(pk, p, pk.PCCL_FLAG_BFS)
    assert_same(p, s, o)
    checker.check_structure(p, s.transfers)
    st = s.stats
    assert st["rows_scanned"] >= st["events"] and st["slow_picks"] >= 1


def test_bfs_mode_many_conditions_per_link(pk):
    """8-node ring, 1040 chunks per node: 8,320 conditions over 16 links -- long busy-run rows, most windows
    conflict at once (almost every round commits few conditions)"""
    p = wl.ring_all_gather(8, True, 2, chunks_per_npu=130, chunk_bytes=4096)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS)
    s = gpu_run(pk, p, pk.PCCL_FLAG_BFS)
    assert_same(p, s, o)


def test_bfs_mode_reruns_when_a_busy_run_row_fills(pk):
    """rows of 8 entries overflow at once on the 8-node ring with 130 chunks per node (gaps open and close on
    every link): the kernel stops at the next round, the phase is rerun with longer rows, same schedule"""
    p = wl.config5_small(1)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS)
    pk.set_option(pk.PCCL_OPT_BFS_ROWS, 8)
    try:
        s = gpu_run(pk, p, pk.PCCL_FLAG_BFS)
    finally:
        pk.set_option(pk.PCCL_OPT_BFS_ROWS, 0)
    assert_same(p, s, o)
    pk.set_option(pk.PCCL_OPT_BFS_WINDOW, 3)      # a 3-wide window: more rounds, same schedule
    try:
        s = gpu_run(pk, p, pk.PCCL_FLAG_BFS)
    finally:
        pk.set_option(pk.PCCL_OPT_BFS_WINDOW, 0)
    assert_same(p, s, o)
    assert s.stats["grid_blocks"] == 3


def test_bfs_mode_ring3000(pk):
    p = _ring3000_a2a(3)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS)
    s = gpu_run(pk, p, pk.PCCL_FLAG_BFS)
    assert_same(p, s, o)
    checker.check_structure(p, s.transfers)


@pytest.mark.slow
def test_bfs_mode_config4_full_size(pk):
    """BASELINE.json configs[3] at full size through the paper's synthesizer: 261,632 conditions, 1.66 M
    transfers (more than the 1,572,864 of minimal routing: detours through idle links)."""
    p = wl.config4(0)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS)
    s = gpu_run(pk, p, pk.PCCL_FLAG_BFS)
    assert_same(p, s, o)
    assert s.size >= 1_572_864
    checker.check_structure(p, s.transfers)


# ------------------------------------------------------------------------------ randomized problems
def _random_problem(i):
    """seeded random directed multigraph with heterogeneous links, a random process group and a random
    collective (copy with multi-dest chunks, reduce, or all-reduce); may be unreachable on purpose"""
    rng = np.random.default_rng(1000 + i)
    n = int(rng.integers(3, 40))
    base = [(a, (a + 1) % n) for a in range(n)] if rng.random() < 0.8 else []          # a ring keeps most cases connected
    extra = int(rng.integers(n, 6 * n))
    src = rng.integers(0, n, extra)
    dst = (src + 1 + rng.integers(0, n - 1, extra)) % n
    pairs = base + list(zip(src.tolist(), dst.tolist()))
    if rng.random() < 0.5:
        pairs += [(b, a) for a, b in pairs]                                            # symmetric half of the time
    links = np.zeros(len(pairs), dtype=wl.LINK_DT)
    links["src"], links["dst"] = zip(*pairs)
    if rng.random() < 0.5:
        links["alpha_ps"], links["bytes_per_ps"] = 500, 10
    else:
        links["alpha_ps"] = rng.integers(0, 2000, len(pairs))
        links["bytes_per_ps"] = rng.integers(1, 50, len(pairs))
    g = int(rng.integers(2, n + 1))
    members = np.sort(rng.choice(n, size=g, replace=False)).astype(np.uint32)
    kind = int(rng.integers(0, 3))
    nc = int(rng.integers(1, 200))
    pre, post = [], []
    for c in range(nc):
        if kind == 0:      # copy: one holder, 1..g dests
            s = int(rng.choice(members))
            pre.append((s, c))
            for d in rng.choice(members, size=int(rng.integers(1, g + 1)), replace=False):
                post.append((int(d), c))
        elif kind == 1:    # reduce: several holders, one root
            hs = rng.choice(members, size=int(rng.integers(2, g + 1)), replace=False) if g >= 2 else members
            pre += [(int(h), c) for h in hs]
            post.append((int(rng.choice(members)), c))
        else:              # all-reduce
            hs = rng.choice(members, size=int(rng.integers(2, g + 1)), replace=False)
            ds = rng.choice(members, size=int(rng.integers(2, g + 1)), replace=False)
            pre += [(int(h), c) for h in hs]
            post += [(int(d), c) for d in ds]
    pre = np.array(pre, dtype=wl.PAIR_DT)
    post = np.array(post, dtype=wl.PAIR_DT)
    return wl.Problem(f"random{i}", n, links, members, nc, pre, post, int(rng.integers(1, 5000)), int(rng.integers(0, 2 ** 63)))


def _random_multi_dest_problem(i):
    """40..150 nodes, a ring plus random (often symmetric) extra links, 20..100 chunks with up to |group| dests each:
    chunks with a handful of holders and chunks with more arrivals than a holder row has slots in one problem"""
    rng = np.random.default_rng(50000 + i)
    n = int(rng.integers(40, 150))
    extra = int(rng.integers(n // 2, 3 * n))
    src = rng.integers(0, n, extra)
    dst = (src + 1 + rng.integers(0, n - 1, extra)) % n
    pairs = [(a, (a + 1) % n) for a in range(n)] + list(zip(src.tolist(), dst.tolist()))
    if rng.random() < 0.6:
        pairs += [(b, a) for a, b in pairs]
    links = np.zeros(len(pairs), dtype=wl.LINK_DT)
    links["src"], links["dst"] = zip(*pairs)
    if rng.random() < 0.5:
        links["alpha_ps"], links["bytes_per_ps"] = 500, 10
    else:
        links["alpha_ps"] = rng.integers(0, 2000, len(pairs))
        links["bytes_per_ps"] = rng.integers(1, 50, len(pairs))
    g = int(rng.integers(n // 2, n + 1))
    members = np.sort(rng.choice(n, size=g, replace=False)).astype(np.uint32)
    nc = int(rng.integers(20, 100))
    pre, post = [], []
    for c in range(nc):
        pre.append((int(rng.choice(members)), c))
        k = int(rng.integers(1, g + 1)) if rng.random() < 0.5 else int(rng.integers(1, 34))
        for d in rng.choice(members, size=min(k, g), replace=False):
            post.append((int(d), c))
    return wl.Problem(f"multidest{i}", n, links, members, nc, np.array(pre, dtype=wl.PAIR_DT),
                      np.array(post, dtype=wl.PAIR_DT), int(rng.integers(1, 5000)), int(rng.integers(0, 2 ** 63)))


def test_dynamic_relay_random_multi_dest_problems(pk):
    """The holder-list form of the dynamic rule (lazy wants bits, fall-back to the all-nodes scan per chunk) and the
    all-nodes form against the oracle on 24 medium-sized random problems."""
    for i in range(24):
        p = _random_multi_dest_problem(i)
        try:
            o = oracle.synthesize(*p.args(), relay=oracle.RELAY_DYNAMIC)
        except oracle.OracleError:
            continue
        for fl in (0, pk.PCCL_FLAG_DENSE_SWEEP):
            assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_DYNAMIC_RELAY | fl), o)


@pytest.mark.parametrize("block", range(6))
def test_randomized_problems_all_modes(pk, block):
    """120 random problems: each must give the oracle's schedule (or the oracle's error) under both relay rules
    and under the paper's BFS synthesizer; every sixth also under the recount modes and the two-barrier loop."""
    for i in range(block * 20, block * 20 + 20):
        p = _random_problem(i)
        for relay, rflag in ((0, 0), (1, pk.PCCL_FLAG_DYNAMIC_RELAY), (2, pk.PCCL_FLAG_BFS)):
            try:
                o = oracle.synthesize(*p.args(), relay=relay)
            except oracle.OracleError as e:
                with pytest.raises(pk.PcclError) as g:
                    gpu_run(pk, p, rflag | pk.PCCL_FLAG_KEEP_ON_DEVICE)
                assert g.value.code == {oracle.ERR_UNREACHABLE: pk.PCCL_ERR_UNREACHABLE,
                                        oracle.ERR_UNSUPPORTED: pk.PCCL_ERR_UNSUPPORTED,
                                        oracle.ERR_INVALID: pk.PCCL_ERR_INVALID}[e.code], p.name
                continue
            assert_same(p, gpu_run(pk, p, rflag | pk.PCCL_FLAG_KEEP_ON_DEVICE), o)
            if i % 6 == 0 and relay != 2:
                for fl in (pk.PCCL_FLAG_TWO_BARRIERS, pk.PCCL_FLAG_RESCAN, pk.PCCL_FLAG_DENSE_SWEEP):
                    assert_same(p, gpu_run(pk, p, rflag | fl), o)
            if relay == 0:   # the barrier-free loop with heterogeneous link costs, and the one-barrier loop
                assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_ASYNC), o)
                assert_same(p, gpu_run(pk, p, pk.PCCL_FLAG_BARRIER_LOOP), o)
            if relay == 0:
                checker.check_schedule(p, o.transfers)


# ------------------------------------------------------------------------------ switch model (NEXT-3)
def _bfs_with_switches(pk, p, bl, nm):
    topo = pk.Topology(p.n_npus, p.links)
    topo.set_switch_model(bl, nm)
    prob = pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)
    return prob.synthesize(p.seed, pk.PCCL_FLAG_BFS)


def _random_switch_problem(i):
    """a random heterogeneous multigraph problem (copy / reduce / all-reduce) with buffer limits of 1..3 chunks on a few
    nodes and some nodes without multicast"""
    p = _random_problem(300 + i)
    rng = np.random.default_rng(4200 + i)
    n = p.n_npus
    bl = np.full(n, oracle.NO_LIMIT, dtype=np.uint32)
    nm = np.zeros(n, dtype=np.uint8)
    members = set(int(x) for x in p.group)
    others = [v for v in range(n) if v not in members] or list(range(n))
    for v in rng.choice(others, size=min(len(others), int(rng.integers(1, 5))), replace=False):
        bl[int(v)] = int(rng.integers(1, 4))
    if i % 3:
        for v in rng.choice(n, size=int(rng.integers(1, 4)), replace=False):
            nm[int(v)] = 1
    if i % 5 == 4:
        bl[:] = oracle.NO_LIMIT            # no multicast only
    return p, bl, nm


@pytest.mark.parametrize("block", range(3))
def test_switch_model_random_problems(pk, block):
    """PCCL_FLAG_BFS with per-node buffer limits and no-multicast nodes against the oracle's switch model, 30 problems"""
    for i in range(block * 10, block * 10 + 10):
        p, bl, nm = _random_switch_problem(i)
        try:
            o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS, buffer_limit=bl, no_multicast=nm)
        except oracle.OracleError as e:
            with pytest.raises(pk.PcclError) as g:
                _bfs_with_switches(pk, p, bl, nm)
            assert g.value.code == {oracle.ERR_UNREACHABLE: pk.PCCL_ERR_UNREACHABLE, oracle.ERR_UNSUPPORTED: pk.PCCL_ERR_UNSUPPORTED,
                                    oracle.ERR_INVALID: pk.PCCL_ERR_INVALID}[e.code], p.name
            continue
        assert_same(p, _bfs_with_switches(pk, p, bl, nm), o)


@pytest.mark.parametrize("limit,unicast", [(2, True), (1, False), (oracle.NO_LIMIT, True)])
def test_switch_model_config3(pk, limit, unicast):
    """config 3's eight pod switches with finite buffers and / or without multicast (Reduce-Scatter, both directions of
    the model through the transposed phase)"""
    p = wl.config3(0)
    bl = np.full(p.n_npus, oracle.NO_LIMIT, dtype=np.uint32)
    bl[64:] = limit
    nm = np.zeros(p.n_npus, dtype=np.uint8)
    nm[64:] = 1 if unicast else 0
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS, buffer_limit=bl, no_multicast=nm)
    s = _bfs_with_switches(pk, p, bl, nm)
    assert_same(p, s, o)
    checker.check_schedule(p, s.transfers)


def test_switch_model_hand_examples_and_modes(pk):
    links = np.array([(0, 2, 0, 1), (1, 2, 0, 1), (2, 3, 0, 1), (2, 4, 0, 1)], dtype=wl.LINK_DT)
    pre = np.array([(0, 0), (1, 1)], dtype=wl.PAIR_DT)
    post = np.array([(3, 0), (4, 1)], dtype=wl.PAIR_DT)
    p = wl.Problem("two_through_one_switch", 5, links, np.array([0, 1, 3, 4], dtype=np.uint32), 2, pre, post, 1, 0)
    bl = np.array([oracle.NO_LIMIT] * 5, dtype=np.uint32)
    bl[2] = 1
    s = _bfs_with_switches(pk, p, bl, None)
    assert s.time_ps == 3                                        # tests/test_oracle_bfs.py: test_buffer_limit_hand_example
    assert_same(p, s, oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS, buffer_limit=bl))
    bl[2] = 0
    with pytest.raises(pk.PcclError) as e:
        _bfs_with_switches(pk, p, bl, None)
    assert e.value.code == pk.PCCL_ERR_UNREACHABLE
    # the matching loops do not model switches: refused while a model is set, fine again once it is removed
    topo = pk.Topology(p.n_npus, p.links)
    bl[2] = 1
    topo.set_switch_model(bl, None)
    prob = pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)
    with pytest.raises(pk.PcclError) as e:
        prob.synthesize(0, 0)
    assert e.value.code == pk.PCCL_ERR_UNSUPPORTED
    topo.set_switch_model(None, None)
    assert prob.synthesize(0, 0).time_ps == 2


# ------------------------------------------------------------------------------ pipelined All-Reduce (NEXT-4, Q26)
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_pipelined_allreduce_config2(pk, seed):
    p = wl.config2(seed)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS, pipeline=True)
    s = gpu_run(pk, p, pk.PCCL_FLAG_BFS | pk.PCCL_FLAG_PIPELINE)
    assert_same(p, s, o)
    checker.check_schedule(p, s.transfers)
    seq = gpu_run(pk, p, pk.PCCL_FLAG_BFS)
    assert s.stats["time_phase1_ps"] == seq.stats["time_phase1_ps"] and s.time_ps <= seq.time_ps


def test_pipelined_allreduce_random_problems(pk):
    """every all-reduce among 90 random problems (heterogeneous links, random groups), and the flag's no-effect on the
    copy and reduce problems among them"""
    seen = 0
    for i in range(90):
        p = _random_problem(i)
        try:
            o = oracle.synthesize(*p.args(), relay=oracle.RELAY_BFS, pipeline=True)
        except oracle.OracleError:
            continue
        s = gpu_run(pk, p, pk.PCCL_FLAG_BFS | pk.PCCL_FLAG_PIPELINE | pk.PCCL_FLAG_KEEP_ON_DEVICE)
        assert_same(p, s, o)
        seen += o.mode == 2
    assert seen >= 15


def test_pipeline_flag_needs_the_bfs_mode(pk):
    p = wl.config2(0)
    with pytest.raises(pk.PcclError) as e:
        gpu_run(pk, p, pk.PCCL_FLAG_PIPELINE)
    assert e.value.code == pk.PCCL_ERR_UNSUPPORTED
    q = wl.config1(0)                                  # not an all-reduce: the flag has no effect
    assert_same(q, gpu_run(pk, q, pk.PCCL_FLAG_PIPELINE), oracle.synthesize(*q.args()))


# ------------------------------------------------------------------------------ c.dist-priority pick (NEXT-4, Q27)
@pytest.mark.parametrize("maker", [wl.config1, wl.config2, wl.config4_small, wl.config5_small, wl.two_groups_mesh3x3,
                                   lambda s: wl.ring_all_gather(8, True, s, chunks_per_npu=1040, chunk_bytes=4096),
                                   lambda s: _torus_all_gather((12, 12), 2, s)], ids=lambda m: getattr(m, "__name__", "case"))
@pytest.mark.parametrize("seed", [0, 1])
def test_dist_pick_equals_oracle(pk, maker, seed):
    p = maker(seed)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_THIN_DIST_PICK)
    s = gpu_run(pk, p, pk.PCCL_FLAG_DIST_PICK)
    assert_same(p, s, o)
    checker.check_schedule(p, s.transfers)


def test_dist_pick_random_problems(pk):
    """heterogeneous links give many distinct c.dist values (one class per chunk in the extreme); nodes with more than
    8 in-links are refused"""
    ran = 0
    for i in range(60):
        p = _random_problem(i)
        try:
            o = oracle.synthesize(*p.args(), relay=oracle.RELAY_THIN_DIST_PICK)
        except oracle.OracleError:
            continue
        try:
            s = gpu_run(pk, p, pk.PCCL_FLAG_DIST_PICK | pk.PCCL_FLAG_KEEP_ON_DEVICE)
        except pk.PcclError as e:
            assert e.code == pk.PCCL_ERR_UNSUPPORTED
            indeg = np.bincount(p.links["dst"], minlength=p.n_npus).max()
            outdeg = np.bincount(p.links["src"], minlength=p.n_npus).max()
            assert max(indeg, outdeg) > 8, p.name
            continue
        assert_same(p, s, o)
        ran += 1
    assert ran >= 10


@pytest.mark.slow
def test_dist_pick_config4_full_size(pk):
    p = wl.config4(0)
    o = oracle.synthesize(*p.args(), relay=oracle.RELAY_THIN_DIST_PICK)
    s = gpu_run(pk, p, pk.PCCL_FLAG_DIST_PICK | pk.PCCL_FLAG_KEEP_ON_DEVICE)
    assert_same(p, s, o)
    with pytest.raises(pk.PcclError) as e:
        gpu_run(pk, wl.config3(0), pk.PCCL_FLAG_DIST_PICK)          # 15-in-link switches
    assert e.value.code == pk.PCCL_ERR_UNSUPPORTED
