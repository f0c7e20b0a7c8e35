"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the plausible mistake it would catch.  None of them re-types the oracle's own
formula as the expectation: expectations come from the paper's closed forms (tests/golden),
from a library routine (scipy Dijkstra), from brute force, from an independent numpy Philox
(workloads.philox_first_word) driving a 20-line list model on 2-node multigraphs, or from the
schedule simulator in oracle/checker.py.
"""
import os

import numpy as np
import pytest

import oracle
import workloads as wl
from oracle import brute_force, checker

W1M = 520_972  # tests/golden/closed_forms.txt


def _golden_kv(golden_dir, name):
    out = {}
    with open(os.path.join(golden_dir, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            out[k] = v
    return out


def run(p):
    return oracle.synthesize(*p.args())


# --------------------------------------------------------------------------- Philox / a6
def test_philox_known_answers(golden_dir):
    """catches: wrong multiplier/round count/word order/key schedule."""
    n = 0
    with open(os.path.join(golden_dir, "philox_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(x, 16) for x in line.split()]
            assert oracle.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])
            n += 1
    assert n == 3


def test_harness_philox_matches_known_answers():
    """the workloads' numpy generator (used below as an independent RNG) passes the same KAT."""
    assert int(wl.philox_first_word(0, 0, 0, 0, 0)) == 0x6627E8D5
    assert int(wl.philox_first_word(0xFFFFFFFF, 0xFFFFFFFF, 0xFFFFFFFF, 0xFFFFFFFF, (1 << 64) - 1)) == 0x408F276D
    assert int(wl.philox_first_word(0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344,
                                    0xA4093822 | (0x299F31D0 << 32))) == 0xD16CFE09


# --------------------------------------------------------------------------- cost / a0
def test_link_cost_closed_form(golden_dir):
    """catches: floor instead of ceil, alpha inside the division, beta inverted."""
    g = _golden_kv(golden_dir, "closed_forms.txt")
    assert oracle.link_cost(500_000, 50, 1 << 20) == int(g["w_1MiB_500000ps_50Bps"]) == W1M
    assert oracle.link_cost(0, 64, 128) == 2          # exact division: no +1
    assert oracle.link_cost(0, 64, 129) == 3          # ceiling
    assert oracle.link_cost(7, 1000, 1) == 8          # sub-ps payload still costs 1 ps
    assert oracle.link_cost(200_000, 450, 1 << 20) == 200_000 + 2331  # 1048576/450 = 2330.17


# --------------------------------------------------------------------------- distances / a1
def test_distances_match_scipy_dijkstra():
    """catches: wrong edge direction, wrong metric (hops instead of alpha-beta cost)."""
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import dijkstra
    rng = np.random.default_rng(5)
    n = 12
    src = rng.integers(0, n, 40)
    dst = rng.integers(0, n, 40)
    keep = src != dst
    links = np.zeros(keep.sum(), dtype=wl.LINK_DT)
    links["src"], links["dst"] = src[keep], dst[keep]
    links["alpha_ps"] = rng.integers(1, 1000, keep.sum())
    links["bytes_per_ps"] = rng.integers(1, 9, keep.sum())
    cb = 1000
    w = checker.link_costs(links, cb).astype(np.float64)
    dense = np.full((n, n), np.inf)
    for l in range(len(links)):   # parallel links: keep the cheapest
        dense[links["src"][l], links["dst"][l]] = min(dense[links["src"][l], links["dst"][l]], w[l])
    dense[np.isinf(dense)] = 0
    ref = dijkstra(csr_matrix(dense), directed=True)
    for s in range(n):
        got = oracle.distances(n, links, cb, s).astype(np.float64)
        got[got == float(np.iinfo(np.uint64).max)] = np.inf
        assert np.array_equal(got, ref[s])


def test_distances_torus_closed_form():
    """homogeneous torus: distance = wrapped Manhattan hops * w."""
    links = wl.grid_links((4, 4, 4), wrap=True)
    d = oracle.distances(64, links, 64 << 10, 0)
    w = 500_000 + -(-(64 << 10) // 50)
    for v in range(64):
        x, y, z = v % 4, (v // 4) % 4, v // 16
        hops = sum(min(a, 4 - a) for a in (x, y, z))
        assert d[v] == hops * w


# --------------------------------------------------------------------------- wants / a2
def _conds_single_dest(p):
    src = np.zeros(p.n_chunks, dtype=np.uint32)
    src[p.pre["chunk"]] = p.pre["npu"]
    order = np.argsort(p.post["chunk"], kind="stable")
    dests = p.post["npu"][order]
    off = np.arange(p.n_chunks + 1, dtype=np.uint64)
    return src, off, dests


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_wants_is_one_shortest_path_per_chunk(seed):
    """single-destination chunks on a homogeneous torus: wants marks exactly hops(s,d) nodes,
    all on a shortest s->d path, ending at d.  catches: wrong relay rule, off-by-one at the
    source, non-tight predecessor."""
    p = wl.config4_small(seed)
    src, off, dests = _conds_single_dest(p)
    wp = oracle.wants(p.n_npus, p.links, p.n_chunks, src, off, dests, p.chunk_bytes, seed)
    w = int(checker.link_costs(p.links, p.chunk_bytes)[0])
    D = np.stack([oracle.distances(p.n_npus, p.links, p.chunk_bytes, s) for s in range(p.n_npus)])
    hops = (D // np.uint64(w)).astype(np.int64)
    per_chunk = np.bincount(wp["chunk"], minlength=p.n_chunks)
    assert np.array_equal(per_chunk, hops[src, dests])
    s_, d_ = src[wp["chunk"]], dests[wp["chunk"]]
    v_ = wp["npu"]
    assert (hops[s_, v_] + hops[v_, d_] == hops[s_, d_]).all()      # on a shortest path
    assert (v_ != s_).all()                                         # the source wants nothing
    # distinct distances along a chunk's path: one node per hop count 1..hops
    key = wp["chunk"].astype(np.int64) * 1000 + hops[s_, v_]
    assert len(np.unique(key)) == len(key)
    # schedule length equals popcount(wants) and the closed form sum of hop distances
    s = run(p)
    assert len(s.transfers) == s.wants_total == len(wp) == int(hops[src, dests].sum())


def test_wants_multidest_is_a_tree():
    """All-Gather chunks: the marked nodes of a chunk form a tree rooted at the source that
    contains every destination; here (everyone is a destination) it spans all other nodes."""
    p = wl.config1(0)
    s = run(p)
    assert s.wants_total == 16 * 15 == len(s.transfers)


# --------------------------------------------------------------------------- closed forms
@pytest.mark.parametrize("n", [2, 3, 4, 5, 8])
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_ring_unidirectional_exact_schedule(n, seed):
    """ring All-Gather = N-1 steps, optimal; on a unidirectional ring every
    link has exactly one candidate per step so the whole schedule is fixed for every seed.
    catches: early/late forwarding (arrivals), wrong free-time advance, wrong record fields."""
    p = wl.ring_all_gather(n, False, seed)
    s = run(p)
    exp = [((i - k) % n, i, (i + 1) % n, i, k * W1M, (k + 1) * W1M) for k in range(n - 1) for i in range(n)]
    got = [tuple(int(x) for x in r) for r in s.transfers]
    assert got == exp
    assert s.time_ps == (n - 1) * W1M
    assert s.events == n


def test_ring_golden_hash(golden_dir):
    g = _golden_kv(golden_dir, "closed_forms.txt")
    s = run(wl.ring_all_gather(4, False, 0))
    assert oracle.schedule_hash(s.transfers) == g["ring4_uni_allgather_schedule_hash"]
    assert run(wl.ring_all_gather(8, False, 0)).time_ps == int(g["ring8_uni_allgather_time_ps"])
    assert run(wl.ring_all_gather(8, True, 0)).time_ps == int(g["ring8_bi_allgather_time_ps"])


@pytest.mark.parametrize("n", [3, 4, 5, 6, 8, 9])
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_ring_bidirectional_time(n, seed):
    p = wl.ring_all_gather(n, True, seed)
    s = run(p)
    assert s.time_ps == -(-(n - 1) // 2) * W1M
    assert len(s.transfers) == n * (n - 1)
    checker.check_schedule(p, s.transfers)


@pytest.mark.parametrize("kind", ["allgather", "alltoall"])
@pytest.mark.parametrize("n", [2, 4, 7])
def test_full_mesh_one_step(kind, n):
    """full mesh: every (src, dest) pair is one hop: T = w, M = N(N-1)."""
    p = wl.full_mesh_problem(n, kind, seed=3)
    s = run(p)
    assert s.time_ps == W1M and len(s.transfers) == n * (n - 1) and s.events == 2
    checker.check_schedule(p, s.transfers)


@pytest.mark.parametrize("n", [2, 3, 6])
def test_point_to_point_on_a_path(n):
    """T = hops * w; the middle nodes are not group members and only relay."""
    p = wl.path_point_to_point(n, seed=1)
    s = run(p)
    assert s.time_ps == (n - 1) * W1M and len(s.transfers) == n - 1
    assert [int(r["dst"]) for r in s.transfers] == list(range(1, n))
    checker.check_schedule(p, s.transfers)


def test_heterogeneous_two_hop_timing():
    """PAPER.md:334-340 / Fig. 9-10: link times differ; event times are not multiples of one w;
    a busy link stays busy for its whole interval.  0 -> 1 slow, 1 -> 2 fast; two chunks 0 -> 2."""
    links = np.array([(0, 1, 1000, 1), (1, 2, 10, 100)], dtype=wl.LINK_DT)
    pre = np.array([(0, 0), (0, 1)], dtype=wl.PAIR_DT)
    post = np.array([(2, 0), (2, 1)], dtype=wl.PAIR_DT)
    s = oracle.synthesize(3, links, np.array([0, 2], np.uint32), 2, pre, post, 500, 9)
    w0, w1 = 1000 + 500, 10 + 5
    t = s.transfers
    assert [(int(r["link"]), int(r["t_start_ps"]), int(r["t_end_ps"])) for r in t] == [
        (0, 0, w0), (0, w0, 2 * w0), (1, w0, w0 + w1), (1, 2 * w0, 2 * w0 + w1)]
    assert s.time_ps == 2 * w0 + w1
    assert sorted(int(c) for c in t["chunk"][:2]) == [0, 1]
    assert t["chunk"][2] == t["chunk"][0] and t["chunk"][3] == t["chunk"][1]


# --------------------------------------------------------------------------- pick / conflict (a6, a7)
def _list_model_parallel_links(n_links, n_chunks, w, seed):
    """2 nodes, n_links parallel links 0 -> 1, all chunks at 0 wanted by 1.  Written from
    DESIGN.md steps E1-E3 with Python lists and the harness Philox."""
    remaining = list(range(n_chunks))
    recs = []
    t = 0
    while remaining:
        for l in range(n_links):          # ascending link id, each sees earlier claims
            if not remaining:
                break
            r = int(wl.philox_first_word(t & 0xFFFFFFFF, t >> 32, l, 0, seed))
            k = (r * len(remaining)) >> 32
            recs.append((remaining.pop(k), 0, 1, l, t, t + w))
        t += w
    return recs


@pytest.mark.parametrize("n_links,n_chunks,seed", [(1, 9, 0), (1, 70, 1), (2, 33, 2), (3, 100, 0xDEADBEEF12345678)])
def test_pick_rule_and_conflict_order_on_parallel_links(n_links, n_chunks, seed):
    """catches: k-th LARGEST instead of smallest, counter words in the wrong order, seed halves
    swapped, tag not 0, in-links not serial (a later link not seeing an earlier claim)."""
    links = np.array([(0, 1, 5_000_000_000, 3)] * n_links, dtype=wl.LINK_DT)   # t exceeds 2^32
    pre = np.array([(0, c) for c in range(n_chunks)], dtype=wl.PAIR_DT)
    post = np.array([(1, c) for c in range(n_chunks)], dtype=wl.PAIR_DT)
    s = oracle.synthesize(2, links, np.array([0, 1], np.uint32), n_chunks, pre, post, 100, seed)
    w = 5_000_000_000 + 34
    got = [tuple(int(x) for x in r) for r in s.transfers]
    assert got == _list_model_parallel_links(n_links, n_chunks, w, seed)


def test_relay_choice_uses_tag_1_and_chunk_node_key():
    """2x2 mesh, chunk from 0 to 3: two tight predecessors of node 3 (1 via link id order, 2).
    The choice must equal (Philox(ctr=(c, cur, 0, 1)) * 2) >> 32 over in-links in ascending id."""
    links = wl.grid_links((2, 2), wrap=False)
    inl3 = [l for l in range(len(links)) if links["dst"][l] == 3]
    assert len(inl3) == 2
    for seed in range(6):
        for c_id in range(3):
            n_chunks = c_id + 1
            pre = np.array([(0, c) for c in range(n_chunks)], dtype=wl.PAIR_DT)
            post = np.array([(3, c) for c in range(n_chunks)], dtype=wl.PAIR_DT)
            src = np.zeros(n_chunks, np.uint32)
            off = np.arange(n_chunks + 1, dtype=np.uint64)
            dests = np.full(n_chunks, 3, np.uint32)
            wp = oracle.wants(4, links, n_chunks, src, off, dests, 1 << 20, seed)
            relay = [int(v) for v, c in zip(wp["npu"], wp["chunk"]) if c == c_id and v != 3]
            j = (int(wl.philox_first_word(c_id, 3, 0, 1, seed)) * 2) >> 32
            assert relay == [int(links["src"][inl3[j]])]


# --------------------------------------------------------------------------- brute force
def _bf_cases():
    cases = []
    for n in (3, 4):
        cases.append((wl.ring_all_gather(n, False), True))
        cases.append((wl.ring_all_gather(n, True), True))
    cases.append((wl.full_mesh_problem(3, "allgather"), True))
    cases.append((wl.full_mesh_problem(3, "alltoall"), True))
    cases.append((wl.path_point_to_point(4), True))
    links = wl.grid_links((2, 2), wrap=False)
    nc, pre, post = wl.all_gather(np.arange(4))
    cases.append((wl.Problem("mesh2x2_ag", 4, links, np.arange(4, dtype=np.uint32), nc, pre, post, 1 << 20, 0), True))
    nc, pre, post = wl.all_gather(np.arange(4), 2)
    cases.append((wl.Problem("ring4_ag_k2", 4, wl.ring_links(4, False), np.arange(4, dtype=np.uint32), nc, pre, post, 1 << 20, 0), False))
    nc, pre, post = wl.all_to_all(np.arange(4))
    cases.append((wl.Problem("ring4bi_a2a", 4, wl.ring_links(4, True), np.arange(4, dtype=np.uint32), nc, pre, post, 1 << 20, 0), False))
    return cases


@pytest.mark.parametrize("case", _bf_cases(), ids=lambda c: c[0].name)
def test_oracle_time_vs_bruteforce_optimum(case):
    """T_oracle >= T_opt always; equality on the families where greedy is optimal.  catches:
    forwarding before arrival (would beat the optimum), lost parallelism (would exceed it)."""
    p, expect_equal = case
    opt = brute_force.optimal_rounds_problem(p)
    for seed in range(4):
        p.seed = seed
        s = run(p)
        checker.check_schedule(p, s.transfers)
        assert s.time_ps % W1M == 0
        rounds = s.time_ps // W1M
        assert rounds >= opt
        if expect_equal:
            assert rounds == opt


# --------------------------------------------------------------------------- invariants on the configs
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
@pytest.mark.parametrize("maker", [wl.config1, wl.config2, wl.config3, wl.config4_small,
                                   wl.config5_small, wl.two_groups_mesh3x3], ids=lambda f: f.__name__)
def test_invariants_hold_on_configs(maker, seed):
    """V1-V7 (oracle/checker.py) on every small config, plus M = popcount(wants)."""
    p = maker(seed)
    s = run(p)
    st = checker.check_schedule(p, s.transfers)
    assert len(s.transfers) == s.wants_total
    assert st["time_ps"] == s.time_ps


def test_config1_ingress_bound_and_first_step():
    """4x4 torus AG: ingress bound ceil(15/4) = 4 steps; at t = 0 link 4u+j carries chunk u."""
    for seed in range(4):
        s = run(wl.config1(seed))
        assert s.time_ps in (4 * W1M, 5 * W1M)
        first = s.transfers[s.transfers["t_start_ps"] == 0]
        assert len(first) == 64
        assert np.array_equal(first["chunk"], first["link"] // 4)
        assert np.array_equal(first["src"], first["link"] // 4)


def test_config4_small_meets_work_bound_sanely():
    p = wl.config4_small(0)
    s = run(p)
    w = int(checker.link_costs(p.links, p.chunk_bytes)[0])

    def hop(sid):
        return (oracle.distances(p.n_npus, p.links, p.chunk_bytes, sid) // np.uint64(w)).astype(np.int64)
    lb = checker.lower_bound_homogeneous(p, hop)
    assert lb == 32 * w                      # 64 * 192 / 384 link-rounds
    assert lb <= s.time_ps <= 2 * lb


# --------------------------------------------------------------------------- reductions (a9)
@pytest.mark.parametrize("n", [3, 4, 6])
def test_reduce_scatter_on_ring_mirrors_all_gather(n):
    """Reduce-Scatter = reversed All-Gather: same makespan, same transfer count,
    and the simulated reduction delivers every contribution exactly once to the root."""
    links = wl.ring_links(n, False)
    members = list(range(n))
    nc, pre, post = wl.reduce_scatter_groups([members])
    p = wl.Problem("ring_rs", n, links, np.arange(n, dtype=np.uint32), nc, pre, post, 1 << 20, 0)
    s = run(p)
    assert s.mode == 1
    assert s.time_ps == (n - 1) * W1M and len(s.transfers) == n * (n - 1)
    checker.check_schedule(p, s.transfers)
    # transfers run in the links' own direction (transposed synthesis, reading Q10)
    assert np.array_equal(s.transfers["dst"], (s.transfers["src"] + 1) % n)


def test_reduce_on_asymmetric_topology_uses_real_links():
    """directed 3-cycle 0->1->2->0 plus 2->1: Reduce to NPU 0 must only use existing directions."""
    links = np.array([(0, 1, 10, 1), (1, 2, 10, 1), (2, 0, 10, 1), (2, 1, 10, 1)], dtype=wl.LINK_DT)
    pre = np.array([(0, 0), (1, 0), (2, 0)], dtype=wl.PAIR_DT)
    post = np.array([(0, 0)], dtype=wl.PAIR_DT)
    p = wl.Problem("asym_reduce", 3, links, np.arange(3, dtype=np.uint32), 1, pre, post, 5, 0)
    s = run(p)
    checker.check_schedule(p, s.transfers)
    assert [(int(r["src"]), int(r["dst"])) for r in s.transfers] == [(1, 2), (2, 0)]
    assert s.time_ps == 30


@pytest.mark.parametrize("seed", [0, 1])
def test_all_reduce_is_reduce_then_copy(seed):
    p = wl.config2(seed)
    s = run(p)
    assert s.mode == 2
    t = s.transfers
    ph1 = t[t["t_start_ps"] < s.time_phase1_ps]
    ph2 = t[t["t_start_ps"] >= s.time_phase1_ps]
    assert ph1["t_end_ps"].max() == s.time_phase1_ps          # phases do not overlap (reading Q11)
    assert ph2["t_end_ps"].max() == s.time_ps
    assert len(ph1) + len(ph2) == len(t) == s.wants_total
    # phase-2 sources that originate a chunk are the chunk's root G[c mod 16]
    G = p.group
    first_send = {}
    for r in ph2:
        first_send.setdefault(int(r["chunk"]), int(r["src"]))
    assert all(first_send[c] == int(G[c % 16]) for c in first_send)


# --------------------------------------------------------------------------- errors
def test_error_codes():
    links = wl.ring_links(3, False)
    g = np.arange(3, dtype=np.uint32)
    nc, pre, post = wl.all_gather(g)

    def code(**kw):
        a = dict(n_npus=3, links=links, group=g, n_chunks=nc, pre=pre, post=post, chunk_bytes=1024, seed=0)
        a.update(kw)
        try:
            oracle.synthesize(**a)
        except oracle.OracleError as e:
            return e.code
        return 0
    assert code() == 0
    assert code(chunk_bytes=0) == oracle.ERR_INVALID
    bad = links.copy(); bad["dst"][0] = 7
    assert code(links=bad) == oracle.ERR_INVALID
    bad = links.copy(); bad["dst"][0] = bad["src"][0]
    assert code(links=bad) == oracle.ERR_INVALID
    bad = links.copy(); bad["bytes_per_ps"][1] = 0
    assert code(links=bad) == oracle.ERR_INVALID
    assert code(group=np.array([0, 1, 1], np.uint32)) == oracle.ERR_INVALID
    assert code(group=np.array([0, 1], np.uint32)) == oracle.ERR_INVALID      # pair outside group
    assert code(n_chunks=nc + 1) == oracle.ERR_INVALID                        # chunk without holders
    assert code(links=links[:2]) == oracle.ERR_UNREACHABLE                    # ring cut open
    mixed_pre = np.concatenate([pre, np.array([(1, 0)], dtype=wl.PAIR_DT)])   # chunk 0 reduced, others copied
    assert code(pre=mixed_pre) == oracle.ERR_UNSUPPORTED


def test_empty_and_trivial_problems():
    links = wl.ring_links(3, False)
    g = np.arange(3, dtype=np.uint32)
    e = np.zeros(0, dtype=wl.PAIR_DT)
    s = oracle.synthesize(3, links, g, 0, e, e, 1024, 0)
    assert len(s.transfers) == 0 and s.time_ps == 0
    same = np.array([(1, 0)], dtype=wl.PAIR_DT)                               # already in place
    s = oracle.synthesize(3, links, g, 1, same, same, 1024, 0)
    assert len(s.transfers) == 0 and s.time_ps == 0
