"""Pins of the oracle's DYNAMIC relay mode (reading Q18), no GPU.

The rule is not the paper's (the paper floods the TEN and filters paths afterwards,
PAPER.md:294-300); what the paper fixes still binds it and is checked here: valid schedules
(checker), closed forms where every valid greedy must agree, the brute-force lower bound.
The rule itself -- "a node takes a chunk only if it is strictly closer to some destination
than the source and every node that claimed the chunk at an EARLIER event" -- is re-derived
from the emitted schedule with scipy distances, so a wrong sign, a non-strict comparison or
an update applied inside the event instead of at its end fails here.  The first test below is the necessary
side (every claim satisfied the rule); test_the_rule_is_work_conserving is the sufficient side (at every event
every free link whose candidate set under the rule is non-empty starts a transfer of one of exactly those
candidates), which is what catches an update applied too early (claims would go missing) or a link left idle.
"""
import numpy as np
import pytest

import oracle
import workloads as wl
from oracle import brute_force, checker

W1M = 520_972  # tests/golden/closed_forms.txt
DYN = oracle.RELAY_DYNAMIC


def run(p, relay=DYN):
    return oracle.synthesize(*p.args(), relay=relay)


def _dist_to(p):
    """dist[d][v] = alpha-beta shortest path cost v -> d (scipy, independent of the oracle)."""
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import dijkstra
    w = checker.link_costs(p.links, p.chunk_bytes).astype(np.float64)
    n = p.n_npus
    # parallel links: keep the cheapest
    best = {}
    for l, c in zip(p.links, w):
        k = (int(l["dst"]), int(l["src"]))          # reversed graph: distances TO a node
        best[k] = min(best.get(k, np.inf), c)
    rows, cols = zip(*best.keys())
    g = csr_matrix((list(best.values()), (rows, cols)), shape=(n, n))
    return dijkstra(g, directed=True)                # [d][v]


def _conditions(p):
    """chunk -> (src, dests) for COPY problems."""
    src = {int(r["chunk"]): int(r["npu"]) for r in p.pre}
    dests = {}
    for r in p.post:
        c, v = int(r["chunk"]), int(r["npu"])
        if v != src[c]:
            dests.setdefault(c, []).append(v)
    return src, dests


@pytest.mark.parametrize("maker", [wl.config1, wl.config4_small, wl.two_groups_mesh3x3,
                                   lambda s: wl.ring_all_gather(7, True, s, chunks_per_npu=3),
                                   lambda s: wl.path_point_to_point(5, s)])
@pytest.mark.parametrize("seed", [0, 1])
def test_every_claim_was_strictly_closer_than_all_earlier_holders(maker, seed):
    p = maker(seed)
    s = run(p)
    D = _dist_to(p)
    src, dests = _conditions(p)
    holders = {c: [(0 - 1, src[c])] for c in src}    # (claim time, node); the source "claimed" before t = 0
    tr = s.transfers
    for i in np.argsort(tr["t_start_ps"], kind="stable"):
        r = tr[i]
        c, v, t = int(r["chunk"]), int(r["dst"]), int(r["t_start_ps"])
        earlier = [h for (th, h) in holders[c] if th < t]     # claims of the SAME event do not count yet
        assert any(D[d][v] < min(D[d][h] for h in earlier) for d in dests[c]), \
            f"{p.name}: node {v} took chunk {c} at {t} without being strictly closer to any dest"
        assert v not in [h for (_, h) in holders[c]], "a node claims a chunk at most once"
        holders[c].append((t, v))
    # and nothing useful was left undone: every dest holds its chunks (checker V4)
    checker.check_schedule(p, tr)


def _torus3_a2a(seed):
    m = np.arange(27, dtype=np.uint32)
    nc, pre, post = wl.all_to_all(m)
    return wl.Problem("torus3x3x3_alltoall", 27, wl.grid_links((3, 3, 3), wrap=True), m, nc, pre, post, 1 << 16, seed)


def _mesh_multi_dest(seed):
    """4x3 mesh, 10 chunks with 2..6 dests each, heterogeneous links: multi-dest chunks, several claimants per chunk"""
    rng = np.random.default_rng(77 + seed)
    links = wl.grid_links((4, 3), wrap=False).copy()
    links["alpha_ps"] = rng.integers(100, 900, len(links))
    links["bytes_per_ps"] = rng.integers(1, 9, len(links))
    m = np.arange(12, dtype=np.uint32)
    pre, post = [], []
    for c in range(10):
        s = int(rng.integers(0, 12))
        pre.append((s, c))
        for d in rng.choice(12, size=int(rng.integers(2, 7)), replace=False):
            post.append((int(d), c))
    return wl.Problem("mesh4x3_multidest", 12, links, m, 10, np.array(pre, dtype=wl.PAIR_DT), np.array(post, dtype=wl.PAIR_DT),
                      2000, seed)


@pytest.mark.parametrize("maker", [wl.config1, wl.two_groups_mesh3x3, _torus3_a2a, _mesh_multi_dest,
                                   lambda s: wl.ring_all_gather(7, True, s, chunks_per_npu=3),
                                   lambda s: wl.path_point_to_point(5, s)], ids=lambda m: getattr(m, "__name__", "case"))
@pytest.mark.parametrize("seed", [0, 1])
def test_the_rule_is_work_conserving(maker, seed):
    """The sufficient side of reading Q18, event by event, from the emitted schedule alone (scipy distances):
    at every event time t and for every node v, its in-links in ascending id that are free at t are served in turn;
    candidates of link l = chunks its source holds by t (own, or delivered with t_end <= t) that v has not claimed
    before t nor at t through an earlier in-link, and for which v is strictly closer to some dest than the source and
    every claimant of an event BEFORE t.  A non-empty candidate set must start a transfer of one of its members at t;
    an empty one must not start anything."""
    p = maker(seed)
    tr = run(p).transfers
    D = _dist_to(p)
    src, dests = _conditions(p)
    n, L, C = p.n_npus, len(p.links), p.n_chunks
    inl = [[] for _ in range(n)]
    for l in range(L):
        inl[int(p.links[l]["dst"])].append(l)
    starts = {}                                   # (t_start, link) -> chunk
    for r in tr:
        starts[(int(r["t_start_ps"]), int(r["link"]))] = int(r["chunk"])
    events = sorted({0} | {int(x) for x in tr["t_end_ps"]})
    assert {int(x) for x in tr["t_start_ps"]} <= set(events)
    for t in events:
        done = tr[tr["t_end_ps"] <= t]
        before = tr[tr["t_start_ps"] < t]
        have = np.zeros((n, C), dtype=bool)
        for c, s_ in src.items():
            have[s_, c] = True
        have[done["dst"], done["chunk"]] = True
        claimed = np.zeros((n, C), dtype=bool)
        claimed[before["dst"], before["chunk"]] = True
        wants = np.zeros((n, C), dtype=bool)
        for c, ds in dests.items():
            holders = [src[c]] + [int(v) for v in before["dst"][before["chunk"] == c]]
            for d in ds:
                wants[:, c] |= D[d] < min(D[d][h] for h in holders)
        wants &= ~claimed
        busy = set(int(l) for l in before["link"][before["t_end_ps"] > t])
        for v in range(n):
            now = set()
            for l in inl[v]:
                if l in busy:
                    assert (t, l) not in starts
                    continue
                cand = {int(c) for c in np.nonzero(have[int(p.links[l]["src"])] & wants[v])[0]} - now
                got = starts.get((t, l))
                if cand:
                    assert got in cand, f"{p.name}: t={t} link {l}: candidates {sorted(cand)[:8]}.. but the link carries {got}"
                    now.add(got)
                else:
                    assert got is None, f"{p.name}: t={t} link {l} carries {got} with no candidate under the rule"


@pytest.mark.parametrize("maker", [wl.config1, wl.config2, wl.config3, wl.config4_small, wl.config5_small,
                                   wl.two_groups_mesh3x3], ids=lambda m: getattr(m, "__name__", "x"))
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_dynamic_schedules_are_valid(maker, seed):
    p = maker(seed)
    s = run(p)
    checker.check_schedule(p, s.transfers)
    assert s.time_ps == int(s.transfers["t_end_ps"].max())
    assert len(s.transfers) <= s.wants_total          # a (node, chunk) pair is claimed at most once


@pytest.mark.parametrize("n", [2, 3, 5, 8])
@pytest.mark.parametrize("seed", [0, 1])
def test_ring_unidirectional_is_the_same_exact_schedule(n, seed):
    """one candidate per link per event: both relay rules must emit the textbook ring All-Gather."""
    p = wl.ring_all_gather(n, False, seed)
    a, b = run(p, oracle.RELAY_THIN), run(p)
    assert b.time_ps == (n - 1) * W1M and len(b.transfers) == n * (n - 1)
    for f in a.transfers.dtype.names:
        assert np.array_equal(a.transfers[f], b.transfers[f])


@pytest.mark.parametrize("n", [3, 4, 5, 6, 9])
def test_ring_bidirectional_time(n):
    p = wl.ring_all_gather(n, True, seed=2)
    s = run(p)
    assert s.time_ps == -(-(n - 1) // 2) * W1M
    checker.check_schedule(p, s.transfers)


@pytest.mark.parametrize("kind", ["allgather", "alltoall"])
def test_full_mesh_one_step(kind):
    p = wl.full_mesh_problem(5, kind, seed=3)
    s = run(p)
    assert s.time_ps == W1M and s.events == 2
    assert len(s.transfers) == (20 if kind == "allgather" else 20)


@pytest.mark.parametrize("n", [2, 4, 6])
def test_point_to_point_on_a_path(n):
    p = wl.path_point_to_point(n, seed=1)
    s = run(p)
    assert s.time_ps == (n - 1) * W1M
    assert [int(r["dst"]) for r in s.transfers] == list(range(1, n))


def test_heterogeneous_prefers_the_fast_detour_by_distance_not_hops():
    """dist is the alpha-beta cost (reading Q3): 0 -> 3 directly is slow (cost 10000+), the
    two-hop detour 0 -> 1 -> 3 is cheap, 0 -> 2 leads away.  Node 1 is strictly closer to 3 than
    0 is, node 2 is not, so 2 never receives the chunk; the direct slow link is also a
    candidate at t = 0 and is taken (greedy), but the chunk arrives first over the detour."""
    links = np.array([(0, 3, 10_000, 1), (0, 1, 10, 100), (1, 3, 10, 100), (0, 2, 10, 100), (2, 0, 10, 100)],
                     dtype=wl.LINK_DT)
    pre = np.array([(0, 0)], dtype=wl.PAIR_DT)
    post = np.array([(3, 0)], dtype=wl.PAIR_DT)
    s = oracle.synthesize(4, links, np.array([0, 3], np.uint32), 1, pre, post, 100, 5, relay=DYN)
    got = [(int(r["link"]), int(r["t_start_ps"])) for r in s.transfers]
    assert (1, 0) in got and 3 not in [l for l, _ in got]          # 1 relays, 2 never takes it
    assert all(int(r["dst"]) != 2 for r in s.transfers)


def _bf_cases():
    return [wl.ring_all_gather(4, True, 0), wl.ring_all_gather(5, False, 1), wl.full_mesh_problem(4, "alltoall", 2),
            wl.path_point_to_point(4, 0),
            wl.Problem("mesh2x2_ag", 4, wl.grid_links((2, 2), wrap=False), np.arange(4, dtype=np.uint32),
                       *wl.all_gather(np.arange(4)), 1 << 20, 3)]


@pytest.mark.parametrize("case", _bf_cases(), ids=lambda c: c.name)
def test_time_not_below_bruteforce_optimum(case):
    s = run(case)
    rounds = brute_force.optimal_rounds_problem(case)
    assert s.time_ps >= rounds * W1M
    if case.name.startswith(("ring", "fullmesh", "path")):
        assert s.time_ps == rounds * W1M


def test_reductions_use_the_dynamic_rule_too():
    p = wl.config3(0)
    s = run(p)
    assert s.mode == 1
    checker.check_schedule(p, s.transfers)
    p = wl.config2(0)
    s = run(p)
    assert s.mode == 2 and s.time_ps > s.time_phase1_ps > 0
    checker.check_schedule(p, s.transfers)


def test_provisional_quality_4x4x4_all_to_all():
    """an independent scratch model gave 39-40 link-times for the 4x4x4-torus
    All-to-All under this rule (47-53 for the thin tree, lower bound 32)."""
    p = wl.config4_small(0)
    w = int(checker.link_costs(p.links, p.chunk_bytes)[0])
    a, b = run(p, oracle.RELAY_THIN), run(p)
    assert 39 * w <= b.time_ps <= 41 * w < a.time_ps
