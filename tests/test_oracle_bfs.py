"""Pins of the oracle's BFS mode -- the paper's own synthesizer, Algorithms 1-3 with the
heterogeneous rules of section 4.6 (Q19-Q22).  No GPU.

The oracle keeps per-link busy INTERVALS and finds departures by first fit; the pin below is
the paper's literal data structure instead: a boolean TEN[t][link] over integer timesteps,
searched timestep by timestep (Alg. 2), with every overlapping entry removed after a path is
taken (Fig. 10).  The two share nothing but the problem statement.  A dropped tie rule, an
off-by-one in the overlap test, a missed gap in front of a taken interval, a wrong sort
direction in Alg. 3 or a missing path filter all make the record lists differ.
"""
import numpy as np
import pytest

import oracle
import workloads as wl
from oracle import checker

BFS = oracle.RELAY_BFS


def run(p):
    return oracle.synthesize(*p.args(), relay=BFS)


def _links(triples):
    """(src, dst, cost) with integer cost >= 1: alpha = cost - 1, one byte per ps, 1-byte chunks."""
    a = np.zeros(len(triples), dtype=wl.LINK_DT)
    for i, (s, d, c) in enumerate(triples):
        a[i] = (s, d, c - 1, 1)
    return a


def _pairs(items):
    a = np.zeros(len(items), dtype=wl.PAIR_DT)
    for i, (v, c) in enumerate(items):
        a[i] = (v, c)
    return a


def _problem(name, n, triples, conds, seed=0, group=None):
    """conds: list of (src, [dests]); chunk id = index"""
    pre = _pairs([(s, c) for c, (s, _) in enumerate(conds)])
    post = _pairs([(d, c) for c, (_, ds) in enumerate(conds) for d in ds])
    if group is None:
        group = sorted({s for s, _ in conds} | {d for _, ds in conds for d in ds})
    return wl.Problem(name, n, _links(triples), np.array(group, dtype=np.uint32), len(conds), pre, post, 1, seed)


# ------------------------------------------------------------------ the literal TEN (brute force)
def _hop_costs(n, links, w, src):
    """Bellman-Ford on the idle network (ShortestPath of Alg. 3)"""
    D = [None] * n
    D[src] = 0
    for _ in range(n):
        for l, k in enumerate(links):
            u, v = int(k["src"]), int(k["dst"])
            if D[u] is not None and (D[v] is None or D[u] + w[l] < D[v]):
                D[v] = D[u] + w[l]
    return D


def literal_ten(n, links, conds, seed, removed0=None, ready=None):
    """Alg. 3 over Alg. 2 on a boolean TEN[t][link] (stored as the set of removed entries).
    removed0 / ready: entries already taken and the timestep from which each chunk is at its source (pipelined All-Reduce)."""
    w = [int(k["alpha_ps"]) + 1 for k in links]
    removed = set(removed0 or ())                     # (t, link): TEN entry taken
    keyed = []
    for c, (src, dests) in enumerate(conds):
        if not dests:
            continue
        D = _hop_costs(n, links, w, src)
        keyed.append((-max(D[d] for d in dests), int(wl.philox_first_word(c, 0, 0, 2, seed)), c))
    out = []
    for _, _, c in sorted(keyed):                     # Alg. 3 line 7 (+ reading Q19 for ties)
        src, dests = conds[c]
        arr, pred = {src: ready[c] if ready else 0}, {}
        t = 0
        while not all(d in arr and arr[d] <= t for d in dests):   # Alg. 2 line 4
            for l, k in enumerate(links):             # every TEN link that starts at timestep t
                u, v = int(k["src"]), int(k["dst"])
                if u not in arr or arr[u] > t:        # 4.6: the chunk must have arrived at `current`
                    continue
                if any((t + i, l) in removed for i in range(w[l])):
                    continue                          # overlaps a taken entry (Fig. 10)
                a = t + w[l]
                if v == src:
                    continue
                if v not in arr or a < arr[v] or (a == arr[v] and l < pred[v][0]):
                    arr[v], pred[v] = a, (l, t)
            t += 1
            assert t < 10_000
        keep = set()
        for d in dests:                               # keep the useful paths
            v = d
            while v != src and v not in keep:
                keep.add(v)
                v = int(links[pred[v][0]]["src"])
        for v in sorted(keep):
            l, ts = pred[v]
            out.append((ts, l, c, int(links[l]["src"]), v, ts + w[l]))
            for i in range(w[l]):                     # Alg. 3 line 13
                assert (ts + i, l) not in removed
                removed.add((ts + i, l))
    out.sort()
    return out


def _as_tuples(tr):
    return [(int(r["t_start_ps"]), int(r["link"]), int(r["chunk"]), int(r["src"]), int(r["dst"]), int(r["t_end_ps"]))
            for r in tr]


def _random_case(i):
    rng = np.random.default_rng(7000 + i)
    n = int(rng.integers(4, 10))
    triples = []
    perm = rng.permutation(n)
    for a in range(n):                                # a ring through all nodes keeps it strongly connected
        triples.append((int(perm[a]), int(perm[(a + 1) % n]), int(rng.integers(1, 5))))
    for _ in range(int(rng.integers(n, 3 * n))):
        u, v = rng.choice(n, 2, replace=False)
        triples.append((int(u), int(v), int(rng.integers(1, 5))))   # parallel links allowed
    members = sorted(rng.choice(n, int(rng.integers(2, n + 1)), replace=False).tolist())
    conds = []
    kind = i % 3
    for s in members:
        others = [m for m in members if m != s]
        if kind == 0:                                 # All-Gather like, several chunks per member
            conds += [(s, others)] * int(rng.integers(1, 4))
        elif kind == 1:                               # All-to-All like
            conds += [(s, [d]) for d in others for _ in range(int(rng.integers(0, 3)))]
        else:                                         # random dest subsets
            for _ in range(int(rng.integers(1, 4))):
                k = int(rng.integers(1, len(others) + 1))
                conds.append((s, sorted(rng.choice(others, k, replace=False).tolist())))
    if not conds:
        conds = [(members[0], [members[1]])]
    return n, triples, conds, members


@pytest.mark.parametrize("i", range(30))
def test_equals_the_literal_boolean_ten(i):
    n, triples, conds, members = _random_case(i)
    p = _problem(f"rand{i}", n, triples, conds, seed=i, group=members)
    s = run(p)
    assert _as_tuples(s.transfers) == literal_ten(n, p.links, conds, i)
    checker.check_schedule(p, s.transfers)


def test_reduction_is_the_reversed_search_on_the_transposed_links():
    """Reduce-Scatter = reversed All-Gather.  Literal TEN on the transposed links, every
    transfer reversed in direction and in time."""
    n, triples, _, _ = _random_case(3)
    members = list(range(n))
    # chunk c is reduced from all members into root c % n
    conds_b = [(c % n, [m for m in members if m != c % n]) for c in range(n + 2)]
    pre = _pairs([(m, c) for c in range(len(conds_b)) for m in members])
    post = _pairs([(c % n, c) for c in range(len(conds_b))])
    p = wl.Problem("rs", n, _links(triples), np.array(members, dtype=np.uint32), len(conds_b), pre, post, 1, 5)
    s = run(p)
    tl = p.links.copy()
    tl["src"], tl["dst"] = p.links["dst"], p.links["src"]
    b = literal_ten(n, tl, conds_b, 5)
    T = max(r[5] for r in b)
    want = sorted((T - te, l, c, v, u, T - ts) for ts, l, c, u, v, te in b)
    assert _as_tuples(s.transfers) == want
    assert s.time_ps == T


# ------------------------------------------------------------------ worked examples and closed forms
def test_worked_example_gap_in_front_of_a_taken_interval():
    """links: l0 = 0->1 cost 10, l1 = 1->2 cost 4, l2 = 3->1 cost 1.  Conditions (chunk: src -> dest):
    c0: 0->2 (dist 14), c1..c3: 3->2 (dist 5).  Alg. 3 routes c0 first: l0 [0,10), l1 [10,14).
    The three short ones follow in the order of their tie draws, whichever it is; the k-th of them leaves
    node 3 at k-1 (l2 is busy one step per chunk) and needs 4 free steps on l1:
      1st: l2 [0,1), l1 [1,5)      2nd: l2 [1,2), l1 [5,9)   (fits in front of [10,14))
      3rd: l2 [2,3), l1 [14,18)    ([9,13) would overlap [10,14))."""
    p = _problem("gap", 4, [(0, 1, 10), (1, 2, 4), (3, 1, 1)], [(0, [2]), (3, [2]), (3, [2]), (3, [2])], seed=11)
    s = run(p)
    got = sorted((int(r["link"]), int(r["t_start_ps"]), int(r["t_end_ps"])) for r in s.transfers)
    assert got == [(0, 0, 10), (1, 1, 5), (1, 5, 9), (1, 10, 14), (1, 14, 18), (2, 0, 1), (2, 1, 2), (2, 2, 3)]
    on_l1 = {int(r["t_start_ps"]): int(r["chunk"]) for r in s.transfers if r["link"] == 1}
    assert on_l1[10] == 0
    assert s.time_ps == 18


@pytest.mark.parametrize("k,m,cost", [(1, 5, 3), (4, 1, 7), (5, 6, 2)])
def test_pipeline_on_a_line(k, m, cost):
    """m chunks over a line of k equal links: the j-th routed leaves at j*cost on every hop's first free
    slot, so T = (k + m - 1) * cost and every link carries back-to-back transfers."""
    triples = [(i, i + 1, cost) for i in range(k)]
    p = _problem("line", k + 1, triples, [(0, [k])] * m)
    s = run(p)
    assert s.time_ps == (k + m - 1) * cost
    assert len(s.transfers) == k * m
    for l in range(k):
        starts = sorted(int(r["t_start_ps"]) for r in s.transfers if r["link"] == l)
        assert starts == [(l + j) * cost for j in range(m)]


def test_longest_condition_goes_first_and_gets_its_shortest_path():
    """Alg. 3 line 7: the condition with the largest c.dist is routed on the idle network, so it arrives
    after exactly c.dist even though a shorter condition competes for its first link."""
    #  0 -> 1 -> 2 -> 3   and a short condition 0 -> 1
    p = _problem("order", 4, [(0, 1, 2), (1, 2, 2), (2, 3, 2)], [(0, [1]), (0, [3])])
    s = run(p)
    long_ = s.transfers[s.transfers["chunk"] == 1]
    assert sorted(int(t) for t in long_["t_end_ps"]) == [2, 4, 6]
    short = s.transfers[s.transfers["chunk"] == 0]
    assert (int(short["t_start_ps"][0]), int(short["t_end_ps"][0])) == (2, 4)


def test_lowest_link_id_wins_equal_arrivals():
    """reading Q20: two parallel links and a two-hop detour all reach node 1 at time 4"""
    p = _problem("tie", 3, [(0, 2, 2), (0, 1, 4), (2, 1, 2), (0, 1, 4)], [(0, [1])])
    s = run(p)
    assert [(int(r["link"]), int(r["t_start_ps"])) for r in s.transfers] == [(1, 0)]


def test_broadcast_keeps_only_useful_paths():
    """a star with 5 leaves, dests = 2 of them: exactly 2 transfers"""
    p = _problem("filter", 6, [(0, i, 1) for i in range(1, 6)], [(0, [2, 4])])
    s = run(p)
    assert sorted(int(d) for d in s.transfers["dst"]) == [2, 4]


def test_non_members_relay(tmp_path):
    """links outside the process group are used"""
    p = wl.two_groups_mesh3x3(0)
    s = run(p)
    checker.check_schedule(p, s.transfers)
    touched = set(s.transfers["src"].tolist()) | set(s.transfers["dst"].tolist())
    assert touched - set(p.group.tolist())


def test_unreachable():
    p = _problem("unreach", 3, [(0, 1, 1)], [(0, [2])])
    with pytest.raises(oracle.OracleError) as e:
        run(p)
    assert e.value.code == oracle.ERR_UNREACHABLE


# ------------------------------------------------------------------ the paper's workload shapes
@pytest.mark.parametrize("maker", [wl.config1, wl.config2, wl.config3, wl.config4_small, wl.config5_small])
def test_valid_on_the_configs(maker):
    p = maker(0)
    s = run(p)
    checker.check_schedule(p, s.transfers)
    assert s.events > 0


def test_first_routed_condition_takes_c_dist():
    """on config 1 (16 equal conditions on an idle 4x4 torus) T can not be below the eccentricity, and the
    first routed chunk reaches its farthest dest after exactly 4 hops"""
    p = wl.config1(0)
    s = run(p)
    w = int(checker.link_costs(p.links, p.chunk_bytes)[0])
    assert s.time_ps >= 4 * w
    first = int(np.lexsort((np.arange(16), wl.philox_first_word(np.arange(16), 0, 0, 2, p.seed)))[0])
    assert int(s.transfers[s.transfers["chunk"] == first]["t_end_ps"].max()) == 4 * w


# ------------------------------------------------------------------ section 4.7: switches (Q23-Q25)
def literal_ten_switches(n, links, conds, seed, limit, nomc):
    """The literal TEN again, with the paper's two switch rules written timestep by timestep: a visit of node v at
    timestep a is skipped while limit[v] chunks of EARLIER conditions are buffered there at a (a stay lasts from the
    arrival to the end of the last kept transfer out); a node in `nomc` starts its out-links one at a time, in ascending
    link id, the next no earlier than the end of the one before."""
    w = [int(k["alpha_ps"]) + 1 for k in links]
    out_links = [[l for l, k in enumerate(links) if int(k["src"]) == u] for u in range(n)]
    removed = set()
    stays = {v: [] for v in range(n)}
    keyed = []
    for c, (src, dests) in enumerate(conds):
        if dests:
            D = _hop_costs(n, links, w, src)
            keyed.append((-max(D[d] for d in dests), int(wl.philox_first_word(c, 0, 0, 2, seed)), c))
    out = []

    def full(v, a):
        return v in limit and sum(1 for (x, y) in stays[v] if x <= a < y) >= limit[v]

    for _, _, c in sorted(keyed):
        src, dests = conds[c]
        arr, pred = {src: 0}, {}
        ptr, busy_until = {}, {}                       # no-multicast nodes: next out-link to serve, end of the current send
        t = 0
        while not all(d in arr and arr[d] <= t for d in dests):
            for u in range(n):
                if u not in arr or arr[u] > t:
                    continue
                if u in nomc:
                    ptr.setdefault(u, 0)
                    if t < busy_until.get(u, 0) or ptr[u] >= len(out_links[u]):
                        continue
                    todo = [out_links[u][ptr[u]]]
                else:
                    todo = out_links[u]
                for l in todo:
                    v = int(links[l]["dst"])
                    if limit.get(v, 1) == 0:           # never visitable: the turn passes without a send
                        if u in nomc:
                            ptr[u] += 1
                        continue
                    if any((t + i, l) in removed for i in range(w[l])) or full(v, t + w[l]):
                        continue                       # (a serial node waits at this out-link)
                    a = t + w[l]
                    if u in nomc:
                        ptr[u] += 1
                        busy_until[u] = a
                    if v == src:
                        continue
                    if v not in arr or a < arr[v] or (a == arr[v] and l < pred[v][0]):
                        arr[v], pred[v] = a, (l, t)
            t += 1
            assert t < 10_000
        keep = set()
        for d in dests:
            v = d
            while v != src and v not in keep:
                keep.add(v)
                v = int(links[pred[v][0]]["src"])
        last_out = {}
        for v in sorted(keep):
            l, ts = pred[v]
            out.append((ts, l, c, int(links[l]["src"]), v, ts + w[l]))
            for i in range(w[l]):
                assert (ts + i, l) not in removed
                removed.add((ts + i, l))
            u = int(links[l]["src"])
            last_out[u] = max(last_out.get(u, 0), ts + w[l])
        for v in keep:
            if v in limit and v in last_out:
                stays[v].append((arr[v], last_out[v]))
    out.sort()
    return out


def _switch_arrays(n, limit, nomc):
    bl = np.full(n, oracle.NO_LIMIT, dtype=np.uint32)
    for v, k in limit.items():
        bl[v] = k
    nm = np.zeros(n, dtype=np.uint8)
    nm[list(nomc)] = 1
    return bl, nm


@pytest.mark.parametrize("i", range(40))
def test_switch_rules_against_the_literal_ten(i):
    n, triples, conds, members = _random_case(i)
    rng = np.random.default_rng(8100 + i)
    others = [v for v in range(n) if v not in members] or list(range(n))
    limit = {int(v): int(rng.integers(1, 3)) for v in rng.choice(others, size=min(len(others), int(rng.integers(1, 4))), replace=False)} if i % 4 != 3 else {}
    nomc = set(int(v) for v in rng.choice(n, size=int(rng.integers(1, 3)), replace=False)) if i % 2 else set()
    p = _problem(f"sw{i}", n, triples, conds, seed=i, group=members)
    bl, nm = _switch_arrays(n, limit, nomc)
    s = oracle.synthesize(*p.args(), relay=BFS, buffer_limit=bl, no_multicast=nm)
    assert _as_tuples(s.transfers) == literal_ten_switches(n, p.links, conds, i, limit, nomc)
    checker.check_structure(p, s.transfers)


def test_no_limits_is_the_plain_bfs_mode():
    for i in range(6):
        n, triples, conds, members = _random_case(i)
        p = _problem(f"sw_none{i}", n, triples, conds, seed=i, group=members)
        bl, nm = _switch_arrays(n, {}, set())
        a = oracle.synthesize(*p.args(), relay=BFS, buffer_limit=bl, no_multicast=nm)
        b = run(p)
        assert _as_tuples(a.transfers) == _as_tuples(b.transfers)
    for mk in (wl.config3, wl.config4_small):
        p = mk(0)
        bl, nm = _switch_arrays(p.n_npus, {}, set())
        a = oracle.synthesize(*p.args(), relay=BFS, buffer_limit=bl, no_multicast=nm)
        assert _as_tuples(a.transfers) == _as_tuples(run(p).transfers)


def test_buffer_limit_hand_example():
    """NPUs 0, 1 -> switch 2 -> NPUs 3, 4, unit links.  Two chunks (0 -> 3, 1 -> 4) cross the switch side by side in two
    timesteps when it buffers two chunks; with a one-chunk buffer the second may only ARRIVE once the first has left:
    it starts at 1 (arrival 2 = the first one's release), leaves over [2, 3): three timesteps."""
    tri = [(0, 2, 1), (1, 2, 1), (2, 3, 1), (2, 4, 1)]
    conds = [(0, [3]), (1, [4])]
    p = _problem("two_through_one_switch", 5, tri, conds, seed=0, group=[0, 1, 3, 4])
    assert run(p).time_ps == 2
    bl, nm = _switch_arrays(5, {2: 1}, set())
    s = oracle.synthesize(*p.args(), relay=BFS, buffer_limit=bl, no_multicast=nm)
    assert s.time_ps == 3
    t = _as_tuples(s.transfers)
    into = sorted(r for r in t if r[4] == 2)
    assert [r[0] for r in into] == [0, 1] and [r[5] for r in into] == [1, 2]      # arrivals at the switch: 1, then 2
    bl2, _ = _switch_arrays(5, {2: 2}, set())
    assert oracle.synthesize(*p.args(), relay=BFS, buffer_limit=bl2, no_multicast=nm).time_ps == 2
    bl0, _ = _switch_arrays(5, {2: 0}, set())
    with pytest.raises(oracle.OracleError) as e:                                    # a switch without buffers cannot relay
        oracle.synthesize(*p.args(), relay=BFS, buffer_limit=bl0, no_multicast=nm)
    assert e.value.code == oracle.ERR_UNREACHABLE


def test_no_multicast_hand_example():
    """0 -> switch 1 -> {2, 3, 4}: one chunk for all three.  With multicast the switch sends the three copies at once
    (arrivals 2, 2, 2); without, one after the other in link order (arrivals 2, 3, 4)."""
    tri = [(0, 1, 1), (1, 2, 1), (1, 3, 1), (1, 4, 1)]
    p = _problem("fanout", 5, tri, [(0, [2, 3, 4])], seed=0, group=[0, 2, 3, 4])
    assert sorted(r[5] for r in _as_tuples(run(p).transfers) if r[3] == 1) == [2, 2, 2]
    bl, nm = _switch_arrays(5, {}, {1})
    s = oracle.synthesize(*p.args(), relay=BFS, buffer_limit=bl, no_multicast=nm)
    assert [(r[4], r[0], r[5]) for r in _as_tuples(s.transfers) if r[3] == 1] == [(2, 1, 2), (3, 2, 3), (4, 3, 4)]
    assert s.time_ps == 4


def test_switch_model_on_config3():
    """config 3's pod switches with two-chunk buffers and no multicast: still a valid Reduce-Scatter, not faster than
    with ideal switches, and every visit respected the buffers of the conditions routed before it."""
    p = wl.config3(0)
    base = run(p)
    bl = np.full(p.n_npus, oracle.NO_LIMIT, dtype=np.uint32)
    bl[64:] = 2
    nm = np.zeros(p.n_npus, dtype=np.uint8)
    nm[64:] = 1
    s = oracle.synthesize(*p.args(), relay=BFS, buffer_limit=bl, no_multicast=nm)
    checker.check_schedule(p, s.transfers)
    assert s.time_ps >= base.time_ps and len(s.transfers) >= 1408


# ------------------------------------------------------------------ pipelined All-Reduce (Q26)
def _allreduce_case(i):
    rng = np.random.default_rng(9100 + i)
    n = int(rng.integers(4, 9))
    triples = []
    perm = rng.permutation(n)
    for a in range(n):
        u, v = int(perm[a]), int(perm[(a + 1) % n])
        c = int(rng.integers(1, 4))
        triples += [(u, v, c), (v, u, c)]              # both directions: the reduce phase runs on the transposed links
    for _ in range(int(rng.integers(0, n))):
        u, v = rng.choice(n, 2, replace=False)
        triples.append((int(u), int(v), int(rng.integers(1, 4))))
    members = sorted(rng.choice(n, int(rng.integers(2, n + 1)), replace=False).tolist())
    nc = int(rng.integers(1, 7))
    return n, triples, members, nc


def literal_pipelined_allreduce(n, links, members, nc, seed):
    """Reduce phase = the literal TEN on the transposed links, reversed in time and direction; the copy
    phase of chunk c starts at the end of the last transfer of c into its root, on a TEN from which the reduce phase's
    entries are already removed."""
    w = [int(k["alpha_ps"]) + 1 for k in links]
    tl = links.copy()
    tl["src"], tl["dst"] = links["dst"], links["src"]
    root = [members[c % len(members)] for c in range(nc)]          # pre = post = members: I = members (DESIGN.md step R)
    others = [[m for m in members if m != root[c]] for c in range(nc)]
    b = literal_ten(n, tl, [(root[c], others[c]) for c in range(nc)], seed)
    T1 = max(r[5] for r in b)
    red = [(T1 - te, l, c, dst, src, T1 - ts) for (ts, l, c, src, dst, te) in b]
    removed, ready = set(), [0] * nc
    for ts, l, c, src, dst, te in red:
        for t in range(ts, te):
            removed.add((t, l))
        if dst == root[c]:
            ready[c] = max(ready[c], te)
    cp = literal_ten(n, links, [(root[c], others[c]) for c in range(nc)], seed, removed, ready)
    return sorted(red + cp), T1


@pytest.mark.parametrize("i", range(25))
def test_pipelined_allreduce_against_the_literal_ten(i):
    n, triples, members, nc = _allreduce_case(i)
    links = _links(triples)
    pairs = _pairs([(m, c) for c in range(nc) for m in members])
    p = wl.Problem(f"ar{i}", n, links, np.array(members, dtype=np.uint32), nc, pairs, pairs.copy(), 1, i)
    s = oracle.synthesize(*p.args(), relay=BFS, pipeline=True)
    want, T1 = literal_pipelined_allreduce(n, links, members, nc, i)
    assert _as_tuples(s.transfers) == want
    assert s.time_phase1_ps == T1 and s.time_ps == max(r[5] for r in want) and s.mode == 2
    checker.check_schedule(p, s.transfers)             # one collective: link exclusivity and sums across both phases
    seq = oracle.synthesize(*p.args(), relay=BFS)
    assert seq.time_phase1_ps == T1                    # the reduce phase is the same; only the copy phase moves


def test_pipelined_allreduce_hand_example():
    """Path 0 - 1 - 2 (unit links both ways), one chunk, all three reduce, root = node 0 (chunk 0 mod 3).  Reduce: 2 -> 1
    over [0, 1), 1 -> 0 over [1, 2): the root is complete at 2 either way, so the copy phase 0 -> 1 [2, 3), 1 -> 2 [3, 4)
    cannot start earlier: pipelined = sequential = 4.  With a second chunk rooted at node 1 (chunk 1 mod 3) the reduce
    of chunk 1 ends at ... the broadcast from 1 reaches 0 and 2 at timestep 1, reversed it ends at T1 = 2 as well; its copy
    phase 1 -> 0, 1 -> 2 over [2, 3) shares no link with chunk 0's copy 0 -> 1 [2, 3), but chunk 0's second hop 1 -> 2 now
    waits for chunk 1's copy on that link or takes it first: T = 4 in both compositions, and the pipelined records are a
    valid all-reduce."""
    tri = [(0, 1, 1), (1, 0, 1), (1, 2, 1), (2, 1, 1)]
    links = _links(tri)
    for nc in (1, 2):
        pairs = _pairs([(m, c) for c in range(nc) for m in (0, 1, 2)])
        p = wl.Problem("path3_ar", 3, links, np.array([0, 1, 2], dtype=np.uint32), nc, pairs, pairs.copy(), 1, 0)
        a = oracle.synthesize(*p.args(), relay=BFS)
        b = oracle.synthesize(*p.args(), relay=BFS, pipeline=True)
        assert a.time_ps == 4 and b.time_ps == 4 and b.time_phase1_ps == 2
        checker.check_schedule(p, b.transfers)


def test_pipelining_a_staggered_reduce_helps():
    """Two chunks rooted at the two ends of a 4-node path with a slow middle link: the reduce of the chunk whose root
    sits next to the fast links completes well before the whole reduce phase does, and its copy phase starts then."""
    tri = [(0, 1, 1), (1, 0, 1), (1, 2, 3), (2, 1, 3), (2, 3, 1), (3, 2, 1)]
    links = _links(tri)
    members = [0, 1]
    pairs = _pairs([(m, c) for c in range(2) for m in members])
    p = wl.Problem("path4_ar_stagger", 4, links, np.array(members, dtype=np.uint32), 2, pairs, pairs.copy(), 1, 0)
    a = oracle.synthesize(*p.args(), relay=BFS)
    b = oracle.synthesize(*p.args(), relay=BFS, pipeline=True)
    assert b.time_ps <= a.time_ps
    checker.check_schedule(p, b.transfers)


def test_pipeline_flag_leaves_other_collectives_alone():
    for mk in (wl.config1, wl.config3, wl.config4_small):
        p = mk(1)
        a, b = run(p), oracle.synthesize(*p.args(), relay=BFS, pipeline=True)
        assert _as_tuples(a.transfers) == _as_tuples(b.transfers)
