"""Pin of the oracle's step E -- candidates, pick policy, conflict order, link occupancy -- re-derived event by event from
the emitted schedule with an independent Philox (workloads.philox_first_word, numpy) and scipy distances.  No GPU.

Given only the wants relation of step C (pinned on its own in tests/test_oracle_pins.py) and the schedule, at every event
time and for every node the free in-links are served in ascending link id; link l's candidates are the chunks its source
holds by t that the node still wants; the chunk it must carry is
    default policy (reading Q5):   the k-th candidate in ascending chunk id, k = (Philox(t, l) * n) >> 32
    c.dist policy (reading Q27):   the same draw over the candidates with the largest c.dist = max over dests of the
                                   alpha-beta shortest path from the chunk's source (Alg. 3 lines 1-6)
and a link without candidates must stay idle.  A wrong tie order, a draw keyed on the wrong counter, a pick among all
candidates instead of the farthest ones, or a claim that is not seen by the next in-link all fail here.
"""
import numpy as np
import pytest

import oracle
import workloads as wl
from oracle import checker


def _conds(p):
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


def _cdist(p, src, off, dests):
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import dijkstra
    w = checker.link_costs(p.links, p.chunk_bytes)
    best = {}
    for l, c in zip(p.links, w):
        k = (int(l["src"]), int(l["dst"]))
        best[k] = min(best.get(k, 1 << 62), int(c))
    rows, cols = zip(*best.keys())
    g = csr_matrix((np.array(list(best.values()), dtype=np.float64), (rows, cols)), shape=(p.n_npus, p.n_npus))
    D = dijkstra(g, directed=True)
    return [max((int(D[src[c]][d]) for d in dests[int(off[c]):int(off[c + 1])]), default=0) for c in range(p.n_chunks)]


def rederive(p, tr, by_dist):
    src, off, dests = _conds(p)
    want = oracle.wants(p.n_npus, p.links, p.n_chunks, src, off, dests, p.chunk_bytes, p.seed)
    wanted = [set() for _ in range(p.n_npus)]
    for v, c in zip(want["npu"].tolist(), want["chunk"].tolist()):
        wanted[v].add(c)
    cd = _cdist(p, src, off, dests) if by_dist else None
    n, L = p.n_npus, len(p.links)
    inl = [[] for _ in range(n)]
    for l in range(L):
        inl[int(p.links[l]["dst"])].append(l)
    starts = {(int(r["t_start_ps"]), int(r["link"])): int(r["chunk"]) for r in tr}
    have = [set() for _ in range(n)]
    for c, s in enumerate(src.tolist()):
        have[s].add(c)
    arrivals = sorted((int(r["t_end_ps"]), int(r["dst"]), int(r["chunk"])) for r in tr)
    busy_until = [0] * L
    ai = 0
    seen = 0
    for t in sorted({0} | {int(x) for x in tr["t_end_ps"]}):
        while ai < len(arrivals) and arrivals[ai][0] <= t:
            have[arrivals[ai][1]].add(arrivals[ai][2]); ai += 1
        for v in range(n):
            for l in inl[v]:
                if busy_until[l] > t:
                    assert (t, l) not in starts
                    continue
                cand = sorted(have[int(p.links[l]["src"])] & wanted[v])
                got = starts.get((t, l))
                if not cand:
                    assert got is None, f"{p.name}: t={t} link {l} carries {got} without a candidate"
                    continue
                if by_dist:
                    far = max(cd[c] for c in cand)
                    cand = [c for c in cand if cd[c] == far]
                r = int(wl.philox_first_word(t & 0xFFFFFFFF, t >> 32, l, 0, p.seed))
                expect = cand[(r * len(cand)) >> 32]
                assert got == expect, f"{p.name}: t={t} link {l}: expected chunk {expect} of {len(cand)} candidates, schedule has {got}"
                wanted[v].discard(got)
                w = int(checker.link_costs(p.links[l:l + 1], p.chunk_bytes)[0])
                busy_until[l] = t + w
                seen += 1
    assert seen == len(tr)
    assert all(not s for s in wanted), "wants left over"


def _hetero_mesh(seed):
    rng = np.random.default_rng(300 + seed)
    links = wl.grid_links((4, 4), wrap=False).copy()
    links["alpha_ps"] = rng.integers(100, 900, len(links))
    links["bytes_per_ps"] = rng.integers(1, 9, len(links))
    m = np.sort(rng.choice(16, 9, replace=False)).astype(np.uint32)
    nc, pre, post = wl.all_to_all(m, rng.integers(0, 3, (9, 9)))
    return wl.Problem("mesh4x4_hetero_a2av", 16, links, m, nc, pre, post, 3000, seed)


CASES = [wl.config1, wl.config4_small, wl.two_groups_mesh3x3, _hetero_mesh,
         lambda s: wl.ring_all_gather(7, True, s, chunks_per_npu=3), lambda s: wl.full_mesh_problem(6, "allgather", seed=s)]


@pytest.mark.parametrize("maker", CASES, ids=lambda m: getattr(m, "__name__", "case"))
@pytest.mark.parametrize("seed", [0, 1])
@pytest.mark.parametrize("by_dist", [False, True], ids=["uniform_pick", "cdist_pick"])
def test_step_e_rederived_from_the_schedule(maker, seed, by_dist):
    p = maker(seed)
    s = oracle.synthesize(*p.args(), relay=oracle.RELAY_THIN_DIST_PICK if by_dist else oracle.RELAY_THIN)
    rederive(p, s.transfers, by_dist)
    checker.check_schedule(p, s.transfers)


def test_the_two_policies_differ_where_distances_differ_and_agree_where_they_do_not():
    p = wl.config4_small(0)                 # hop distances 1..6: the farthest candidate is usually a strict subset
    a = oracle.synthesize(*p.args())
    b = oracle.synthesize(*p.args(), relay=oracle.RELAY_THIN_DIST_PICK)
    assert len(a.transfers) == len(b.transfers) and not np.array_equal(a.transfers["chunk"], b.transfers["chunk"])
    q = wl.full_mesh_problem(6, "alltoall", seed=1)     # every chunk one hop: c.dist is the same for all, same schedule
    a, b = oracle.synthesize(*q.args()), oracle.synthesize(*q.args(), relay=oracle.RELAY_THIN_DIST_PICK)
    for f in a.transfers.dtype.names:
        assert np.array_equal(a.transfers[f], b.transfers[f])


def test_dist_pick_applies_to_reductions_through_the_reversed_broadcast():
    for mk in (wl.config2, wl.config3):
        p = mk(1)
        s = oracle.synthesize(*p.args(), relay=oracle.RELAY_THIN_DIST_PICK)
        checker.check_schedule(p, s.transfers)
