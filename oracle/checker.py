"""Schedule validity checker -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Independent of the synthesizer's logic: it never computes wants, candidates or picks.  It
re-derives only what the paper fixes and checks a schedule (from the oracle or from the
CUDA path) against it:

  V1  every transfer runs on a real link, in the link's direction, for exactly the link's
      alpha-beta time
  V2  no link carries two chunks at once: per-link intervals [t_start, t_end) are pairwise
      disjoint
  V3  causality / store-and-forward: a node sends only what it holds, i.e. its own
      precondition chunk or something that ARRIVED (t_end <= t_start) earlier
  V4  every postcondition is met, with the fully reduced value for reduction chunks
      
  V5  non-group NPUs only relay: they originate nothing
  V6  (copy chunks) a chunk is delivered to a node at most once
  V7  (reduction chunks) no contribution is summed twice

V3/V4/V7 are checked by SIMULATING the schedule as a collective: each (node, chunk) holds
the set of NPUs whose contribution it contains; a send carries the sender's set at t_start;
it is merged at t_end.  This is mode-agnostic (All-Gather, All-to-All(v), Reduce-Scatter,
All-Reduce).
"""
from __future__ import annotations

import numpy as np


class ScheduleInvalid(AssertionError):
    pass


def _fail(msg):
    raise ScheduleInvalid(msg)


def link_costs(links: np.ndarray, chunk_bytes: int) -> np.ndarray:
    a = links["alpha_ps"].astype(object)
    b = links["bytes_per_ps"].astype(object)
    return np.array([int(x) + (chunk_bytes + int(y) - 1) // int(y) for x, y in zip(a, b)], dtype=np.uint64)


def check_structure(problem, tr: np.ndarray) -> dict:
    """V1, V2, canonical order.  Vectorised; fine for millions of records."""
    links = problem.links
    L = len(links)
    if len(tr) == 0:
        return {"max_link_load": 0}
    if tr["link"].max() >= L:
        _fail("link id out of range")
    lk = links[tr["link"]]
    if not (np.array_equal(lk["src"], tr["src"]) and np.array_equal(lk["dst"], tr["dst"])):
        _fail("V1: transfer endpoints do not match its link")
    w = link_costs(links, problem.chunk_bytes)
    if not np.array_equal(tr["t_end_ps"] - tr["t_start_ps"], w[tr["link"]]):
        _fail("V1: transfer duration differs from the link's alpha-beta time")
    if tr["chunk"].max() >= problem.n_chunks:
        _fail("chunk id out of range")
    # canonical order: strictly increasing (t_start, link)
    ts, ln = tr["t_start_ps"], tr["link"].astype(np.uint64)
    ok = (ts[1:] > ts[:-1]) | ((ts[1:] == ts[:-1]) & (ln[1:] > ln[:-1]))
    if not ok.all():
        _fail("records are not in canonical (t_start, link) order / key not unique")
    # V2
    order = np.lexsort((tr["t_start_ps"], tr["link"]))
    s = tr[order]
    same = s["link"][1:] == s["link"][:-1]
    if (same & (s["t_end_ps"][:-1] > s["t_start_ps"][1:])).any():
        _fail("V2: a link carries two chunks at once")
    return {"max_link_load": int(np.bincount(tr["link"], minlength=L).max())}


def check_copy_vectorised(problem, tr: np.ndarray) -> dict:
    """V3, V4, V5, V6 for COPY-mode problems (every chunk has one pre-holder), vectorised."""
    C = problem.n_chunks
    src_of = np.full(C, -1, dtype=np.int64)
    src_of[problem.pre["chunk"]] = problem.pre["npu"]
    if len(problem.pre) != C or (src_of < 0).any():
        _fail("not a copy-mode problem")
    member = np.zeros(problem.n_npus, dtype=bool)
    member[problem.group] = True
    key_d = tr["dst"].astype(np.int64) * C + tr["chunk"].astype(np.int64)
    order = np.argsort(key_d, kind="stable")
    kd, te = key_d[order], tr["t_end_ps"][order]
    if len(kd) > 1 and (kd[1:] == kd[:-1]).any():
        _fail("V6: a chunk is delivered to the same node twice")
    if (tr["dst"].astype(np.int64) == src_of[tr["chunk"]]).any():
        _fail("V6: a chunk is delivered back to its source")
    key_s = tr["src"].astype(np.int64) * C + tr["chunk"].astype(np.int64)
    pos = np.searchsorted(kd, key_s)
    posc = np.minimum(pos, max(len(kd) - 1, 0))
    found = (pos < len(kd)) & (kd[posc] == key_s) if len(kd) else np.zeros(len(tr), bool)
    is_src = tr["src"].astype(np.int64) == src_of[tr["chunk"]]
    if (~found & ~is_src).any():
        _fail("V3: a node sends a chunk it never holds")
    late = found & ~is_src & (te[posc] > tr["t_start_ps"])
    if late.any():
        _fail("V3: a chunk is forwarded before it arrived")
    if (is_src & ~member[tr["src"]]).any():
        _fail("V5: a non-group NPU originates a chunk")
    # V4
    pk = problem.post["npu"].astype(np.int64) * C + problem.post["chunk"].astype(np.int64)
    need = pk[problem.post["npu"].astype(np.int64) != src_of[problem.post["chunk"]]]
    p2 = np.searchsorted(kd, need)
    p2c = np.minimum(p2, max(len(kd) - 1, 0))
    if len(need) and (len(kd) == 0 or ((p2 >= len(kd)) | (kd[p2c] != need)).any()):
        _fail("V4: a postcondition is not met")
    # dead-end relay deliveries: received by a non-destination that never forwards it
    post_keys = np.unique(pk)
    is_dest = np.isin(key_d, post_keys)
    fwd = np.isin(key_d, np.unique(key_s))
    return {"dead_end_deliveries": int((~is_dest & ~fwd).sum())}


def simulate(problem, tr: np.ndarray) -> dict:  # noqa: C901
    """V3, V4, V5, V6/V7 by simulating the schedule as a collective (pure Python; use on
    schedules up to a few hundred thousand transfers)."""
    C = problem.n_chunks
    pre_mask = [0] * C
    state = {}
    for npu, c in zip(problem.pre["npu"].tolist(), problem.pre["chunk"].tolist()):
        pre_mask[c] |= 1 << npu
        state[(npu, c)] = state.get((npu, c), 0) | (1 << npu)
    member = set(problem.group.tolist())
    for (npu, c) in state:
        if npu not in member:
            _fail("V5: a non-group NPU holds a precondition chunk")
    reduction = [bin(m).count("1") > 1 for m in pre_mask]
    sends = sorted(range(len(tr)), key=lambda i: (int(tr["t_start_ps"][i]), int(tr["link"][i])))
    arrivals = sorted(range(len(tr)), key=lambda i: int(tr["t_end_ps"][i]))
    payload = [0] * len(tr)
    chunk = tr["chunk"].tolist(); src = tr["src"].tolist(); dst = tr["dst"].tolist()
    ts = tr["t_start_ps"].tolist(); te = tr["t_end_ps"].tolist()
    ai = 0
    delivered = set()
    sent_partial = set()
    empty_partials = 0

    def land(i):
        c, v, p = chunk[i], dst[i], payload[i]
        old = state.get((v, c), 0)
        if reduction[c]:
            if p != pre_mask[c] and (old & p):
                _fail(f"V7: a contribution to chunk {c} is summed twice at node {v}")
        else:
            if (v, c) in delivered or old:
                _fail(f"V6: chunk {c} delivered twice to node {v}")
            delivered.add((v, c))
        state[(v, c)] = old | p

    for i in sends:
        while ai < len(arrivals) and te[arrivals[ai]] <= ts[i]:
            land(arrivals[ai]); ai += 1
        p = state.get((src[i], chunk[i]), 0)
        if p == 0:
            # Reversal of a dead-end relay delivery (reading Q15): in the broadcast a
            # non-destination relay received the chunk and never forwarded it; reversed, that
            # relay sends an EMPTY partial sum (the identity).  Harmless, counted, and only
            # legal for a node that contributes nothing to this reduction chunk.
            if reduction[chunk[i]] and not (pre_mask[chunk[i]] >> src[i]) & 1 and (src[i], chunk[i]) not in sent_partial:
                empty_partials += 1
                sent_partial.add((src[i], chunk[i]))
            else:
                _fail(f"V3: node {src[i]} sends chunk {chunk[i]} at {ts[i]} before holding it")
        payload[i] = p
        if reduction[chunk[i]] and p != pre_mask[chunk[i]]:
            # a partial sum leaves the node: what it held moves on (it must not send it again)
            state[(src[i], chunk[i])] = 0
            sent_partial.add((src[i], chunk[i]))
    while ai < len(arrivals):
        land(arrivals[ai]); ai += 1
    for npu, c in zip(problem.post["npu"].tolist(), problem.post["chunk"].tolist()):
        if state.get((npu, c), 0) != pre_mask[c]:
            _fail(f"V4: postcondition (npu {npu}, chunk {c}) not met: has "
                  f"{state.get((npu, c), 0):b}, needs {pre_mask[c]:b}")
    return {"empty_partial_sends": empty_partials}


def check_schedule(problem, tr: np.ndarray, simulate_limit: int = 300_000) -> dict:
    """All checks that apply.  Returns a stats dict; raises ScheduleInvalid on a violation."""
    stats = check_structure(problem, tr)
    copy_mode = len(problem.pre) == problem.n_chunks and len(np.unique(problem.pre["chunk"])) == problem.n_chunks
    if copy_mode:
        stats.update(check_copy_vectorised(problem, tr))
    if len(tr) <= simulate_limit:
        stats.update(simulate(problem, tr))
        stats["simulated"] = True
    elif not copy_mode:
        _fail("schedule too large to simulate and not copy-mode")
    stats["time_ps"] = int(tr["t_end_ps"].max()) if len(tr) else 0
    stats["transfers"] = int(len(tr))
    return stats


# ---------------------------------------------------------------------------------------
# bandwidth lower bound on the collective time of a COPY-mode problem on a homogeneous
# network (all links the same cost w): max of ingress, egress and work bounds, in ps.
# ---------------------------------------------------------------------------------------
def lower_bound_homogeneous(problem, hop_dist) -> int:
    """hop_dist(s) -> array of hop distances from s.  Work bound uses sum of (src,dest) hop
    distances for single-destination chunks and (#dests) for multi-destination chunks."""
    w = int(link_costs(problem.links, problem.chunk_bytes)[0])
    n = problem.n_npus
    indeg = np.bincount(problem.links["dst"], minlength=n)
    outdeg = np.bincount(problem.links["src"], minlength=n)
    C = problem.n_chunks
    src_of = np.zeros(C, dtype=np.int64)
    src_of[problem.pre["chunk"]] = problem.pre["npu"]
    need = problem.post[problem.post["npu"] != src_of[problem.post["chunk"]]]
    need_in = np.bincount(need["npu"], minlength=n)
    ndest = np.bincount(need["chunk"], minlength=C)
    has_dest = ndest > 0
    need_out = np.bincount(src_of[has_dest], minlength=n)
    ingress = max((-(-int(a) // int(b)) for a, b in zip(need_in, indeg) if a), default=0)
    egress = max((-(-int(a) // int(b)) for a, b in zip(need_out, outdeg) if a), default=0)
    work = 0
    cache = {}
    single = ndest == 1
    for s in np.unique(src_of[has_dest]):
        cache[int(s)] = hop_dist(int(s))
    ns, nd = src_of[need["chunk"]], need["npu"]
    sel = single[need["chunk"]]
    for s in cache:
        m = sel & (ns == s)
        work += int(cache[s][nd[m]].sum())
    work += int(ndest[~single & has_dest].sum())
    work_rounds = -(-work // len(problem.links))
    return max(ingress, egress, work_rounds) * w
