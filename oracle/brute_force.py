"""Brute-force optimal collective time on tiny homogeneous instances -- TEST INFRASTRUCTURE.

Pins the oracle's "near-optimal" behaviour: on a network whose links all
have the same cost w, time advances in synchronous rounds of length w, and the optimum is the
minimum number of rounds R such that, sending at most one chunk per link per round
 and only chunks the sender held at the start of the round,
every postcondition holds.  Breadth-first search over holdings states.  Exponential: use only
for N <= 5 nodes and a handful of chunks.

Monotonicity used for pruning: a holdings state that is a component-wise superset of another
is never worse, so per destination only the maximal reachable holding sets are kept, and a
frontier state dominated by another frontier state is dropped.
"""
from __future__ import annotations

from itertools import product


def _maximal(sets):
    sets = sorted(set(sets), key=lambda s: -bin(s).count("1"))
    keep = []
    for s in sets:
        if not any((s | k) == k for k in keep):
            keep.append(s)
    return keep


def optimal_rounds(n_nodes, links, have0, need, max_rounds=12):
    """links: list of (src, dst); have0[v], need[v]: chunk bitmasks.  Returns min rounds."""
    inl = [[] for _ in range(n_nodes)]
    for (s, d) in links:
        inl[d].append(s)

    def done(state):
        return all((state[v] & need[v]) == need[v] for v in range(n_nodes))

    start = tuple(have0)
    if done(start):
        return 0
    frontier = [start]
    for rnd in range(1, max_rounds + 1):
        nxt = set()
        for st in frontier:
            per_node = []
            for v in range(n_nodes):
                choice_sets = []
                for u in inl[v]:
                    avail = st[u] & ~st[v]
                    bits = [1 << b for b in range(avail.bit_length()) if (avail >> b) & 1]
                    choice_sets.append(bits if bits else [0])
                opts = set()
                for combo in product(*choice_sets):
                    m = st[v]
                    for b in combo:
                        m |= b
                    opts.add(m)
                per_node.append(_maximal(opts))
            for combo in product(*per_node):
                if done(combo):
                    return rnd
                nxt.add(combo)
        # drop dominated frontier states
        lst = sorted(nxt, key=lambda s: -sum(bin(x).count("1") for x in s))
        keep = []
        for s in lst:
            if not any(all((s[v] | k[v]) == k[v] for v in range(n_nodes)) for k in keep):
                keep.append(s)
        frontier = keep
        if not frontier:
            break
    raise RuntimeError("no solution within max_rounds")


def optimal_rounds_problem(problem, max_rounds=12):
    """Optimal rounds for a COPY-mode workloads.Problem on a homogeneous network."""
    n = problem.n_npus
    have0 = [0] * n
    need = [0] * n
    for npu, c in zip(problem.pre["npu"].tolist(), problem.pre["chunk"].tolist()):
        have0[npu] |= 1 << c
    for npu, c in zip(problem.post["npu"].tolist(), problem.post["chunk"].tolist()):
        need[npu] |= 1 << c
    links = list(zip(problem.links["src"].tolist(), problem.links["dst"].tolist()))
    return optimal_rounds(n, links, have0, need, max_rounds)
