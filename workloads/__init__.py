"""Seeded synthetic input generators shared by the tests, the oracle legs and the CUDA legs.

This module holds NONE of the method's arithmetic (no link costs, no distances, no wants, no
matching): it only emits problem statements -- topology link lists, process groups and
pre/postconditions -- in the shape of BASELINE.json's five configs (recipe in DESIGN.md,
"Input recipe").  The only random draws are the harness-only ones (Philox domain tags 2 =
group draw, 3 = Zipf count draw); the Philox below is a numpy-vectorised generator of its
own, separate from the oracle's (C++) and the CUDA path's (device) implementations.

The paper evaluates on synthetic topologies (2D Mesh, 3D Hypercube/torus, 2D Switch;
PAPER.md:378, :394) and uses no public dataset, so these generators ARE the workloads.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

LINK_DT = np.dtype([("src", "<u4"), ("dst", "<u4"), ("alpha_ps", "<u8"), ("bytes_per_ps", "<u8")])
PAIR_DT = np.dtype([("npu", "<u4"), ("chunk", "<u4")])


@dataclass
class Problem:
    """One problem statement at the boundary of include/pccl.h (all host numpy arrays)."""
    name: str
    n_npus: int                     # all nodes: NPUs and switch nodes
    links: np.ndarray               # LINK_DT, link id = index
    group: np.ndarray               # uint32, union of the process groups' members
    n_chunks: int
    pre: np.ndarray                 # PAIR_DT "npu holds chunk" before
    post: np.ndarray                # PAIR_DT "npu holds chunk" after
    chunk_bytes: int
    seed: int
    meta: dict = field(default_factory=dict)

    def args(self):
        return (self.n_npus, self.links, self.group, self.n_chunks, self.pre, self.post,
                self.chunk_bytes, self.seed)


# ---------------------------------------------------------------------------------------
# harness-only counter-based generator (numpy, vectorised over counters)
# ---------------------------------------------------------------------------------------
def philox_first_word(c0, c1, c2, c3, seed: int) -> np.ndarray:
    """First output word of Philox4x32-10 for arrays of counters; key = (seed lo, seed hi)."""
    c0, c1, c2, c3 = np.broadcast_arrays(*(np.asarray(x, dtype=np.uint64) for x in (c0, c1, c2, c3)))
    c0, c1, c2, c3 = (x.copy() for x in (c0, c1, c2, c3))
    m32 = np.uint64(0xFFFFFFFF)
    k0 = np.uint64(seed & 0xFFFFFFFF)
    k1 = np.uint64((seed >> 32) & 0xFFFFFFFF)
    MA, MB = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
    WA, WB = np.uint64(0x9E3779B9), np.uint64(0xBB67AE85)
    s32 = np.uint64(32)
    for _ in range(10):
        pa = MA * c0
        pb = MB * c2
        n0 = (pb >> s32) ^ c1 ^ k0
        n1 = pb & m32
        n2 = (pa >> s32) ^ c3 ^ k1
        n3 = pa & m32
        c0, c1, c2, c3 = n0, n1, n2, n3
        k0 = (k0 + WA) & m32
        k1 = (k1 + WB) & m32
    return c0.astype(np.uint32)


# ---------------------------------------------------------------------------------------
# topologies
# ---------------------------------------------------------------------------------------
def grid_links(dims, wrap: bool, alpha_ps: int = 500_000, bytes_per_ps: int = 50) -> np.ndarray:
    """k-D torus (wrap) or mesh.  node id = x + X*(y + Y*z); links emitted for node u
    ascending, dimension 0..K-1, direction +1 then -1; link id = emission index."""
    dims = [int(d) for d in dims]
    n = int(np.prod(dims))
    strides = [int(np.prod(dims[:k])) for k in range(len(dims))]
    out = []
    for u in range(n):
        coord = [(u // strides[k]) % dims[k] for k in range(len(dims))]
        for k in range(len(dims)):
            for step in (+1, -1):
                x = coord[k] + step
                if wrap:
                    x %= dims[k]
                elif x < 0 or x >= dims[k]:
                    continue
                v = u + (x - coord[k]) * strides[k]
                if v == u:
                    continue          # size-1 dimension
                out.append((u, v, alpha_ps, bytes_per_ps))
    return np.array(out, dtype=LINK_DT)


def ring_links(n: int, bidirectional: bool, alpha_ps: int = 500_000, bytes_per_ps: int = 50) -> np.ndarray:
    """Unidirectional ring: link i = i -> (i+1) mod n.  Bidirectional: then link n+i = i -> (i-1) mod n."""
    out = [(i, (i + 1) % n, alpha_ps, bytes_per_ps) for i in range(n)]
    if bidirectional:
        out += [(i, (i - 1) % n, alpha_ps, bytes_per_ps) for i in range(n)]
    return np.array(out, dtype=LINK_DT)


def full_mesh_links(n: int, alpha_ps: int = 500_000, bytes_per_ps: int = 50) -> np.ndarray:
    return np.array([(a, b, alpha_ps, bytes_per_ps) for a in range(n) for b in range(n) if a != b],
                    dtype=LINK_DT)


def pods_links(n_pods: int = 8, pod: int = 8) -> np.ndarray:
    """2-level topology of config 3 (reading Q16): nodes 0..n_pods*pod-1 are NPUs, then one
    switch node per pod.  Intra-pod full mesh (200000 ps, 450 B/ps), uplinks, downlinks and the
    switch full mesh (500000 ps, 50 B/ps), in that order."""
    sw = n_pods * pod
    out = []
    for p in range(n_pods):
        for a in range(pod):
            for b in range(pod):
                if a != b:
                    out.append((pod * p + a, pod * p + b, 200_000, 450))
    for p in range(n_pods):
        for a in range(pod):
            out.append((pod * p + a, sw + p, 500_000, 50))
    for p in range(n_pods):
        for a in range(pod):
            out.append((sw + p, pod * p + a, 500_000, 50))
    for p in range(n_pods):
        for q in range(n_pods):
            if p != q:
                out.append((sw + p, sw + q, 500_000, 50))
    return np.array(out, dtype=LINK_DT)


def draw_group(n_npus: int, size: int, seed: int) -> np.ndarray:
    """The `size` nodes with the smallest (Philox(ctr=(v,0,0,2), key)[0], v), sorted ascending."""
    v = np.arange(n_npus, dtype=np.uint64)
    score = philox_first_word(v, 0, 0, 2, seed).astype(np.uint64)
    order = np.lexsort((v, score))
    return np.sort(order[:size]).astype(np.uint32)


def _pairs(npus, chunks) -> np.ndarray:
    a = np.zeros(len(npus), dtype=PAIR_DT)
    a["npu"] = npus
    a["chunk"] = chunks
    return a


# ---------------------------------------------------------------------------------------
# collectives as pre/postconditions
# ---------------------------------------------------------------------------------------
def all_gather(members, chunks_per_npu: int = 1):
    """chunk id = i*chunks_per_npu + j for the i-th member; pre {member i}, post all members."""
    members = np.asarray(members, dtype=np.uint32)
    g, k = len(members), chunks_per_npu
    n_chunks = g * k
    pre = _pairs(np.repeat(members, k), np.arange(n_chunks))
    post = _pairs(np.tile(members, n_chunks), np.repeat(np.arange(n_chunks), g))
    return n_chunks, pre, post


def all_to_all(members, counts=None):
    """for s in members asc, d in members asc, d != s: counts[s_idx, d_idx] chunks (default 1)
    with pre {s}, post {d}."""
    members = np.asarray(members, dtype=np.uint32)
    g = len(members)
    si, di = np.meshgrid(np.arange(g), np.arange(g), indexing="ij")
    keep = si != di
    si, di = si[keep], di[keep]
    if counts is None:
        cnt = np.ones(len(si), dtype=np.int64)
    else:
        cnt = np.asarray(counts, dtype=np.int64)[si, di]
    s_rep = np.repeat(members[si], cnt)
    d_rep = np.repeat(members[di], cnt)
    n_chunks = int(cnt.sum())
    ids = np.arange(n_chunks)
    return n_chunks, _pairs(s_rep, ids), _pairs(d_rep, ids)


def all_reduce(members, n_chunks: int):
    """every chunk pre = post = members."""
    members = np.asarray(members, dtype=np.uint32)
    g = len(members)
    both = _pairs(np.tile(members, n_chunks), np.repeat(np.arange(n_chunks), g))
    return n_chunks, both, both.copy()


def reduce_scatter_groups(groups):
    """concurrent groups; chunk id = running index; chunk (g, i): pre = group g, post = {i-th member}."""
    pre_n, pre_c, post_n, post_c = [], [], [], []
    cid = 0
    for grp in groups:
        for i in range(len(grp)):
            pre_n += list(grp)
            pre_c += [cid] * len(grp)
            post_n.append(grp[i])
            post_c.append(cid)
            cid += 1
    return cid, _pairs(pre_n, pre_c), _pairs(post_n, post_c)


ZIPF_THR = np.array([1786133164, 2563592779, 3041527221, 3379936174, 3638846773, 3846879822,
                     4019780297, 4167081349, 2 ** 32], dtype=np.uint64)
"""cumulative (k+1)^-1.2 / sum for k = 0..8, scaled by 2^32: Zipf(s = 1.2) on [0, 8]."""


def zipf_counts(members, seed: int) -> np.ndarray:
    """counts[s_idx, d_idx] = first k with Philox(ctr=(s,d,0,3))[0] < ZIPF_THR[k]."""
    members = np.asarray(members, dtype=np.uint64)
    s, d = np.meshgrid(members, members, indexing="ij")
    u = philox_first_word(s, d, 0, 3, seed).astype(np.uint64)
    return np.searchsorted(ZIPF_THR, u, side="right").astype(np.int64)


# ---------------------------------------------------------------------------------------
# BASELINE.json configs (1-based) and reduced variants
# ---------------------------------------------------------------------------------------
def config1(seed: int = 0) -> Problem:
    links = grid_links((4, 4), wrap=True)
    members = np.arange(16, dtype=np.uint32)
    nc, pre, post = all_gather(members, 1)
    return Problem("cfg1_torus4x4_allgather", 16, links, members, nc, pre, post, 1 << 20, seed)


def config2(seed: int = 0, dims=(8, 8), group_size: int = 16, chunks_per_npu: int = 4,
            chunk_bytes: int = 256 << 10) -> Problem:
    links = grid_links(dims, wrap=False)
    n = int(np.prod(dims))
    members = draw_group(n, group_size, seed)
    nc, pre, post = all_reduce(members, group_size * chunks_per_npu)
    return Problem(f"cfg2_mesh{dims[0]}x{dims[1]}_allreduce_g{group_size}", n, links, members, nc,
                   pre, post, chunk_bytes, seed)


def config3(seed: int = 0, n_pods: int = 8, pod: int = 8) -> Problem:
    links = pods_links(n_pods, pod)
    groups = [[pod * g + a for a in range(pod)] for g in range(n_pods)]
    groups += [[pod * p + j for p in range(n_pods)] for j in range(pod)]
    nc, pre, post = reduce_scatter_groups(groups)
    members = np.arange(n_pods * pod, dtype=np.uint32)
    return Problem(f"cfg3_pods{n_pods}x{pod}_reducescatter", n_pods * pod + n_pods, links, members,
                   nc, pre, post, 1 << 20, seed, meta={"groups": groups})


def config4(seed: int = 0, dims=(8, 8, 8), chunk_bytes: int = 64 << 10) -> Problem:
    links = grid_links(dims, wrap=True)
    n = int(np.prod(dims))
    members = np.arange(n, dtype=np.uint32)
    nc, pre, post = all_to_all(members)
    return Problem("cfg4_torus" + "x".join(map(str, dims)) + "_alltoall", n, links, members, nc,
                   pre, post, chunk_bytes, seed)


def config5(seed: int = 0, dims=(32, 32), group_size: int = 512, chunk_bytes: int = 32 << 10) -> Problem:
    links = grid_links(dims, wrap=True)
    n = int(np.prod(dims))
    members = draw_group(n, group_size, seed)
    counts = zipf_counts(members, seed)
    nc, pre, post = all_to_all(members, counts)
    return Problem("cfg5_torus" + "x".join(map(str, dims)) + f"_alltoallv_g{group_size}", n, links,
                   members, nc, pre, post, chunk_bytes, seed)


def config4_small(seed: int = 0) -> Problem:
    return config4(seed, dims=(4, 4, 4))


def config5_small(seed: int = 0) -> Problem:
    return config5(seed, dims=(16, 16), group_size=128)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


# ---------------------------------------------------------------------------------------
# small structured cases for pins
# ---------------------------------------------------------------------------------------
def ring_all_gather(n: int, bidirectional: bool, seed: int = 0, chunks_per_npu: int = 1,
                    chunk_bytes: int = 1 << 20) -> Problem:
    links = ring_links(n, bidirectional)
    members = np.arange(n, dtype=np.uint32)
    nc, pre, post = all_gather(members, chunks_per_npu)
    return Problem(f"ring{n}_{'bi' if bidirectional else 'uni'}_allgather", n, links, members, nc,
                   pre, post, chunk_bytes, seed)


def full_mesh_problem(n: int, kind: str, seed: int = 0, chunk_bytes: int = 1 << 20) -> Problem:
    links = full_mesh_links(n)
    members = np.arange(n, dtype=np.uint32)
    nc, pre, post = all_gather(members, 1) if kind == "allgather" else all_to_all(members)
    return Problem(f"fullmesh{n}_{kind}", n, links, members, nc, pre, post, chunk_bytes, seed)


def path_point_to_point(n: int, seed: int = 0, chunk_bytes: int = 1 << 20) -> Problem:
    """bidirectional path 0-1-...-(n-1); one chunk from NPU 0 to NPU n-1; group = {0, n-1}."""
    links = grid_links((n,), wrap=False)
    members = np.array([0, n - 1], dtype=np.uint32)
    return Problem(f"path{n}_p2p", n, links, members, 1, _pairs([0], [0]), _pairs([n - 1], [0]),
                   chunk_bytes, seed)


def two_groups_mesh3x3(seed: int = 0, chunk_bytes: int = 1 << 20) -> Problem:
    """Scenario of PAPER.md Fig. 15 / section 6.4: 3x3 mesh, group 1 = NPUs 0-2 running
    All-to-Allv (NPU 0 sends twice as much as NPUs 1-2), group 2 = NPUs 6-8 running
    All-Gather with two chunks per NPU; NPUs 3-5 belong to no group and may only relay.
    Only the scenario is from the paper; the figure's schedule is not in the text."""
    links = grid_links((3, 3), wrap=False)
    g1 = np.array([0, 1, 2], dtype=np.uint32)
    counts = np.array([[0, 2, 2], [1, 0, 1], [1, 1, 0]])
    n1, pre1, post1 = all_to_all(g1, counts)
    g2 = np.array([6, 7, 8], dtype=np.uint32)
    n2, pre2, post2 = all_gather(g2, 2)
    pre2["chunk"] += n1
    post2["chunk"] += n1
    members = np.concatenate([g1, g2])
    return Problem("mesh3x3_two_groups", 9, links, members, n1 + n2, np.concatenate([pre1, pre2]),
                   np.concatenate([post1, post2]), chunk_bytes, seed,
                   meta={"groups": [list(g1), list(g2)]})
