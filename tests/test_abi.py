"""No-GPU tests of the boundary: libpccl.so builds, loads and exports every symbol that
include/pccl.h declares; the host-side logic (validation, step R normalisation, in-link
tables) behaves as documented; compute entry points fail loudly without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pk():
    import paper_2606_07019_b200 as pk
    return pk


def header_symbols():
    src = open(os.path.join(ROOT, "include", "pccl.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pccl_[a-z0-9_]+)\s*\(", src)) - {"pccl_alloc_fn", "pccl_free_fn"})


def test_library_exports_every_declared_symbol(pk):
    names = header_symbols()
    assert len(names) >= 25
    raw = C.CDLL(pk.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"libpccl.so lacks {n}"
    assert set(names) == set(pk.SIGNATURES), "binding and header disagree on the symbol list"
    assert pk.pccl_version() == 100
    assert pk.pccl_strerror(0) == b"ok" and b"unreachable" in pk.pccl_strerror(-3)


def test_binding_is_marshalling_only():
    """the package holds no arithmetic of the method and never touches the oracle."""
    for fn in ("__init__.py", "_build.py"):
        src = open(os.path.join(ROOT, "paper_2606_07019_b200", fn)).read()
        assert "import oracle" not in src and "from oracle" not in src
        assert "philox" not in src.replace("device_philox", "").replace("pccl_device_philox", "").lower()


def test_struct_layouts(pk):
    assert pk.LINK_DT.itemsize == 24 and pk.PAIR_DT.itemsize == 8 and pk.TRANSFER_DT.itemsize == 32
    assert C.sizeof(pk.pccl_stats_t) == 8 * 8 + 3 * 4 + 2 * 4 + 4   # tail padding to 8


def test_topology_validation(pk):
    ok = np.array([(0, 1, 5, 1), (1, 0, 5, 1)], dtype=wl.LINK_DT)
    t = pk.Topology(2, ok)
    assert (t.n_npus, t.n_links) == (2, 2)
    assert pk.pccl_topology_n_npus(t.handle) == 2 and pk.pccl_topology_n_links(t.handle) == 2
    for bad in ([(0, 2, 5, 1)], [(2, 0, 5, 1)], [(1, 1, 5, 1)], [(0, 1, 5, 0)]):
        with pytest.raises(pk.PcclError) as e:
            pk.Topology(2, np.array(bad, dtype=wl.LINK_DT))
        assert e.value.code == pk.PCCL_ERR_INVALID
    h = C.c_void_p()
    assert pk.pccl_topology_create(2, None, 1, C.byref(h)) == pk.PCCL_ERR_INVALID
    assert pk.pccl_topology_create(2, None, 0, None) == pk.PCCL_ERR_INVALID
    assert not h.value                                          # out untouched on error
    pk.pccl_topology_destroy(None)                              # NULL accepted


def _problem(pk, p):
    topo = pk.Topology(p.n_npus, p.links)
    return pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)


def test_step_R_copy_mode(pk):
    p = wl.config1()
    pr = _problem(pk, p)
    assert pr.mode == 0 and pk.pccl_problem_n_chunks(pr.handle) == 16
    for c in (0, 7, 15):
        src, d = pr.condition(0, c)
        assert src == c and d.tolist() == [v for v in range(16) if v != c]
    with pytest.raises(pk.PcclError):
        pr.condition(1, 0)
    with pytest.raises(pk.PcclError):
        pr.condition(0, 16)


def _conditions(pk, p, pre, post):
    pr = pk.Problem(pk.Topology(p.n_npus, p.links), p.group, p.n_chunks, pre, post, p.chunk_bytes)
    out = []
    for c in range(p.n_chunks):
        src, d = pr.condition(0, c)
        out.append((src, tuple(d.tolist())))
    return pr.mode, out


@pytest.mark.parametrize("maker", [wl.config1, wl.config4_small, wl.config5_small,
                                   lambda s=0: wl.full_mesh_problem(9, "alltoall", seed=s),
                                   lambda s=0: wl.ring_all_gather(7, True, s, chunks_per_npu=3)])
def test_step_R_one_pass_and_general_normaliser_agree(pk, maker):
    """Chunk-ordered COPY input takes the one-pass normaliser; any other arrangement of the same pairs (shuffled,
    dests descending, duplicated pairs) takes the general grouping path.  Both must give the same conditions --
    and those are the definition: source = the one pre-holder, dests = post(c) minus the source, ascending."""
    p = maker(0)
    rng = np.random.default_rng(7)
    mode, ref = _conditions(pk, p, p.pre, p.post)
    assert mode == 0
    pre_of = {int(c): int(n) for n, c in zip(p.pre["npu"], p.pre["chunk"])}
    post_of = {}
    for n, c in zip(p.post["npu"], p.post["chunk"]):
        post_of.setdefault(int(c), set()).add(int(n))
    assert ref == [(pre_of[c], tuple(sorted(post_of[c] - {pre_of[c]}))) for c in range(p.n_chunks)]
    variants = [(rng.permutation(p.pre), rng.permutation(p.post)),
                (p.pre, p.post[::-1].copy()),
                (np.concatenate([p.pre, p.pre[:3]]), np.concatenate([p.post, p.post[-5:]])),
                (p.pre[::-1].copy(), p.post)]
    for pre, post in variants:
        assert _conditions(pk, p, pre, post) == (0, ref)


def test_step_R_reduce_mode_and_duplicates(pk):
    p = wl.config3()
    pr = _problem(pk, p)
    assert pr.mode == 1
    groups = p.meta["groups"]
    for g, grp in enumerate(groups):
        for i in (0, 5):
            root, d = pr.condition(0, 8 * g + i)
            assert root == grp[i] and d.tolist() == sorted(set(grp) - {grp[i]})
    # duplicated pairs are ignored
    dup = wl.Problem("dup", p.n_npus, p.links, p.group, p.n_chunks, np.concatenate([p.pre, p.pre[:50]]),
                     np.concatenate([p.post, p.post]), p.chunk_bytes, 0)
    pr2 = _problem(pk, dup)
    assert pr2.mode == 1
    assert pr2.condition(0, 9)[1].tolist() == pr.condition(0, 9)[1].tolist()


def test_step_R_all_reduce_roots(pk):
    p = wl.config2()
    pr = _problem(pk, p)
    assert pr.mode == 2
    G = sorted(int(x) for x in p.group)
    for c in (0, 1, 17, 63):
        root, d = pr.condition(0, c)
        root2, d2 = pr.condition(1, c)
        assert root == root2 == G[c % 16]                      # root(c) = I[c mod |I|], I = pre & post sorted
        assert d.tolist() == d2.tolist() == [v for v in G if v != root]
    # disjoint pre / post: I falls back to sorted(post)
    links = wl.full_mesh_links(4)
    pre = np.array([(0, 0), (1, 0), (0, 1), (1, 1)], dtype=wl.PAIR_DT)
    post = np.array([(2, 0), (3, 0), (2, 1), (3, 1)], dtype=wl.PAIR_DT)
    pr = pk.Problem(pk.Topology(4, links), np.arange(4, dtype=np.uint32), 2, pre, post, 64)
    assert pr.mode == 2
    assert pr.condition(0, 0) [0] == 2 and pr.condition(0, 1)[0] == 3
    assert pr.condition(0, 0)[1].tolist() == [0, 1] and pr.condition(1, 0)[1].tolist() == [3]


def test_problem_validation_errors(pk):
    links = wl.ring_links(4, True)
    topo = pk.Topology(4, links)
    g = np.arange(4, dtype=np.uint32)
    pre = np.array([(0, 0)], dtype=wl.PAIR_DT)
    post = np.array([(1, 0)], dtype=wl.PAIR_DT)

    def code(*a):
        with pytest.raises(pk.PcclError) as e:
            pk.Problem(topo, *a)
        return e.value.code
    assert pk.Problem(topo, g, 1, pre, post, 64).mode == 0
    assert code(g, 1, pre, post, 0) == pk.PCCL_ERR_INVALID                          # chunk_bytes == 0
    assert code(np.array([0, 0, 1], np.uint32), 1, pre, post, 64) == pk.PCCL_ERR_INVALID   # duplicate member
    assert code(np.array([0, 9], np.uint32), 1, pre, post, 64) == pk.PCCL_ERR_INVALID      # member out of range
    assert code(np.array([0], np.uint32), 1, pre, post, 64) == pk.PCCL_ERR_INVALID         # pair outside the group
    assert code(g, 1, np.array([(0, 1)], wl.PAIR_DT), post, 64) == pk.PCCL_ERR_INVALID     # chunk id >= n_chunks
    assert code(g, 2, pre, post, 64) == pk.PCCL_ERR_INVALID                          # chunk 1 has no holder
    assert code(g, 1, pre, np.zeros(0, wl.PAIR_DT), 64) == pk.PCCL_ERR_INVALID      # no post-holder
    # mixed copy / reduction chunks
    pre2 = np.array([(0, 0), (0, 1), (1, 1)], dtype=wl.PAIR_DT)
    post2 = np.array([(1, 0), (2, 1)], dtype=wl.PAIR_DT)
    assert code(g, 2, pre2, post2, 64) == pk.PCCL_ERR_UNSUPPORTED
    # pre.n_chunks != post.n_chunks at the C level
    pc = pk.pccl_condition_t(1, 1, pre.ctypes.data)
    qc = pk.pccl_condition_t(2, 1, post.ctypes.data)
    h = C.c_void_p()
    assert pk.pccl_problem_create(topo.handle, g.ctypes.data, 4, C.byref(pc), C.byref(qc), 64, C.byref(h)) == pk.PCCL_ERR_INVALID
    assert pk.pccl_problem_create(None, g.ctypes.data, 4, C.byref(pc), C.byref(pc), 64, C.byref(h)) == pk.PCCL_ERR_INVALID
    assert not h.value


def test_compute_fails_loudly_without_a_device(pk):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    p = wl.config1()
    with pytest.raises(pk.PcclError) as e:
        pk.synthesize(*p.args())
    assert e.value.code == pk.PCCL_ERR_CUDA                     # no CPU fallback
    with pytest.raises(RuntimeError):
        pk.use_torch()
    with pytest.raises(pk.PcclError):
        pk.device_philox([[0, 0, 0, 0]], [0, 0])


def test_flag_constants_match_the_header(pk):
    src = open(os.path.join(ROOT, "include", "pccl.h")).read()
    flags = dict(re.findall(r"#define (PCCL_FLAG_[A-Z_]+) (\d+)u", src))
    assert len(flags) == 15
    for name, val in flags.items():
        assert getattr(pk, name) == int(val), name
    assert int(re.search(r"#define PCCL_TRACE_SLOTS (\d+)", src).group(1)) == pk.PCCL_TRACE_SLOTS


def test_static_entry_point_checks_its_arguments_before_touching_the_device(pk):
    """pccl_candidate_totals_static (the entry point that allocates nothing): argument and size checks come first, so
    they can be exercised without a GPU; with valid arguments and no device the call fails loudly."""
    import torch
    fake = 0x1000                                                # non-null, 16-byte aligned; never dereferenced here
    call = lambda **k: pk.pccl_candidate_totals_static(k.get("have", fake), fake, k.get("n", 4), k.get("links", 4),  # noqa: E731
                                                       k.get("words", 2), fake, fake, fake, k.get("totals", fake), None)
    assert call(n=0) == pk.PCCL_OK and call(links=0) == pk.PCCL_OK
    assert call(totals=None) == pk.PCCL_ERR_INVALID and call(words=3) == pk.PCCL_ERR_INVALID
    assert call(words=0) == pk.PCCL_ERR_INVALID and call(have=fake + 8) == pk.PCCL_ERR_INVALID
    src = open(os.path.join(ROOT, "include", "pccl.h")).read()
    assert int(re.search(r"#define PCCL_STATIC_SCRATCH_BYTES \((\d+)u << (\d+)\)", src).group(1)) << 20 == pk.PCCL_STATIC_SCRATCH_BYTES
    per_link = 8                                                 # 2 words per row: one segment count + one row sum
    assert call(links=pk.PCCL_STATIC_SCRATCH_BYTES // per_link + 1) == pk.PCCL_ERR_TOO_LARGE
    assert b"PCCL_STATIC_SCRATCH_BYTES" in pk.pccl_strerror(pk.PCCL_ERR_TOO_LARGE)
    if not torch.cuda.is_available():
        assert call() == pk.PCCL_ERR_CUDA


def test_step_R_threaded_one_pass_normaliser_at_full_size(pk):
    """From 2^15 post pairs on, the one-pass normaliser works on slices of the chunk range, one per host thread (count
    and validate, then write).  Config 5 at full size (0.48 M post pairs, uneven chunks per NPU): the conditions against
    the definition, computed here with numpy; a deviation from the chunk order in the middle of the list must fall back
    to the general path with the same result, and an invalid pair in a late slice must be refused."""
    p = wl.config5(0)
    assert len(p.post) >= 1 << 17

    def conditions(pre, post):
        pr = pk.Problem(pk.Topology(p.n_npus, p.links), p.group, p.n_chunks, pre, post, p.chunk_bytes)
        assert pr.mode == 0
        cs = np.random.default_rng(3).integers(0, p.n_chunks, 4000)
        cs = np.concatenate([cs, np.arange(64), np.arange(p.n_chunks - 64, p.n_chunks),
                             (np.arange(1, 8)[:, None] * p.n_chunks // 8 + np.arange(-3, 4)).ravel()])
        return pr, {int(c): (lambda sd: (sd[0], tuple(sd[1].tolist())))(pr.condition(0, int(c))) for c in cs}

    src = np.zeros(p.n_chunks, dtype=np.int64)
    src[p.pre["chunk"]] = p.pre["npu"]
    order = np.lexsort((p.post["npu"], p.post["chunk"]))
    pc, pn = p.post["chunk"][order].astype(np.int64), p.post["npu"][order].astype(np.int64)
    keep = pn != src[pc]
    pc, pn = pc[keep], pn[keep]
    off = np.concatenate([[0], np.cumsum(np.bincount(pc, minlength=p.n_chunks))])
    pr, got = conditions(p.pre, p.post)
    for c, (s, d) in got.items():
        assert s == src[c] and d == tuple(pn[off[c]:off[c + 1]].tolist()), c
    # total number of destinations = what the device would be given
    n = pk.lib.pccl_problem_condition(pr.handle, 0, p.n_chunks - 1, None, None, 0)
    assert n == off[-1] - off[-2]
    # two adjacent pairs of different chunks swapped in the middle: not chunk-ordered any more -> general path, same result
    post2 = p.post.copy()
    m = len(post2) // 2
    while post2["chunk"][m] == post2["chunk"][m + 1]:
        m += 1
    post2[[m, m + 1]] = post2[[m + 1, m]]
    assert conditions(p.pre, post2)[1] == got
    # an out-of-range NPU near the end
    post3 = p.post.copy()
    post3["npu"][-7] = p.n_npus
    with pytest.raises(pk.PcclError) as e:
        conditions(p.pre, post3)
    assert e.value.code == pk.PCCL_ERR_INVALID
