"""pccl_candidate_totals_static -- the entry point that allocates nothing (include/pccl.h) -- against the existing
path, pccl_device_candidate_sweep, on the same bitmaps: |have[src_l] & wants[dst_l]| of every link, integer work, so
the comparison is bit-exact like every other parity test here.

The file is named to be collected LAST (the suite runs with pytest -x).  It needs nothing from the other test files
and passes alone in a fresh process as well as after them: the entry point shares no state with the other entry points
except the library's fixed scratch array, which each call clears before use.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import workloads as wl  # noqa: E402


@pytest.fixture(scope="module")
def pk():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_07019_b200 as pk
    pk.use_torch(0)
    return pk


def _bitmaps(pk, p):
    """(existing path's totals, have, wants, words_per_row, link_src, in_off, in_link) of phase 0 of problem p: the
    bitmaps are rebuilt on the host from the precondition and the library's wants accessor, laid out as the header
    asks: rows of an even number of 64-bit words, bit c = chunk c."""
    topo = pk.Topology(p.n_npus, p.links)
    prob = pk.Problem(topo, p.group, p.n_chunks, p.pre, p.post, p.chunk_bytes)
    _, _, ref = prob.candidate_sweep(0, p.seed)                  # the existing path (allocates its workspace)
    n_chunks = int(pk.pccl_problem_n_chunks(prob.handle))
    wp = max(2, (n_chunks + 63) // 64 + ((n_chunks + 63) // 64) % 2)
    have = np.zeros((p.n_npus, wp), dtype=np.uint64)
    wants = np.zeros((p.n_npus, wp), dtype=np.uint64)
    assert prob.mode == 0 and len(np.unique(p.pre["chunk"])) == len(p.pre) == n_chunks   # copy mode, one holder per chunk
    np.bitwise_or.at(have, (p.pre["npu"].astype(np.int64), (p.pre["chunk"] >> 6).astype(np.int64)),
                     np.uint64(1) << (p.pre["chunk"] & 63).astype(np.uint64))
    w = prob.wants(0, p.seed)
    np.bitwise_or.at(wants, (w["npu"].astype(np.int64), (w["chunk"] >> 6).astype(np.int64)),
                     np.uint64(1) << (w["chunk"] & 63).astype(np.uint64))
    dst = p.links["dst"].astype(np.int64)
    in_link = np.argsort(dst, kind="stable").astype(np.uint32)  # CSR by destination, ascending link id inside a node
    in_off = np.zeros(p.n_npus + 1, dtype=np.uint32)
    np.add.at(in_off, dst + 1, 1)
    in_off = np.cumsum(in_off).astype(np.uint32)
    # the same thing once more with numpy alone (guards the rebuilt bitmaps themselves)
    host = np.array([int(np.bitwise_count(have[int(l["src"])] & wants[int(l["dst"])]).sum()) for l in p.links], dtype=np.uint32)
    assert np.array_equal(host, ref), "rebuilt bitmaps disagree with the existing path"
    return ref, have, wants, wp, p.links["src"].astype(np.uint32), in_off, in_link


def _upload(torch, case):
    _, have, wants, _, src, in_off, in_link = case
    dev = [torch.from_numpy(x.view(np.int64) if x.dtype == np.uint64 else x.view(np.int32)).cuda()
           for x in (have, wants, src, in_off, in_link)]
    totals = torch.full((len(src),), -7, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    return dev, totals


def _static_call(pk, torch, case, stream=0, bufs=None):
    dev, totals = bufs or _upload(torch, case)
    pk.candidate_totals_static(dev[0], dev[1], case[1].shape[0], len(case[4]), case[3], dev[2], dev[3], dev[4], totals, stream)
    torch.cuda.synchronize()
    return totals.cpu().numpy().view(np.uint32)


def test_static_entry_point_equals_the_existing_path_on_calls_in_a_row(pk):
    """Three problems of different shape back to back (rows of 130, 2 and 64 words; 2, 39 and 6 in-links per node), then
    the first again: each call finds the previous call's counts in the shared array and must not see them."""
    import torch
    cases = [_bitmaps(pk, wl.ring_all_gather(8, True, 2, chunks_per_npu=1040, chunk_bytes=4096)),
             _bitmaps(pk, wl.full_mesh_problem(40, "allgather", seed=2)),
             _bitmaps(pk, wl.config4_small(1))]
    for i in (0, 1, 2, 0, 0):
        got = _static_call(pk, torch, cases[i])
        assert np.array_equal(got, cases[i][0]), f"case {i}"
    assert cases[0][0].sum() > 0 and cases[1][0].sum() > 0


def test_static_entry_point_allocates_nothing_and_runs_on_the_callers_stream(pk):
    import torch
    case = _bitmaps(pk, wl.config5_small(3))
    bufs = _upload(torch, case)
    assert np.array_equal(_static_call(pk, torch, case, 0, bufs), case[0])    # (set-up of the device done here)
    s = torch.cuda.Stream()
    bufs[1].fill_(-7)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    n0 = pk.launch_count()
    for _ in range(3):
        pk.candidate_totals_static(*bufs[0][:2], case[1].shape[0], len(case[4]), case[3], *bufs[0][2:], bufs[1], s.cuda_stream)
    s.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert pk.launch_count() - n0 == 6                           # the sweep kernel and the totals kernel per call, nothing else
    assert free1 == free0                                        # no device memory taken from the driver
    assert np.array_equal(bufs[1].cpu().numpy().view(np.uint32), case[0])


def test_static_entry_point_rejects_what_does_not_fit(pk):
    import torch
    z = torch.zeros(64, dtype=torch.int64, device="cuda")
    limit = pk.PCCL_STATIC_SCRATCH_BYTES
    # n_links * (ceil(words / 64) + 1) * 4 bytes must fit: 2 words per row -> 8 bytes per link
    ok_links = limit // 8
    with pytest.raises(pk.PcclError) as e:
        pk.candidate_totals_static(z, z, 4, ok_links + 1, 2, z, z, z, z)
    assert e.value.code == pk.PCCL_ERR_TOO_LARGE and b"scratch" in pk.pccl_strerror(pk.PCCL_ERR_TOO_LARGE)
    with pytest.raises(pk.PcclError) as e:
        pk.candidate_totals_static(z, z, 4, 1 << 10, 1 << 18, z, z, z, z)     # (4096 + 1) segments x 1024 links x 4 B
    assert e.value.code == pk.PCCL_ERR_TOO_LARGE
    for bad in (dict(words=3), dict(words=0), dict(have=z.data_ptr() + 8), dict(totals=0)):
        with pytest.raises(pk.PcclError) as e:
            pk.candidate_totals_static(bad.get("have", z), z, 4, 4, bad.get("words", 2), z, z, z, bad.get("totals", z))
        assert e.value.code == pk.PCCL_ERR_INVALID, bad
    pk.candidate_totals_static(z, z, 0, 0, 2, z, z, z, z)         # empty problem: nothing to do
    torch.cuda.synchronize()
