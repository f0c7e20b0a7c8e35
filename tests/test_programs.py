"""Per-node programs (translation step): pins of the oracle's definition (no GPU) and
parity of the CUDA export against it (GPU)."""
import numpy as np
import pytest

import oracle
import workloads as wl


def test_programs_of_a_two_hop_relay_by_hand():
    """0 -> 1 -> 2, one chunk: node 1 receives at w and sends at w (receive listed first)."""
    p = wl.path_point_to_point(3, seed=0)
    s = oracle.synthesize(*p.args())
    w = 520_972
    off, ops = oracle.programs(s.transfers, 3)
    assert off.tolist() == [0, 1, 3, 4]
    rows = [(int(o["kind"]), int(o["peer"]), int(o["chunk"]), int(o["time_ps"])) for o in ops]
    assert rows == [(1, 1, 0, 0), (0, 0, 0, w), (1, 2, 0, w), (0, 1, 0, 2 * w)]


@pytest.mark.parametrize("maker", [wl.config1, wl.config2, wl.config3, wl.config4_small])
def test_program_invariants(maker):
    p = maker(1)
    s = oracle.synthesize(*p.args())
    off, ops = oracle.programs(s.transfers, p.n_npus)
    assert off[-1] == 2 * len(s.transfers) == len(ops)
    sends = {}
    for v in range(p.n_npus):
        prog = ops[int(off[v]):int(off[v + 1])]
        key = list(zip(prog["time_ps"].tolist(), prog["kind"].tolist(), prog["link"].tolist()))
        assert key == sorted(key)                                 # time-ordered, receive before send, then link
        for o in prog[prog["kind"] == 1]:
            sends[(v, int(o["peer"]), int(o["chunk"]), int(o["link"]), int(o["time_ps"]))] = True
        assert np.all(p.links["dst"][prog["link"][prog["kind"] == 0]] == v)
        assert np.all(p.links["src"][prog["link"][prog["kind"] == 1]] == v)
    for r in s.transfers:                                         # every transfer appears as exactly one send
        assert (int(r["src"]), int(r["dst"]), int(r["chunk"]), int(r["link"]), int(r["t_start_ps"])) in sends


@pytest.mark.gpu
@pytest.mark.parametrize("maker", [wl.config1, wl.config2, wl.config3, wl.config4_small, wl.config5_small,
                                   wl.two_groups_mesh3x3])
def test_cuda_programs_match_the_definition(maker):
    import torch
    assert torch.cuda.is_available()
    import paper_2606_07019_b200 as pk
    pk.use_torch(0)
    p = maker(2)
    s = pk.synthesize(*p.args())
    off, ops = s.programs(p.n_npus)
    woff, wops = oracle.programs(s.transfers, p.n_npus)
    assert np.array_equal(off, woff)
    for f in ops.dtype.names:
        assert np.array_equal(ops[f], wops[f]), f


@pytest.mark.gpu
def test_cuda_programs_empty_schedule():
    import paper_2606_07019_b200 as pk
    pk.use_torch(0)
    links = wl.ring_links(4, True)
    members = np.arange(4, dtype=np.uint32)
    pre = np.array([(0, 0)], dtype=wl.PAIR_DT)
    s = pk.synthesize(4, links, members, 1, pre, pre.copy(), 64, 0)
    off, ops = s.programs(4)
    assert off.tolist() == [0] * 5 and len(ops) == 0
