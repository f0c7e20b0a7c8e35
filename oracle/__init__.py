"""CPU oracle of the link-chunk matching synthesizer -- TEST INFRASTRUCTURE ONLY.

Nothing under ``paper_2606_07019_b200/`` may import this package.  Allowed callers:
``tests/``, ``__graft_entry__.smoke()``, and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs.  The arithmetic lives in ``pccl_oracle.cpp`` (plain C++17, one
thread); this file only builds it with g++ and marshals numpy arrays through ctypes.

Paper anchors are in the header of ``pccl_oracle.cpp``; the readings of the paper it follows
are listed in ``DESIGN.md``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pccl_oracle.cpp")
_LIB = os.path.join(_HERE, "libpccl_oracle.so")

LINK_DT = np.dtype([("src", "<u4"), ("dst", "<u4"), ("alpha_ps", "<u8"), ("bytes_per_ps", "<u8")])
PAIR_DT = np.dtype([("npu", "<u4"), ("chunk", "<u4")])
REC_DT = np.dtype([("chunk", "<u4"), ("src", "<u4"), ("dst", "<u4"), ("link", "<u4"),
                   ("t_start_ps", "<u8"), ("t_end_ps", "<u8")])

OK, ERR_INVALID, ERR_UNSUPPORTED, ERR_UNREACHABLE, ERR_INTERNAL = 0, -1, -2, -3, -6


class OracleError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"oracle error {code}")
        self.code = code


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (single thread, no CUDA).  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, u32, u64, i64 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_int64
        L.oracle_philox4x32_10.argtypes = [vp, vp, vp]
        L.oracle_philox4x32_10.restype = None
        L.oracle_link_cost.argtypes = [u64, u64, u64]
        L.oracle_link_cost.restype = u64
        L.oracle_distances.argtypes = [u32, vp, u32, u64, u32, vp]
        L.oracle_distances.restype = C.c_int
        L.oracle_synthesize.argtypes = [u32, vp, u32, vp, u32, u32, vp, u64, vp, u64, u64, u64,
                                        C.POINTER(vp)]
        L.oracle_synthesize.restype = C.c_int
        L.oracle_synthesize_relay.argtypes = [u32, vp, u32, vp, u32, u32, vp, u64, vp, u64, u64, u64, C.c_int,
                                              C.POINTER(vp)]
        L.oracle_synthesize_relay.restype = C.c_int
        L.oracle_synthesize_switches.argtypes = [u32, vp, u32, vp, u32, u32, vp, u64, vp, u64, u64, u64, vp, vp,
                                                 C.POINTER(vp)]
        L.oracle_synthesize_switches.restype = C.c_int
        L.oracle_synthesize_pipelined.argtypes = [u32, vp, u32, vp, u32, u32, vp, u64, vp, u64, u64, u64, C.POINTER(vp)]
        L.oracle_synthesize_pipelined.restype = C.c_int
        L.oracle_wants.argtypes = [u32, vp, u32, u32, vp, vp, vp, u64, u64, vp, u64]
        L.oracle_wants.restype = i64
        for name in ("oracle_size", "oracle_time", "oracle_events", "oracle_wants_total",
                     "oracle_time_phase1"):
            getattr(L, name).argtypes = [vp]
            getattr(L, name).restype = u64
        L.oracle_records.argtypes = [vp]
        L.oracle_records.restype = vp
        L.oracle_mode.argtypes = [vp]
        L.oracle_mode.restype = C.c_int
        L.oracle_free.argtypes = [vp]
        L.oracle_free.restype = None
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p) if a.size else None


def philox4x32_10(ctr, key) -> tuple:
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    o = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_ptr(c), _ptr(k), _ptr(o))
    return tuple(int(x) for x in o)


def link_cost(alpha_ps: int, bytes_per_ps: int, chunk_bytes: int) -> int:
    return int(lib().oracle_link_cost(alpha_ps, bytes_per_ps, chunk_bytes))


def distances(n_npus: int, links: np.ndarray, chunk_bytes: int, s: int) -> np.ndarray:
    links = np.ascontiguousarray(links, dtype=LINK_DT)
    out = np.zeros(n_npus, dtype=np.uint64)
    rc = lib().oracle_distances(n_npus, _ptr(links), len(links), chunk_bytes, s, _ptr(out))
    if rc:
        raise OracleError(rc)
    return out


class OracleSchedule:
    """Result of one oracle run (host numpy copies; nothing refers to the C object)."""

    def __init__(self, transfers, time_ps, events, wants_total, time_phase1_ps, mode, seconds):
        self.transfers = transfers            # REC_DT array, canonical order
        self.time_ps = time_ps                # max t_end
        self.events = events                  # event times processed
        self.wants_total = wants_total        # popcount(wants) after step C
        self.time_phase1_ps = time_phase1_ps  # all-reduce: reduce-phase time
        self.mode = mode                      # 0 copy, 1 reduce, 2 all-reduce
        self.seconds = seconds                # wall time of the C++ call (steady clock)


RELAY_THIN, RELAY_DYNAMIC, RELAY_BFS = 0, 1, 2
RELAY_THIN_DIST_PICK = 3      # the thin relay tree with the c.dist-priority pick (Q27)


NO_LIMIT = 0xFFFFFFFF


def synthesize(n_npus, links, group, n_chunks, pre, post, chunk_bytes, seed, relay: int = RELAY_THIN,
               buffer_limit=None, no_multicast=None, pipeline: bool = False) -> OracleSchedule:
    """Same problem statement as the product boundary (include/pccl.h), host arrays only.
    relay: RELAY_THIN (static thin relay tree, the default), RELAY_DYNAMIC (Q18) or RELAY_BFS (the paper's
    own per-condition search, Alg. 1-3, Q19-Q22; `events` then counts conditions routed).
    buffer_limit / no_multicast (RELAY_BFS only): the switch model of PAPER.md:348, per node (Q23-Q25).
    pipeline (RELAY_BFS only): an All-Reduce's copy phase of a chunk starts when its root is complete (Q26)."""
    links = np.ascontiguousarray(links, dtype=LINK_DT)
    group = np.ascontiguousarray(group, dtype=np.uint32)
    pre = np.ascontiguousarray(pre, dtype=PAIR_DT)
    post = np.ascontiguousarray(post, dtype=PAIR_DT)
    h = C.c_void_p()
    t0 = time.perf_counter()
    if pipeline:
        if relay != RELAY_BFS or buffer_limit is not None or no_multicast is not None:
            raise ValueError("pipelined All-Reduce: RELAY_BFS without a switch model")
        rc = lib().oracle_synthesize_pipelined(n_npus, _ptr(links), len(links), _ptr(group), len(group),
                                               n_chunks, _ptr(pre), len(pre), _ptr(post), len(post), chunk_bytes, seed,
                                               C.byref(h))
    elif buffer_limit is not None or no_multicast is not None:
        if relay != RELAY_BFS:
            raise ValueError("the switch model applies to RELAY_BFS only")
        bl = None if buffer_limit is None else np.ascontiguousarray(buffer_limit, dtype=np.uint32)
        nm = None if no_multicast is None else np.ascontiguousarray(no_multicast, dtype=np.uint8)
        assert (bl is None or len(bl) == n_npus) and (nm is None or len(nm) == n_npus)
        rc = lib().oracle_synthesize_switches(n_npus, _ptr(links), len(links), _ptr(group), len(group),
                                              n_chunks, _ptr(pre), len(pre), _ptr(post), len(post), chunk_bytes, seed,
                                              None if bl is None else _ptr(bl), None if nm is None else _ptr(nm), C.byref(h))
    else:
        rc = lib().oracle_synthesize_relay(n_npus, _ptr(links), len(links), _ptr(group), len(group),
                                           n_chunks, _ptr(pre), len(pre), _ptr(post), len(post),
                                           chunk_bytes, seed, int(relay), C.byref(h))
    dt = time.perf_counter() - t0
    if rc:
        raise OracleError(rc)
    try:
        n = int(lib().oracle_size(h))
        recs = np.zeros(n, dtype=REC_DT)
        if n:
            C.memmove(recs.ctypes.data, lib().oracle_records(h), n * REC_DT.itemsize)
        return OracleSchedule(recs, int(lib().oracle_time(h)), int(lib().oracle_events(h)),
                              int(lib().oracle_wants_total(h)), int(lib().oracle_time_phase1(h)),
                              int(lib().oracle_mode(h)), dt)
    finally:
        lib().oracle_free(h)


def wants(n_npus, links, n_chunks, cond_src, dest_off, dests, chunk_bytes, seed) -> np.ndarray:
    """Step C relation for COPY-mode conditions: PAIR_DT array sorted by (node, chunk)."""
    links = np.ascontiguousarray(links, dtype=LINK_DT)
    cond_src = np.ascontiguousarray(cond_src, dtype=np.uint32)
    dest_off = np.ascontiguousarray(dest_off, dtype=np.uint64)
    dests = np.ascontiguousarray(dests, dtype=np.uint32)
    cap = int(n_npus) * max(int(n_chunks), 1)
    cap = min(cap, 64_000_000)
    out = np.zeros(cap, dtype=PAIR_DT)
    k = lib().oracle_wants(n_npus, _ptr(links), len(links), n_chunks, _ptr(cond_src),
                           _ptr(dest_off), _ptr(dests), chunk_bytes, seed, _ptr(out), cap)
    if k < 0:
        raise OracleError(int(k))
    if k > cap:
        raise OracleError(ERR_INTERNAL)
    return out[:k].copy()


def schedule_hash(transfers: np.ndarray) -> str:
    """FNV-1a-style 64-bit hash over fields (chunk, src, dst, link, t_start, t_end), each as a
    64-bit integer, records in canonical order (quick comparison only)."""
    h = 0xCBF29CE484222325
    mask = (1 << 64) - 1
    for r in transfers:
        for f in ("chunk", "src", "dst", "link", "t_start_ps", "t_end_ps"):
            h = ((h ^ int(r[f])) * 0x100000001B3) & mask
    return f"{h:016x}"


OP_DT = np.dtype([("kind", "<u4"), ("peer", "<u4"), ("chunk", "<u4"), ("link", "<u4"), ("time_ps", "<u8")])


def programs(transfers: np.ndarray, n_npus: int):
    """Translation step (section 4.8) written out: every transfer is a RECEIVE (kind 0) at its
    destination, complete at t_end, and a SEND (kind 1) at its source, starting at t_start; a node's program is
    its operations ordered by (time, kind, link).  Returns (offsets[n_npus + 1], ops)."""
    m = len(transfers)
    node = np.concatenate([transfers["dst"], transfers["src"]]).astype(np.int64)
    ops = np.zeros(2 * m, dtype=OP_DT)
    ops["kind"] = np.concatenate([np.zeros(m, np.uint32), np.ones(m, np.uint32)])
    ops["peer"] = np.concatenate([transfers["src"], transfers["dst"]])
    ops["chunk"] = np.concatenate([transfers["chunk"], transfers["chunk"]])
    ops["link"] = np.concatenate([transfers["link"], transfers["link"]])
    ops["time_ps"] = np.concatenate([transfers["t_end_ps"], transfers["t_start_ps"]])
    order = np.lexsort((ops["link"], ops["kind"], ops["time_ps"], node))   # last key is the primary one
    offsets = np.zeros(n_npus + 1, dtype=np.uint64)
    offsets[1:] = np.cumsum(np.bincount(node, minlength=n_npus))
    return offsets, ops[order]
