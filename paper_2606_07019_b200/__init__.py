"""paper_2606_07019_b200 -- Python binding of libpccl.so (include/pccl.h).

Argument marshalling only: every step of the synthesis (link costs, distances, wants
bitmaps, the event loop, the emitter) runs in the CUDA kernels behind the C-ABI.  PyTorch
supplies device memory (its caching allocator, through ``pccl_set_allocator``) and the
current CUDA stream (``pccl_set_stream``); nothing else.  There is no CPU fallback: if the
library cannot be built or loaded, importing this package raises.

The module-level functions carry the C names (``pccl_topology_create`` ...) with ctypes
signatures; ``Topology`` / ``Problem`` / ``Schedule`` are thin RAII holders around the
handles, and ``synthesize`` is the one-call form of the paper's problem statement
(PAPER.md:149-156): topology + process group + pre/postcondition + chunk size -> schedule.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import _build

LINK_DT = np.dtype([("src", "<u4"), ("dst", "<u4"), ("alpha_ps", "<u8"), ("bytes_per_ps", "<u8")])
PAIR_DT = np.dtype([("npu", "<u4"), ("chunk", "<u4")])
OP_DT = np.dtype([("kind", "<u4"), ("peer", "<u4"), ("chunk", "<u4"), ("link", "<u4"), ("time_ps", "<u8")])
TRANSFER_DT = np.dtype([("chunk", "<u4"), ("src", "<u4"), ("dst", "<u4"), ("link", "<u4"),
                        ("t_start_ps", "<u8"), ("t_end_ps", "<u8")])

PCCL_OK, PCCL_ERR_INVALID, PCCL_ERR_UNSUPPORTED, PCCL_ERR_UNREACHABLE = 0, -1, -2, -3
PCCL_ERR_CUDA, PCCL_ERR_NOMEM, PCCL_ERR_INTERNAL, PCCL_ERR_TOO_LARGE = -4, -5, -6, -7
PCCL_STATIC_SCRATCH_BYTES = 4 << 20
PCCL_FLAG_KEEP_ON_DEVICE, PCCL_FLAG_NO_IDLE_SKIP, PCCL_FLAG_TIME_LOOP, PCCL_FLAG_TRACE = 1, 2, 4, 8
PCCL_FLAG_DENSE_SWEEP = 16
PCCL_FLAG_RESCAN = 32
PCCL_FLAG_DYNAMIC_RELAY = 64
PCCL_FLAG_KEPT_COUNTS = 128
PCCL_FLAG_TWO_BARRIERS = 256
PCCL_FLAG_BFS = 512
PCCL_FLAG_BARRIER_LOOP = 1024
PCCL_FLAG_ASYNC = 2048
PCCL_FLAG_LSU_SWEEP = 4096
PCCL_FLAG_PIPELINE = 8192
PCCL_FLAG_DIST_PICK = 16384
PCCL_TRACE_SLOTS = 12
PCCL_OPT_BFS_WINDOW, PCCL_OPT_BFS_ROWS, PCCL_OPT_DYNAMIC_RECORDS = 1, 2, 3


class pccl_condition_t(C.Structure):
    _fields_ = [("n_chunks", C.c_uint32), ("n_pairs", C.c_uint64), ("pairs", C.c_void_p)]


class pccl_stats_t(C.Structure):
    _fields_ = [("events", C.c_uint64), ("wants_total", C.c_uint64), ("rows_scanned", C.c_uint64),
                ("bytes_requested", C.c_uint64), ("row_bytes", C.c_uint64), ("links_scanned", C.c_uint64), ("slow_picks", C.c_uint64),
                ("time_phase1_ps", C.c_uint64), ("loop_ms", C.c_float), ("setup_ms", C.c_float),
                ("emit_ms", C.c_float), ("mode", C.c_uint32), ("grid_blocks", C.c_uint32)]


pccl_alloc_fn = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
pccl_free_fn = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

#: every symbol include/pccl.h declares: name -> (restype, argtypes)
_vp, _u32, _u64, _i64, _int = C.c_void_p, C.c_uint32, C.c_uint64, C.c_int64, C.c_int
SIGNATURES = {
    "pccl_set_stream": (None, [_vp]),
    "pccl_set_allocator": (None, [pccl_alloc_fn, pccl_free_fn, _vp]),
    "pccl_strerror": (C.c_char_p, [_int]),
    "pccl_version": (_int, []),
    "pccl_set_option": (_int, [_int, _u64]),
    "pccl_get_option": (_u64, [_int]),
    "pccl_launch_count": (_u64, []),
    "pccl_topology_create": (_int, [_u32, _vp, _u32, C.POINTER(_vp)]),
    "pccl_topology_set_switch_model": (_int, [_vp, _vp, _vp]),
    "pccl_topology_destroy": (None, [_vp]),
    "pccl_topology_n_npus": (_u32, [_vp]),
    "pccl_topology_n_links": (_u32, [_vp]),
    "pccl_synthesize": (_int, [_vp, _vp, _u32, C.POINTER(pccl_condition_t), C.POINTER(pccl_condition_t),
                               _u64, _u64, C.POINTER(_vp)]),
    "pccl_problem_create": (_int, [_vp, _vp, _u32, C.POINTER(pccl_condition_t),
                                   C.POINTER(pccl_condition_t), _u64, C.POINTER(_vp)]),
    "pccl_problem_destroy": (None, [_vp]),
    "pccl_problem_upload": (_int, [_vp]),
    "pccl_problem_mode": (_int, [_vp]),
    "pccl_problem_n_chunks": (_u32, [_vp]),
    "pccl_problem_condition": (_i64, [_vp, _u32, _u32, C.POINTER(_u32), _vp, _u64]),
    "pccl_problem_synthesize": (_int, [_vp, _u64, _u32, C.POINTER(_vp)]),
    "pccl_schedule_time": (_u64, [_vp]),
    "pccl_schedule_size": (_u64, [_vp]),
    "pccl_schedule_transfers": (_vp, [_vp]),
    "pccl_schedule_transfers_device": (_vp, [_vp]),
    "pccl_schedule_destroy": (None, [_vp]),
    "pccl_schedule_stats": (_int, [_vp, C.POINTER(pccl_stats_t)]),
    "pccl_schedule_trace": (_i64, [_vp, _vp, _u64]),
    "pccl_schedule_programs": (_int, [_vp, _vp, _vp]),
    "pccl_device_philox": (_int, [_vp, _u64, _vp, _vp]),
    "pccl_device_link_costs": (_int, [_vp, _u64, _vp]),
    "pccl_device_distances": (_int, [_vp, _u64, _u32, _int, _vp]),
    "pccl_device_wants": (_i64, [_vp, _u32, _u64, _vp, _u64]),
    "pccl_device_candidate_sweep": (_int, [_vp, _u32, _u64, _u32, _u32, C.POINTER(C.c_float), C.POINTER(_u64), _vp]),
    "pccl_device_read_bandwidth": (_int, [_u64, _u32, C.POINTER(C.c_float)]),
    "pccl_candidate_totals_static": (_int, [_vp, _vp, _u32, _u32, _u32, _vp, _vp, _vp, _vp, _vp]),
}


def _load() -> C.CDLL:
    path = _build.build()          # raises if nvcc is missing or the build fails: no fallback
    lib = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)    # AttributeError if the library lacks a declared symbol
        fn.restype = res
        fn.argtypes = args
    return lib


LIB_PATH = _build.LIB
lib = _load()
globals().update({name: getattr(lib, name) for name in SIGNATURES})


class PcclError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"pccl error {code}: {lib.pccl_strerror(code).decode()}")
        self.code = code


def _check(rc: int) -> None:
    if rc != PCCL_OK:
        raise PcclError(int(rc))


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p) if a.size else None


# ------------------------------------------------------------------------------------------
# PyTorch plumbing: device memory and stream
# ------------------------------------------------------------------------------------------
_hooks = None


def use_torch(device: int | None = None) -> None:
    """Route the library's device allocations to torch's caching allocator and its work to
    torch's current stream on ``device`` (default: the current device)."""
    global _hooks
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2606_07019_b200 needs a CUDA device; there is no CPU path")
    if device is not None:
        torch.cuda.set_device(device)
    dev = torch.cuda.current_device()
    torch.cuda.init()

    def _alloc(nbytes, stream, _user):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), dev, int(stream or 0))
        except Exception:
            return None

    _delete = torch.cuda.caching_allocator_delete

    def _free(ptr, _user):
        try:
            _delete(int(ptr))
        except Exception:   # interpreter shutdown: torch is already torn down, the context goes with the process
            pass

    _hooks = (pccl_alloc_fn(_alloc), pccl_free_fn(_free))
    lib.pccl_set_allocator(_hooks[0], _hooks[1], None)
    lib.pccl_set_stream(C.c_void_p(torch.cuda.current_stream().cuda_stream))


def set_option(option: int, value: int) -> None:
    _check(lib.pccl_set_option(option, value))


def launch_count() -> int:
    """Kernels the library has launched so far in this process."""
    return int(lib.pccl_launch_count())


def sync_stream() -> None:
    """Re-read torch's current stream (call after entering a ``torch.cuda.stream`` context)."""
    import torch
    lib.pccl_set_stream(C.c_void_p(torch.cuda.current_stream().cuda_stream))


# ------------------------------------------------------------------------------------------
# RAII holders
# ------------------------------------------------------------------------------------------
class Topology:
    def __init__(self, n_npus: int, links: np.ndarray):
        self._links = np.ascontiguousarray(links, dtype=LINK_DT)
        h = C.c_void_p()
        _check(lib.pccl_topology_create(n_npus, _ptr(self._links), len(self._links), C.byref(h)))
        self.handle = h
        self.n_npus, self.n_links = int(n_npus), len(self._links)

    def set_switch_model(self, buffer_limit=None, no_multicast=None) -> None:
        """per-node buffer limits (0xFFFFFFFF = none) and no-multicast flags for PCCL_FLAG_BFS."""
        bl = None if buffer_limit is None else np.ascontiguousarray(buffer_limit, dtype=np.uint32)
        nm = None if no_multicast is None else np.ascontiguousarray(no_multicast, dtype=np.uint8)
        assert (bl is None or len(bl) == self.n_npus) and (nm is None or len(nm) == self.n_npus)
        _check(lib.pccl_topology_set_switch_model(self.handle, None if bl is None else _ptr(bl), None if nm is None else _ptr(nm)))

    def link_costs(self, chunk_bytes: int) -> np.ndarray:
        out = np.zeros(self.n_links, dtype=np.uint64)
        _check(lib.pccl_device_link_costs(self.handle, chunk_bytes, _ptr(out)))
        return out

    def distances(self, chunk_bytes: int, src: int, transposed: bool = False) -> np.ndarray:
        out = np.zeros(self.n_npus, dtype=np.uint64)
        _check(lib.pccl_device_distances(self.handle, chunk_bytes, src, int(transposed), _ptr(out)))
        return out

    def close(self):
        if getattr(self, "handle", None) and lib is not None:
            lib.pccl_topology_destroy(self.handle)
            self.handle = None

    __del__ = close


def _condition(n_chunks: int, pairs: np.ndarray):
    pairs = np.ascontiguousarray(pairs, dtype=PAIR_DT)
    return pccl_condition_t(n_chunks, len(pairs), pairs.ctypes.data if pairs.size else None), pairs


class Schedule:
    def __init__(self, handle):
        self.handle = handle
        self.time_ps = int(lib.pccl_schedule_time(handle))
        self.size = int(lib.pccl_schedule_size(handle))

    @property
    def transfers(self) -> np.ndarray:
        """TRANSFER_DT records in canonical order (a host copy owned by numpy)."""
        if self.size == 0:
            return np.zeros(0, dtype=TRANSFER_DT)
        p = lib.pccl_schedule_transfers(self.handle)
        if not p:
            raise PcclError(PCCL_ERR_CUDA)
        buf = (C.c_char * (self.size * TRANSFER_DT.itemsize)).from_address(p)
        return np.frombuffer(buf, dtype=TRANSFER_DT).copy()

    @property
    def device_ptr(self) -> int:
        return int(lib.pccl_schedule_transfers_device(self.handle) or 0)

    @property
    def stats(self) -> dict:
        s = pccl_stats_t()
        _check(lib.pccl_schedule_stats(self.handle, C.byref(s)))
        return {k: getattr(s, k) for k, _ in pccl_stats_t._fields_}

    def programs(self, n_npus: int):
        """(offsets, ops): the program of node v is ops[offsets[v]:offsets[v+1]] (OP_DT records)."""
        offsets = np.zeros(n_npus + 1, dtype=np.uint64)
        ops = np.zeros(2 * self.size, dtype=OP_DT)
        _check(lib.pccl_schedule_programs(self.handle, _ptr(offsets), _ptr(ops)))
        return offsets, ops

    @property
    def trace(self) -> np.ndarray:
        """[events, PCCL_TRACE_SLOTS] ns stamps (needs PCCL_FLAG_TRACE), else an empty array."""
        n = int(lib.pccl_schedule_trace(self.handle, None, 0))
        out = np.zeros(max(n, 0), dtype=np.uint64)
        if n > 0:
            lib.pccl_schedule_trace(self.handle, _ptr(out), n)
        return out.reshape(-1, PCCL_TRACE_SLOTS)

    def close(self):
        if getattr(self, "handle", None) and lib is not None:
            lib.pccl_schedule_destroy(self.handle)
            self.handle = None

    __del__ = close


class Problem:
    def __init__(self, topo: Topology, group, n_chunks: int, pre, post, chunk_bytes: int):
        self.topo = topo                      # keeps the topology alive
        group = np.ascontiguousarray(group, dtype=np.uint32)
        pc, pa = _condition(n_chunks, pre)
        qc, qa = _condition(n_chunks, post)
        h = C.c_void_p()
        _check(lib.pccl_problem_create(topo.handle, _ptr(group), len(group), C.byref(pc), C.byref(qc),
                                       chunk_bytes, C.byref(h)))
        del pa, qa
        self.handle = h
        self.n_chunks = int(n_chunks)
        self.mode = int(lib.pccl_problem_mode(h))

    def upload(self) -> None:
        _check(lib.pccl_problem_upload(self.handle))

    def condition(self, phase: int, chunk: int):
        src = C.c_uint32()
        n = lib.pccl_problem_condition(self.handle, phase, chunk, C.byref(src), None, 0)
        if n < 0:
            raise PcclError(int(n))
        d = np.zeros(int(n), dtype=np.uint32)
        lib.pccl_problem_condition(self.handle, phase, chunk, C.byref(src), _ptr(d), int(n))
        return int(src.value), d

    def synthesize(self, seed: int, flags: int = 0) -> Schedule:
        h = C.c_void_p()
        _check(lib.pccl_problem_synthesize(self.handle, seed, flags, C.byref(h)))
        return Schedule(h)

    def wants(self, phase: int, seed: int) -> np.ndarray:
        n = lib.pccl_device_wants(self.handle, phase, seed, None, 0)
        if n < 0:
            raise PcclError(int(n))
        out = np.zeros(int(n), dtype=PAIR_DT)
        m = lib.pccl_device_wants(self.handle, phase, seed, _ptr(out), int(n))
        if m != n:
            raise PcclError(PCCL_ERR_INTERNAL if m >= 0 else int(m))
        return out

    def candidate_sweep(self, phase: int, seed: int, flags: int = 0, iters: int = 1):
        """(ms per sweep, algorithmic bytes per sweep, |cand(l)| of every link at t = 0)."""
        ms, nbytes = C.c_float(), C.c_uint64()
        tot = np.zeros(self.topo.n_links, dtype=np.uint32)
        _check(lib.pccl_device_candidate_sweep(self.handle, phase, seed, flags, iters, C.byref(ms), C.byref(nbytes), _ptr(tot)))
        return float(ms.value), int(nbytes.value), tot

    def close(self):
        if getattr(self, "handle", None) and lib is not None:
            lib.pccl_problem_destroy(self.handle)
            self.handle = None

    __del__ = close


def synthesize(n_npus, links, group, n_chunks, pre, post, chunk_bytes, seed) -> Schedule:
    """One call of ``pccl_synthesize`` with host numpy buffers (the e2e path)."""
    topo = Topology(n_npus, links)
    try:
        group = np.ascontiguousarray(group, dtype=np.uint32)
        pc, pa = _condition(n_chunks, pre)
        qc, qa = _condition(n_chunks, post)
        h = C.c_void_p()
        _check(lib.pccl_synthesize(topo.handle, _ptr(group), len(group), C.byref(pc), C.byref(qc),
                                   chunk_bytes, seed, C.byref(h)))
        del pa, qa
        return Schedule(h)
    finally:
        topo.close()


def read_bandwidth_gbs(nbytes: int, iters: int = 20) -> float:
    """GB/s of a sequential 128-bit read of an nbytes device buffer (L2-resident or not, by its size)."""
    ms = C.c_float()
    _check(lib.pccl_device_read_bandwidth(nbytes, iters, C.byref(ms)))
    return nbytes / (ms.value * 1e-3) / 1e9


def candidate_totals_static(have, wants, n_npus: int, n_links: int, words_per_row: int, link_src, in_off, in_link,
                            totals, stream: int = 0) -> None:
    """``pccl_candidate_totals_static``: |have[src_l] & wants[dst_l]| of every link into ``totals``, with no allocation
    (fixed scratch of PCCL_STATIC_SCRATCH_BYTES in the library).  Every array is a DEVICE buffer: an object with
    ``data_ptr()`` (a torch CUDA tensor) or a raw address.  Enqueues on ``stream`` (a cudaStream_t as int) and returns."""
    def dp(x):
        return C.c_void_p(int(x.data_ptr()) if hasattr(x, "data_ptr") else int(x))
    _check(lib.pccl_candidate_totals_static(dp(have), dp(wants), n_npus, n_links, words_per_row, dp(link_src), dp(in_off),
                                            dp(in_link), dp(totals), C.c_void_p(int(stream) or None)))


def device_philox(ctr, key) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros_like(ctr)
    _check(lib.pccl_device_philox(_ptr(ctr), len(ctr), _ptr(key), _ptr(out)))
    return out


# ------------------------------------------------------------------------------------------
# multi-GPU: replicas only.  The natural use of N GPUs is a
# best-of-K seed sweep: K independent syntheses, keep the smallest schedule time.
# ------------------------------------------------------------------------------------------
def shard_seeds(seeds, rank: int, world_size: int) -> list:
    """Seeds of this rank: a strided slice, so every rank gets floor or ceil of K / world."""
    return list(seeds)[rank::world_size]


def best_of_seeds(times_by_seed: dict, group=None):
    """Reduce {seed: schedule_time_ps} over the ranks of a torch.distributed group: returns
    (best_time_ps, best_seed) with ties broken by the smaller seed -- identical on every rank.
    Works with any backend (gloo on CPU, nccl on GPU); with no process group it is local."""
    import torch
    import torch.distributed as dist
    local = min(((int(t), int(s)) for s, t in times_by_seed.items()), default=((1 << 63) - 1, (1 << 63) - 1))
    if not (dist.is_available() and dist.is_initialized()):
        return local
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    mine = torch.tensor(list(local), dtype=torch.int64, device=dev)
    every = [torch.zeros_like(mine) for _ in range(dist.get_world_size(group))]
    dist.all_gather(every, mine, group=group)
    return min((int(e[0]), int(e[1])) for e in every)
