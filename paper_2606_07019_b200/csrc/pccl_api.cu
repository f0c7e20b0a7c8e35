// =========================================================================================
// pccl_api.cu -- host side of libpccl.so: the C-ABI of include/pccl.h, the normaliser
// (DESIGN.md step R), device-memory layout and kernel orchestration.  All arithmetic of
// steps A..F runs in the kernels of pccl_device.cuh; this file only validates, lays out
// memory, launches and copies.
// =========================================================================================
#include "../../include/pccl.h"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <future>
#include <system_error>
#include <mutex>
#include <new>
#include <memory>
#include <atomic>
#if defined(__x86_64__)
#include <immintrin.h>
#endif
#include <chrono>
#include <condition_variable>
#include <functional>
#include <thread>
#include <unordered_set>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "pccl_device.cuh"
#include "pccl_loop1.cuh"
#include "pccl_loop2.cuh"
#include "pccl_sweep.cuh"
#include "pccl_bfs.cuh"

using namespace pccl;

static_assert(sizeof(pccl_transfer_t) == sizeof(Rec), "record layout");
static_assert(sizeof(pccl_link_t) == 24 && sizeof(pccl_pair_t) == 8, "abi layout");

// -----------------------------------------------------------------------------------------
// process-wide plumbing
// -----------------------------------------------------------------------------------------
namespace {

struct Globals {
    cudaStream_t stream = nullptr;
    pccl_alloc_fn alloc = nullptr;
    pccl_free_fn release = nullptr;
    void* user = nullptr;
    std::mutex mu;
    // device entry points share the mailbox, the copy stream and G.stream: one call at a time (re-entrant: an
    // entry point may call another)
    std::recursive_mutex call_mu;
    // pinned host memory: a small mailbox for control blocks and a free-list of result buffers
    void* mailbox = nullptr;
    struct Pinned { void* p; size_t bytes; };
    std::vector<Pinned> pinned_free;
    int sm_count = 0;
    int dev = -1;
    // streaming the records out while the event loop runs: a copy stream of our own and the event the
    // polling host thread watches
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t loop_done = nullptr;
    // the barrier-free loop's emitter runs in windows on a stream of its own while the loop is going
    cudaStream_t emit_stream = nullptr;
    cudaEvent_t win_done = nullptr, pre_loop = nullptr;
    std::atomic<uint64_t> launches{0};   // kernels launched by the library (pccl_launch_count)
    // process-wide options (pccl_set_option); 0 = default
    std::atomic<uint64_t> opt_bfs_window{0}, opt_bfs_rows{0}, opt_dyn_records{0};
} G;

// every kernel launch of the library passes its stream through here: the count is the library's own evidence of what
// ran on the device (bench.py reports it as gpu_launches)
inline cudaStream_t counted(cudaStream_t s) { G.launches.fetch_add(1, std::memory_order_relaxed); return s; }

#define SERIALISE std::lock_guard<std::recursive_mutex> call_lock__(G.call_mu)

#ifdef PCCL_DEBUG_TIMELINE   /* debugging build: host-side time between marks of one call, to stderr */
static thread_local std::chrono::steady_clock::time_point dbgt_last__;
#define DBGT(label)                                                                                              \
    do {                                                                                                         \
        const auto now__ = std::chrono::steady_clock::now();                                                     \
        fprintf(stderr, "[t] %-28s %8.1f us\n", label,                                                           \
                std::chrono::duration<double, std::micro>(now__ - dbgt_last__).count());                         \
        dbgt_last__ = now__;                                                                                     \
    } while (0)
#else
#define DBGT(label) ((void)0)
#endif
#ifdef PCCL_DEBUG_CU   /* debugging build: say which call failed */
#define CU_REPORT(e) fprintf(stderr, "[pccl] line %d: %s\n", __LINE__, cudaGetErrorString(e))
#else
#define CU_REPORT(e) ((void)0)
#endif
#define CU(call)                                   \
    do {                                           \
        cudaError_t e__ = (call);                  \
        if (e__ != cudaSuccess) {                  \
            CU_REPORT(e__);                        \
            (void)cudaGetLastError();              \
            return PCCL_ERR_CUDA;                  \
        }                                          \
    } while (0)

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int dev_alloc(size_t bytes, void** out) {
    if (bytes == 0) bytes = 256;
    void* p = nullptr;
    if (G.alloc) {
        p = G.alloc(bytes, (void*)G.stream, G.user);
        if (!p) return PCCL_ERR_NOMEM;
    } else {
        cudaError_t e = cudaMallocAsync(&p, bytes, G.stream);
        if (e == cudaErrorMemoryAllocation) { (void)cudaGetLastError(); return PCCL_ERR_NOMEM; }
        if (e != cudaSuccess) { (void)cudaGetLastError(); return PCCL_ERR_CUDA; }
    }
    *out = p;
    return PCCL_OK;
}

void dev_free(void* p) {
    if (!p) return;
    if (G.release) G.release(p, G.user);
    else if (cudaFreeAsync(p, G.stream) != cudaSuccess) (void)cudaGetLastError();
}

// The library binds to the CUDA device that is current at its first device call (mailbox, copy stream, SM count);
// a later call with another current device is refused instead of mixing contexts.
int ensure_device() {
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (G.dev >= 0) return dev == G.dev ? PCCL_OK : PCCL_ERR_INVALID;
    int sms = 0, coop = 0;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CU(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    if (!coop) return PCCL_ERR_CUDA;
    void* mb = nullptr;
    cudaStream_t cs = nullptr, es = nullptr;
    cudaEvent_t ev = nullptr, ev2 = nullptr, ev3 = nullptr;
    if (cudaHostAlloc(&mb, 4096, cudaHostAllocDefault) != cudaSuccess ||
        cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&es, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ev2, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ev3, cudaEventDisableTiming) != cudaSuccess) {
        (void)cudaGetLastError();
        if (ev3) (void)cudaEventDestroy(ev3);
        if (ev2) (void)cudaEventDestroy(ev2);
        if (ev) (void)cudaEventDestroy(ev);
        if (es) (void)cudaStreamDestroy(es);
        if (cs) (void)cudaStreamDestroy(cs);
        if (mb) (void)cudaFreeHost(mb);
        return PCCL_ERR_CUDA;
    }
    G.mailbox = mb; G.copy_stream = cs; G.loop_done = ev;
    G.emit_stream = es; G.win_done = ev2; G.pre_loop = ev3;
    G.sm_count = sms;
    G.dev = dev;
    return PCCL_OK;
}

void* pinned_get(size_t bytes) {
    {
        std::lock_guard<std::mutex> lk(G.mu);
        size_t best = (size_t)-1;
        for (size_t i = 0; i < G.pinned_free.size(); ++i)
            if (G.pinned_free[i].bytes >= bytes && (best == (size_t)-1 || G.pinned_free[i].bytes < G.pinned_free[best].bytes)) best = i;
        if (best != (size_t)-1 && G.pinned_free[best].bytes <= 2 * bytes + (1u << 20)) {
            void* p = G.pinned_free[best].p;
            G.pinned_free.erase(G.pinned_free.begin() + best);
            return p;
        }
    }
    void* p = nullptr;
    if (cudaHostAlloc(&p, bytes ? bytes : 32, cudaHostAllocDefault) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    return p;
}

void pinned_put(void* p, size_t bytes) {
    if (!p) return;
    std::lock_guard<std::mutex> lk(G.mu);
    if (G.pinned_free.size() >= 4) {   // keep the cache small: drop the smallest
        size_t s = 0;
        for (size_t i = 1; i < G.pinned_free.size(); ++i) if (G.pinned_free[i].bytes < G.pinned_free[s].bytes) s = i;
        if (G.pinned_free[s].bytes < bytes) {
            (void)cudaFreeHost(G.pinned_free[s].p);
            G.pinned_free[s] = {p, bytes};
        } else {
            (void)cudaFreeHost(p);
        }
        return;
    }
    G.pinned_free.push_back({p, bytes});
}

// Host arrays of the normaliser: blocks of 64 KB and more come from a small process-wide cache (power-of-two
// size classes) instead of a fresh mmap per call -- at config 4 the ~17 MB of per-call vectors cost more in page
// faults than the grouping itself.  Smaller blocks go to malloc.
struct HostPool {
    static constexpr int MIN_LOG = 16, MAX_LOG = 34;
    static constexpr size_t CACHE_CAP = (size_t)256 << 20;
    std::mutex mu;
    std::vector<void*> free_[MAX_LOG + 1];
    size_t cached = 0;
    // pooled blocks are page-locked when a CUDA device is there (the condition arrays are uploaded straight from
    // them); without one -- the no-GPU tests -- they are plain malloc blocks
    std::unordered_set<void*> pinned;
    std::atomic<bool> try_pinned{true};
    void* fresh(size_t bytes) {
        if (try_pinned && bytes <= ((size_t)256 << 20)) {
            void* p = nullptr;
            if (cudaHostAlloc(&p, bytes, cudaHostAllocDefault) == cudaSuccess) {
                std::lock_guard<std::mutex> lk(mu);
                pinned.insert(p);
                return p;
            }
            (void)cudaGetLastError();
            try_pinned = false;
        }
        return malloc(bytes);
    }
    void release(void* p) {
        bool was_pinned;
        {
            std::lock_guard<std::mutex> lk(mu);
            was_pinned = pinned.erase(p) != 0;
        }
        if (was_pinned) (void)cudaFreeHost(p); else free(p);
    }
    static int size_class(size_t bytes) {
        int k = MIN_LOG;
        while (k < MAX_LOG && ((size_t)1 << k) < bytes) ++k;
        return k;
    }
    void* get(size_t bytes) {
        if (bytes < ((size_t)1 << MIN_LOG) || bytes > ((size_t)1 << MAX_LOG)) return malloc(bytes ? bytes : 1);
        const int k = size_class(bytes);
        {
            std::lock_guard<std::mutex> lk(mu);
            if (!free_[k].empty()) {
                void* p = free_[k].back();
                free_[k].pop_back();
                cached -= (size_t)1 << k;
                return p;
            }
        }
        return fresh((size_t)1 << k);
    }
    void put(void* p, size_t bytes) {
        if (!p) return;
        if (bytes >= ((size_t)1 << MIN_LOG) && bytes <= ((size_t)1 << MAX_LOG)) {
            const int k = size_class(bytes);
            {
                std::lock_guard<std::mutex> lk(mu);
                if (cached + ((size_t)1 << k) <= CACHE_CAP) {
                    free_[k].push_back(p);
                    cached += (size_t)1 << k;
                    return;
                }
            }
            release(p);
            return;
        }
        free(p);
    }
} HP;

template <class T>
struct PoolAlloc {
    using value_type = T;
    PoolAlloc() = default;
    template <class U> PoolAlloc(const PoolAlloc<U>&) {}
    T* allocate(size_t n) {
        void* p = HP.get(n * sizeof(T));
        if (!p) throw std::bad_alloc();
        return (T*)p;
    }
    void deallocate(T* p, size_t n) { HP.put(p, n * sizeof(T)); }
    // resize(n) leaves new elements uninitialised (every user writes all of them); resize(n, v) / assign still fill
    template <class U> void construct(U* p) noexcept { ::new ((void*)p) U; }
    template <class U, class... A> void construct(U* p, A&&... a) { ::new ((void*)p) U(std::forward<A>(a)...); }
    template <class U> bool operator==(const PoolAlloc<U>&) const { return true; }
    template <class U> bool operator!=(const PoolAlloc<U>&) const { return false; }
};
template <class T> using hvec = std::vector<T, PoolAlloc<T>>;

}  // namespace

// -----------------------------------------------------------------------------------------
// handles
// -----------------------------------------------------------------------------------------
struct pccl_topology {
    uint32_t N = 0, L = 0;
    std::vector<pccl_link_t> links;
    std::vector<uint32_t> in_off, in_link, out_off, out_link;   // ascending link id per node
    uint32_t max_in = 0, max_out = 0;                           // largest in- / out-degree
    // switch model of PAPER.md:348 (pccl_topology_set_switch_model); empty: none
    std::vector<uint32_t> buf_limit;
    std::vector<unsigned char> no_mcast;
    // device copy (one blob)
    void* blob = nullptr;
    uint32_t *d_src = nullptr, *d_dst = nullptr, *d_in_off = nullptr, *d_in_link = nullptr,
             *d_out_off = nullptr, *d_out_link = nullptr;
    // per entry of the out / in tables: the far end; per link: where the tables of its far node start
    uint32_t *d_out_far = nullptr, *d_in_far = nullptr, *d_lo_off_n = nullptr, *d_lo_deg_n = nullptr,
             *d_lo_off_t = nullptr, *d_lo_deg_t = nullptr;
    uint64_t *d_alpha = nullptr, *d_bpp = nullptr;
};

namespace {

struct Phase {
    bool transposed = false;          // run on the reversed links (reductions, Q10)
    hvec<uint32_t> cond_src;   // [C] source (copy) or root (reduce) of each chunk
    hvec<uint64_t> dest_off;   // [C+1]
    hvec<uint32_t> dests;      // ascending per chunk
    hvec<uint32_t> dchunk;     // [n_dests] chunk of each (chunk, dest) pair
    hvec<uint32_t> sources;    // distinct sources, ascending
    hvec<uint32_t> sidx;       // [N] node -> row of D, NONE32 if not a source
    hvec<uint32_t> dsts;       // distinct dests, ascending (dynamic relay: rows of the to-dest distances)
    hvec<uint32_t> didx;       // [N] node -> row, NONE32 if not a dest
    // c.dist-priority pick (PCCL_FLAG_DIST_PICK): this phase with its chunks RELABELLED in (descending c.dist, ascending
    // chunk id) order -- orig[c'] = the caller's chunk id, cls[c'] = index of its c.dist class (0 = farthest)
    hvec<uint32_t> orig, cls;
    uint32_t ncls = 0;
    uint32_t *d_orig = nullptr, *d_cls = nullptr;
    void* blob = nullptr;
    uint32_t *d_cond_src = nullptr, *d_dests = nullptr, *d_dchunk = nullptr, *d_sources = nullptr,
             *d_sidx = nullptr, *d_dsts = nullptr, *d_didx = nullptr;
    uint64_t* d_dest_off = nullptr;
};

}  // namespace

struct pccl_problem {
    const pccl_topology* topo = nullptr;
    uint32_t C = 0;
    uint64_t chunk_bytes = 0;
    int mode = 0;
    std::vector<Phase> phases;
    std::vector<Phase> prio_phases;   // the phases relabelled for PCCL_FLAG_DIST_PICK (built on first use)
    bool uploaded = false;
};

struct pccl_schedule {
    uint64_t M = 0, T = 0;
    uint32_t n_links = 0, n_npus = 0;
    Rec* d_recs = nullptr;
    void* h_recs = nullptr;
    size_t h_bytes = 0;
    bool downloaded = false;
    pccl_stats_t stats;
    std::vector<uint64_t> trace;   // PCCL_FLAG_TRACE: [events][TRACE_SLOTS] ns stamps of the last phase
};

// -----------------------------------------------------------------------------------------
// plumbing entry points
// -----------------------------------------------------------------------------------------
extern "C" void pccl_set_stream(void* s) { G.stream = (cudaStream_t)s; }
extern "C" void pccl_set_allocator(pccl_alloc_fn a, pccl_free_fn f, void* user) {
    if (a && f) { G.alloc = a; G.release = f; G.user = user; }
    else { G.alloc = nullptr; G.release = nullptr; G.user = nullptr; }
}
extern "C" int pccl_version(void) { return PCCL_VERSION; }
extern "C" uint64_t pccl_launch_count(void) { return G.launches.load(std::memory_order_relaxed); }
extern "C" int pccl_set_option(int option, uint64_t value) {
    switch (option) {
        case PCCL_OPT_BFS_WINDOW: G.opt_bfs_window = value; return PCCL_OK;
        case PCCL_OPT_BFS_ROWS: G.opt_bfs_rows = value; return PCCL_OK;
        case PCCL_OPT_DYNAMIC_RECORDS: G.opt_dyn_records = value; return PCCL_OK;
        default: return PCCL_ERR_INVALID;
    }
}
extern "C" uint64_t pccl_get_option(int option) {
    switch (option) {
        case PCCL_OPT_BFS_WINDOW: return G.opt_bfs_window;
        case PCCL_OPT_BFS_ROWS: return G.opt_bfs_rows;
        case PCCL_OPT_DYNAMIC_RECORDS: return G.opt_dyn_records;
        default: return 0;
    }
}
extern "C" const char* pccl_strerror(int err) {
    switch (err) {
        case PCCL_OK: return "ok";
        case PCCL_ERR_INVALID: return "invalid argument";
        case PCCL_ERR_UNSUPPORTED: return "unsupported problem (mixed copy/reduction chunks or size limit)";
        case PCCL_ERR_UNREACHABLE: return "a destination is unreachable from its chunk's source";
        case PCCL_ERR_CUDA: return "CUDA failure (no device, launch or copy error)";
        case PCCL_ERR_NOMEM: return "out of memory";
        case PCCL_ERR_INTERNAL: return "internal invariant violated";
        case PCCL_ERR_TOO_LARGE: return "problem exceeds the fixed scratch of the no-allocation entry point (PCCL_STATIC_SCRATCH_BYTES)";
        default: return "unknown error";
    }
}

// -----------------------------------------------------------------------------------------
// topology store
// -----------------------------------------------------------------------------------------
extern "C" int pccl_topology_create(uint32_t n_npus, const pccl_link_t* links, uint32_t n_links,
                                    pccl_topology_t** out) {
    if (!out || (n_links && !links)) return PCCL_ERR_INVALID;
    for (uint32_t l = 0; l < n_links; ++l) {
        const pccl_link_t& k = links[l];
        if (k.src >= n_npus || k.dst >= n_npus || k.src == k.dst || k.bytes_per_ps == 0) return PCCL_ERR_INVALID;
    }
    pccl_topology* t = new (std::nothrow) pccl_topology();
    if (!t) return PCCL_ERR_NOMEM;
    try {
        t->N = n_npus;
        t->L = n_links;
        t->links.assign(links, links + n_links);
        t->in_off.assign((size_t)n_npus + 1, 0);
        t->out_off.assign((size_t)n_npus + 1, 0);
        for (uint32_t l = 0; l < n_links; ++l) { ++t->in_off[links[l].dst + 1]; ++t->out_off[links[l].src + 1]; }
        for (uint32_t v = 0; v < n_npus; ++v) {
            t->max_in = std::max(t->max_in, t->in_off[v + 1]);
            t->max_out = std::max(t->max_out, t->out_off[v + 1]);
            t->in_off[v + 1] += t->in_off[v];
            t->out_off[v + 1] += t->out_off[v];
        }
        t->in_link.resize(n_links);
        t->out_link.resize(n_links);
        std::vector<uint32_t> ci(t->in_off.begin(), t->in_off.end() - 1), co(t->out_off.begin(), t->out_off.end() - 1);
        for (uint32_t l = 0; l < n_links; ++l) {   // ascending l => each node's list is ascending
            t->in_link[ci[links[l].dst]++] = l;
            t->out_link[co[links[l].src]++] = l;
        }
    } catch (const std::bad_alloc&) {
        delete t;
        return PCCL_ERR_NOMEM;
    }
    *out = t;
    return PCCL_OK;
}

extern "C" int pccl_topology_set_switch_model(pccl_topology_t* t, const uint32_t* buffer_limit, const uint8_t* no_multicast) {
    SERIALISE;
    if (!t) return PCCL_ERR_INVALID;
    try {
        std::vector<uint32_t> bl;
        std::vector<unsigned char> nm;
        bool any = false;
        if (buffer_limit) for (uint32_t v = 0; v < t->N; ++v) any |= buffer_limit[v] != 0xFFFFFFFFu;
        if (no_multicast) for (uint32_t v = 0; v < t->N; ++v) any |= no_multicast[v] != 0;
        if (any) {
            bl.assign(t->N, 0xFFFFFFFFu);
            nm.assign(t->N, 0);
            if (buffer_limit) bl.assign(buffer_limit, buffer_limit + t->N);
            if (no_multicast) nm.assign(no_multicast, no_multicast + t->N);
        }
        t->buf_limit.swap(bl);
        t->no_mcast.swap(nm);
    } catch (const std::bad_alloc&) {
        return PCCL_ERR_NOMEM;
    }
    return PCCL_OK;
}

extern "C" void pccl_topology_destroy(pccl_topology_t* t) {
    SERIALISE;
    if (!t) return;
    dev_free(t->blob);
    delete t;
}
extern "C" uint32_t pccl_topology_n_npus(const pccl_topology_t* t) { return t ? t->N : 0; }
extern "C" uint32_t pccl_topology_n_links(const pccl_topology_t* t) { return t ? t->L : 0; }

namespace {

// carve a blob: returns offset, advances cursor (256-byte aligned pieces)
struct Carver {
    size_t cur = 0;
    size_t take(size_t bytes) { const size_t o = cur; cur = align_up(cur + bytes, 256); return o; }
};

int topo_upload(pccl_topology* t) {
    if (t->blob) return PCCL_OK;
    int rc = ensure_device();
    if (rc) return rc;
    const size_t N = t->N, L = t->L;
    Carver c;
    const size_t o_src = c.take(L * 4), o_dst = c.take(L * 4), o_alpha = c.take(L * 8), o_bpp = c.take(L * 8),
                 o_ino = c.take((N + 1) * 4), o_inl = c.take(L * 4), o_outo = c.take((N + 1) * 4), o_outl = c.take(L * 4),
                 o_of = c.take(L * 4), o_if = c.take(L * 4), o_lon = c.take(L * 4), o_ldn = c.take(L * 4),
                 o_lot = c.take(L * 4), o_ldt = c.take(L * 4);
    std::vector<unsigned char> h;
    try {
        h.assign(c.cur ? c.cur : 256, 0);
    } catch (const std::bad_alloc&) {
        return PCCL_ERR_NOMEM;
    }
    for (size_t l = 0; l < L; ++l) {
        ((uint32_t*)(h.data() + o_src))[l] = t->links[l].src;
        ((uint32_t*)(h.data() + o_dst))[l] = t->links[l].dst;
        ((uint64_t*)(h.data() + o_alpha))[l] = t->links[l].alpha_ps;
        ((uint64_t*)(h.data() + o_bpp))[l] = t->links[l].bytes_per_ps;
    }
    memcpy(h.data() + o_ino, t->in_off.data(), (N + 1) * 4);
    memcpy(h.data() + o_outo, t->out_off.data(), (N + 1) * 4);
    if (L) {
        memcpy(h.data() + o_inl, t->in_link.data(), L * 4);
        memcpy(h.data() + o_outl, t->out_link.data(), L * 4);
    }
    for (size_t e = 0; e < L; ++e) {
        ((uint32_t*)(h.data() + o_of))[e] = t->links[t->out_link[e]].dst;
        ((uint32_t*)(h.data() + o_if))[e] = t->links[t->in_link[e]].src;
    }
    for (size_t l = 0; l < L; ++l) {
        const uint32_t d = t->links[l].dst, sN = t->links[l].src;
        ((uint32_t*)(h.data() + o_lon))[l] = t->out_off[d];
        ((uint32_t*)(h.data() + o_ldn))[l] = t->out_off[d + 1] - t->out_off[d];
        ((uint32_t*)(h.data() + o_lot))[l] = t->in_off[sN];          // transposed view: far node = src, its "out" = in
        ((uint32_t*)(h.data() + o_ldt))[l] = t->in_off[sN + 1] - t->in_off[sN];
    }
    void* blob = nullptr;
    rc = dev_alloc(h.size(), &blob);
    if (rc) return rc;
    if (cudaMemcpyAsync(blob, h.data(), h.size(), cudaMemcpyHostToDevice, G.stream) != cudaSuccess ||
        cudaStreamSynchronize(G.stream) != cudaSuccess) {
        (void)cudaGetLastError();
        dev_free(blob);
        return PCCL_ERR_CUDA;
    }
    unsigned char* b = (unsigned char*)blob;
    t->blob = blob;
    t->d_out_far = (uint32_t*)(b + o_of); t->d_in_far = (uint32_t*)(b + o_if);
    t->d_lo_off_n = (uint32_t*)(b + o_lon); t->d_lo_deg_n = (uint32_t*)(b + o_ldn);
    t->d_lo_off_t = (uint32_t*)(b + o_lot); t->d_lo_deg_t = (uint32_t*)(b + o_ldt);
    t->d_src = (uint32_t*)(b + o_src); t->d_dst = (uint32_t*)(b + o_dst);
    t->d_alpha = (uint64_t*)(b + o_alpha); t->d_bpp = (uint64_t*)(b + o_bpp);
    t->d_in_off = (uint32_t*)(b + o_ino); t->d_in_link = (uint32_t*)(b + o_inl);
    t->d_out_off = (uint32_t*)(b + o_outo); t->d_out_link = (uint32_t*)(b + o_outl);
    return PCCL_OK;
}

// ---------------------------------------------------------------------------------------
// step R: NPU-centric pre/postcondition -> chunk-centric conditions
// (PAPER.md:170-172); |pre(c)| > 1 marks a reduction chunk (Q12).
// ---------------------------------------------------------------------------------------
// per-chunk ascending, duplicate-free NPU lists
int group_pairs(const pccl_condition_t* cnd, uint32_t C, uint32_t N, const std::vector<char>& member,
                hvec<uint64_t>& off, hvec<uint32_t>& npus) {
    off.assign((size_t)C + 1, 0);
    npus.resize(cnd->n_pairs);
    bool ordered = true;   // chunk ids non-decreasing in the caller's array: the pairs are already grouped
    uint32_t prev = 0;
    const char* mem = member.data();
    for (uint64_t i = 0; i < cnd->n_pairs; ++i) {
        const pccl_pair_t p = cnd->pairs[i];
        if (p.chunk >= C || p.npu >= N || !mem[p.npu]) return PCCL_ERR_INVALID;
        ++off[p.chunk + 1];
        ordered &= p.chunk >= prev;
        prev = p.chunk;
        npus[i] = p.npu;
    }
    uint64_t longest = 0;
    for (uint32_t c = 0; c < C; ++c) { longest = std::max(longest, off[c + 1]); off[c + 1] += off[c]; }
    if (!ordered) {
        hvec<uint64_t> cur(off.begin(), off.end() - 1);
        for (uint64_t i = 0; i < cnd->n_pairs; ++i) npus[cur[cnd->pairs[i].chunk]++] = cnd->pairs[i].npu;
    }
    if (longest <= 1) return PCCL_OK;   // every list has at most one holder: already sorted and duplicate-free
    // sort each list; compact only if a duplicate shows up
    bool dup = false;
    for (uint32_t c = 0; c < C; ++c) {
        uint32_t* b = npus.data() + off[c];
        uint32_t* e = npus.data() + off[c + 1];
        if (e - b > 1) {
            std::sort(b, e);
            dup |= std::adjacent_find(b, e) != e;
        }
    }
    if (!dup) return PCCL_OK;
    uint64_t w = 0, rd = 0;
    for (uint32_t c = 0; c < C; ++c) {
        const uint64_t end = off[c + 1];
        off[c] = w;
        for (uint64_t i = rd; i < end; ++i)
            if (i == rd || npus[i] != npus[i - 1]) npus[w++] = npus[i];
        rd = end;
    }
    off[C] = w;
    npus.resize(w);
    return PCCL_OK;
}

// distinct sources / dests (ascending) and their row indices, from per-node flags
void index_phase(Phase& ph, uint32_t N, const std::vector<char>& is_src, const std::vector<char>& is_dst) {
    ph.sidx.assign(N, NONE32);
    for (uint32_t v = 0; v < N; ++v)
        if (is_src[v]) { ph.sidx[v] = (uint32_t)ph.sources.size(); ph.sources.push_back(v); }
    ph.didx.assign(N, NONE32);
    for (uint32_t v = 0; v < N; ++v)
        if (is_dst[v]) { ph.didx[v] = (uint32_t)ph.dsts.size(); ph.dsts.push_back(v); }
}

void finish_phase(Phase& ph, uint32_t N) {
    const uint32_t C = (uint32_t)ph.cond_src.size();
    ph.dchunk.resize(ph.dests.size());
    std::vector<char> is_src(N, 0), is_dst(N, 0);
    for (uint32_t c = 0; c < C; ++c) {
        for (uint64_t i = ph.dest_off[c]; i < ph.dest_off[c + 1]; ++i) ph.dchunk[i] = c;
        if (ph.dest_off[c + 1] > ph.dest_off[c]) is_src[ph.cond_src[c]] = 1;
    }
    for (uint32_t d : ph.dests) is_dst[d] = 1;
    index_phase(ph, N, is_src, is_dst);
}

// A few host threads kept for the life of the process (the normaliser's passes over millions of pairs).
// parallel_for(n, f) runs f(0) .. f(n-1), each once: the caller and whichever workers are awake CLAIM indices from a
// shared counter, and the call returns when every claimed index is done.  Nobody ever waits for a worker to wake up: on
// the GPU box (a VM) a condition-variable wake-up took up to a millisecond, which the earlier one-slice-per-thread form
// paid on every call (normalise 0.24 ms or 1.1 ms at config 4, depending on the run); a worker that wakes late finds
// nothing left to claim and goes back to sleep.  After a job a worker polls for the next one for a short while (the
// normaliser's second pass follows its first within microseconds) before it sleeps.
class HostPool2 {
    struct Job {
        std::function<void(int)> fn;
        int n = 0;
        std::atomic<int> next{0}, done{0};
    };
    std::vector<std::thread> th_;
    std::mutex mu_;
    std::condition_variable cv_;
    std::shared_ptr<Job> job_;                 // (kept alive by every worker that holds it: a late one only reads next/n)
    std::atomic<uint64_t> gen_{0};
    bool stop_ = false;
    static void drain(Job& j) {
        for (;;) {
            const int i = j.next.fetch_add(1, std::memory_order_relaxed);
            if (i >= j.n) return;
            j.fn(i);
            j.done.fetch_add(1, std::memory_order_release);
        }
    }
    void worker() {
        uint64_t seen = 0;
        for (;;) {
            std::shared_ptr<Job> j;
            for (int spin = 0; spin < 2000 && gen_.load(std::memory_order_acquire) == seen; ++spin) cpu_relax_();
            {
                std::unique_lock<std::mutex> lk(mu_);
                cv_.wait(lk, [&] { return stop_ || gen_.load(std::memory_order_relaxed) != seen; });
                if (stop_) return;
                seen = gen_.load(std::memory_order_relaxed);
                j = job_;
            }
            if (j) drain(*j);
        }
    }
    static void cpu_relax_() {
#if defined(__x86_64__)
        _mm_pause();
#else
        std::this_thread::yield();
#endif
    }
public:
    static constexpr int MAX_THREADS = 8;
    int capacity() {
        std::lock_guard<std::mutex> lk(mu_);
        if (th_.empty()) {
            const int hw = (int)std::thread::hardware_concurrency();
            const int n = std::max(1, std::min(MAX_THREADS, hw / 2));
            try {
                for (int i = 1; i < n; ++i) th_.emplace_back([this] { worker(); });
            } catch (const std::system_error&) {
            }
        }
        return (int)th_.size() + 1;
    }
    void parallel_for(int n, const std::function<void(int)>& f) {
        if (n <= 0) return;
        if (n == 1 || capacity() == 1) {
            for (int i = 0; i < n; ++i) f(i);
            return;
        }
        std::shared_ptr<Job> j = std::make_shared<Job>();
        j->fn = f; j->n = n;
        {
            std::lock_guard<std::mutex> lk(mu_);
            job_ = j;
            gen_.fetch_add(1, std::memory_order_release);
        }
        cv_.notify_all();
        drain(*j);
        while (j->done.load(std::memory_order_acquire) < n) cpu_relax_();   // indices claimed by workers that are running
        std::lock_guard<std::mutex> lk(mu_);
        if (job_ == j) job_.reset();
    }
    ~HostPool2() {
        {
            std::lock_guard<std::mutex> lk(mu_);
            stop_ = true;
        }
        cv_.notify_all();
        for (auto& t : th_) t.join();
    }
};
HostPool2 g_threads;
std::mutex g_threads_mu;   // one parallel region at a time

// stores that bypass the caches (x86-64: movnti), for arrays written once, front to back, and read next by DMA
#if defined(__x86_64__)
inline void nt_store32(uint32_t* p, uint32_t v) { _mm_stream_si32((int*)p, (int)v); }
inline void nt_store64(uint64_t* p, uint64_t v) { _mm_stream_si64((long long*)p, (long long)v); }
inline void nt_fence() { _mm_sfence(); }
inline void cpu_relax() { _mm_pause(); }
#else
inline void cpu_relax() { std::this_thread::yield(); }
inline void nt_store32(uint32_t* p, uint32_t v) { *p = v; }
inline void nt_store64(uint64_t* p, uint64_t v) { *p = v; }
inline void nt_fence() {}
#endif

// The common large case straight from the caller's arrays: both pair lists already ordered by chunk, exactly one
// pre-holder per chunk (COPY mode), post-holders of a chunk strictly ascending.  Returns false on ANY deviation
// (including invalid input) without touching P: the general path below then decides, errors included.
// Two passes over slices of the chunk range, one slice per host thread: count and validate, then write at the offsets
// the counts give.  A slice starts at the first post pair whose chunk is >= its first chunk (binary search, right if
// the list is ordered) and must end exactly where the next slice starts -- together with the pair-by-pair check inside
// a slice that proves the order the search assumed.
bool normalise_ordered_copy(const pccl_condition_t* pre, const pccl_condition_t* post, uint32_t C, uint32_t N,
                            const std::vector<char>& member, Phase& cp) {
    if (pre->n_pairs != C || post->n_pairs < C) return false;
    const pccl_pair_t* __restrict__ pp = pre->pairs;
    const pccl_pair_t* __restrict__ qp = post->pairs;
    const uint64_t nq = post->n_pairs;
    const char* mem = member.data();
    std::unique_lock<std::mutex> region(g_threads_mu, std::defer_lock);
    int T = 1;                                                     // slices of the chunk range (>= 2^13 post pairs each)
    if (nq >= (1u << 15)) {
        region.lock();
        if (g_threads.capacity() > 1) T = (int)std::min<uint64_t>(64, nq >> 13);
    }
    struct Slice {
        uint32_t c_lo, c_hi;
        uint64_t k_lo, k_end, nd;
        bool ok;
    };
    std::vector<Slice> sl((size_t)T);
    for (int t = 0; t < T; ++t) {
        sl[t].c_lo = (uint32_t)((uint64_t)C * t / T);
        sl[t].c_hi = (uint32_t)((uint64_t)C * (t + 1) / T);
        sl[t].ok = false;
    }
    // marks "is a source" / "is a destination", shared by the slices (every store writes 1: relaxed atomic byte stores)
    std::vector<unsigned char> f_src(N, 0), f_dst(N, 0);
    unsigned char* fs = f_src.data();
    unsigned char* fd = f_dst.data();
    // pass 1: validate, count the destinations (post-holders other than the source), mark sources and destinations
    const std::function<void(int)> pass1 = [&](int t) {
        Slice& s = sl[t];
        uint64_t lo = 0, hi = nq;                                  // first pair with chunk >= c_lo
        while (lo < hi) {
            const uint64_t mid = (lo + hi) >> 1;
            if (qp[mid].chunk < s.c_lo) lo = mid + 1; else hi = mid;
        }
        s.k_lo = lo;
        uint64_t k = lo, nd = 0;
        for (uint32_t c = s.c_lo; c < s.c_hi; ++c) {
            const pccl_pair_t a = pp[c];
            if (a.chunk != c || a.npu >= N || !mem[a.npu]) return;
            const uint32_t src = a.npu;
            if (k >= nq || qp[k].chunk != c) return;               // no post-holder, or not ordered
            const uint64_t first = nd;
            uint32_t prev = 0;
            bool have_prev = false;
            while (k < nq && qp[k].chunk == c) {
                const uint32_t d = qp[k].npu;
                if (d >= N || !mem[d] || (have_prev && d <= prev)) return;
                prev = d;
                have_prev = true;
                ++k;
                if (d == src) continue;
                if (!__atomic_load_n(fd + d, __ATOMIC_RELAXED)) __atomic_store_n(fd + d, (unsigned char)1, __ATOMIC_RELAXED);
                ++nd;
            }
            if (nd > first && !__atomic_load_n(fs + src, __ATOMIC_RELAXED)) __atomic_store_n(fs + src, (unsigned char)1, __ATOMIC_RELAXED);
        }
        s.k_end = k;
        s.nd = nd;
        s.ok = true;
    };
    g_threads.parallel_for(T, pass1);
    // between the passes: the slices must tile the list; size the arrays, hand out the offsets
    std::vector<uint64_t> nd_base((size_t)T, 0);
    uint64_t nd_total = 0;
    for (int t = 0; t < T; ++t) {
        if (!sl[t].ok) return false;
        if (sl[t].k_lo != (t == 0 ? 0 : sl[t - 1].k_end)) return false;
        nd_base[t] = nd_total;
        nd_total += sl[t].nd;
    }
    if (sl[T - 1].k_end != nq) return false;                     // pairs of a chunk id >= C, or out of order
    cp.cond_src.resize(C);                                       // (std::bad_alloc is the caller's to turn into NOMEM)
    cp.dest_off.resize((size_t)C + 1);
    cp.dests.resize(nd_total);
    cp.dchunk.resize(nd_total);
    uint32_t* o_src = cp.cond_src.data();
    uint64_t* o_off = cp.dest_off.data();
    uint32_t* o_dst = cp.dests.data();
    uint32_t* o_chk = cp.dchunk.data();
    o_off[0] = 0;
    // pass 2: write (everything was validated).  The four arrays go to the device next, by DMA from these very
    // (page-locked) blocks: non-temporal stores put them in memory instead of leaving dirty lines in the caches of
    // whichever cores the slices ran on (measured on the B200 host: DMA of lines that sit modified in other cores'
    // caches ran at 7 GB/s instead of 55).
    const std::function<void(int)> pass2 = [&](int t) {
        const Slice& s = sl[t];
        uint64_t k = s.k_lo, nd = nd_base[t];
        for (uint32_t c = s.c_lo; c < s.c_hi; ++c) {
            const uint32_t src = pp[c].npu;
            while (k < nq && qp[k].chunk == c) {
                const uint32_t d = qp[k].npu;
                ++k;
                if (d == src) continue;
                nt_store32(o_dst + nd, d);
                nt_store32(o_chk + nd, c);
                ++nd;
            }
            nt_store32(o_src + c, src);
            nt_store64(o_off + c + 1, nd);
        }
        nt_fence();
    };
    g_threads.parallel_for(T, pass2);
    std::vector<char> f_src_c(N, 0), f_dst_c(N, 0);
    for (uint32_t v = 0; v < N; ++v) { f_src_c[v] = (char)f_src[v]; f_dst_c[v] = (char)f_dst[v]; }
    index_phase(cp, N, f_src_c, f_dst_c);
    return true;
}

int normalise(const pccl_topology* topo, const uint32_t* group, uint32_t n_members,
              const pccl_condition_t* pre, const pccl_condition_t* post, uint64_t chunk_bytes,
              pccl_problem& P) {
    if (!topo || !pre || !post || (n_members && !group)) return PCCL_ERR_INVALID;
    if ((pre->n_pairs && !pre->pairs) || (post->n_pairs && !post->pairs)) return PCCL_ERR_INVALID;
    if (chunk_bytes == 0 || pre->n_chunks != post->n_chunks) return PCCL_ERR_INVALID;
    const uint32_t N = topo->N, C = pre->n_chunks;
    std::vector<char> member(N, 0);
    for (uint32_t i = 0; i < n_members; ++i) {
        if (group[i] >= N || member[group[i]]) return PCCL_ERR_INVALID;
        member[group[i]] = 1;
    }
    if (C > 0) {
        Phase cp;
        if (normalise_ordered_copy(pre, post, C, N, member, cp)) {
            P.topo = topo;
            P.C = C;
            P.chunk_bytes = chunk_bytes;
            P.mode = 0;
            P.phases.clear();
            P.phases.push_back(std::move(cp));
            return PCCL_OK;
        }
    }
    hvec<uint64_t> pre_off, post_off;
    hvec<uint32_t> pre_n, post_n;
    // the two conditions are grouped independently: the postcondition on a second host thread when it is large
    int rc, rc2;
    if (post->n_pairs >= 65536) {
        std::future<int> fut;
        bool threaded = true;
        try {
            fut = std::async(std::launch::async, [&] { return group_pairs(post, C, N, member, post_off, post_n); });
        } catch (const std::system_error&) {
            threaded = false;
        }
        rc = group_pairs(pre, C, N, member, pre_off, pre_n);
        rc2 = threaded ? fut.get() : group_pairs(post, C, N, member, post_off, post_n);
    } else {
        rc = group_pairs(pre, C, N, member, pre_off, pre_n);
        rc2 = group_pairs(post, C, N, member, post_off, post_n);
    }
    if (rc) return rc;
    if (rc2) return rc2;
    // one pass classifies the call (Q12) and, as long as every chunk so far has a single pre-holder, already writes
    // the COPY conditions -- the common large case (All-to-All(v), All-Gather) needs no second sweep
    bool all_single = true, all_multi_one = true, all_multi_many = true;
    Phase cp;
    cp.cond_src.resize(C);
    cp.dest_off.resize((size_t)C + 1);
    cp.dests.resize(post_n.size());
    cp.dchunk.resize(post_n.size());
    cp.dest_off[0] = 0;
    std::vector<uint32_t> cp_src32(N, 0), cp_dst32(N, 0);
    uint64_t nd = 0;
    {
        // raw restrict pointers: the arrays are distinct (the pass is bound by one core's streaming rate either way)
        const uint64_t* __restrict__ po = pre_off.data();
        const uint64_t* __restrict__ qo = post_off.data();
        const uint32_t* __restrict__ pn = pre_n.data();
        const uint32_t* __restrict__ qn = post_n.data();
        uint32_t* __restrict__ o_src = cp.cond_src.data();
        uint64_t* __restrict__ o_off = cp.dest_off.data();
        uint32_t* __restrict__ o_dst = cp.dests.data();
        uint32_t* __restrict__ o_chk = cp.dchunk.data();
        uint32_t* __restrict__ f_src = cp_src32.data();
        uint32_t* __restrict__ f_dst = cp_dst32.data();
        for (uint32_t c = 0; c < C; ++c) {
            const uint64_t pb = po[c], np = po[c + 1] - pb, qb = qo[c], qe = qo[c + 1], nq = qe - qb;
            if (np == 0 || nq == 0) return PCCL_ERR_INVALID;
            const bool single = np == 1;
            all_single &= single;
            all_multi_one &= (!single && nq == 1);
            all_multi_many &= (!single && nq > 1);
            if (all_single) {
                const uint32_t src = pn[pb];
                const uint64_t first = nd;
                o_src[c] = src;
                for (uint64_t i = qb; i < qe; ++i) {
                    const uint32_t d = qn[i];
                    if (d == src) continue;
                    o_dst[nd] = d;
                    o_chk[nd] = c;
                    f_dst[d] = 1;
                    ++nd;
                }
                o_off[c + 1] = nd;
                if (nd > first) f_src[src] = 1;
            }
        }
    }
    std::vector<char> cp_src(cp_src32.begin(), cp_src32.end()), cp_dst(cp_dst32.begin(), cp_dst32.end());
    P.topo = topo;
    P.C = C;
    P.chunk_bytes = chunk_bytes;
    P.phases.clear();
    auto fill = [&](Phase& ph, uint32_t c, uint32_t src, const uint32_t* b, const uint32_t* e) {
        ph.cond_src[c] = src;
        for (const uint32_t* p = b; p != e; ++p) if (*p != src) ph.dests.push_back(*p);
        ph.dest_off[c + 1] = ph.dests.size();
    };
    if (all_single) {   // COPY: the one pre-holder is the source
        P.mode = 0;
        cp.dests.resize(nd);
        cp.dchunk.resize(nd);
        index_phase(cp, N, cp_src, cp_dst);
        P.phases.push_back(std::move(cp));
        return PCCL_OK;
    } else if (all_multi_one) {   // REDUCE: broadcast root -> holders on the transposed links
        P.mode = 1;
        P.phases.resize(1);
        Phase& ph = P.phases[0];
        ph.transposed = true;
        ph.cond_src.resize(C);
        ph.dest_off.assign((size_t)C + 1, 0);
        for (uint32_t c = 0; c < C; ++c)
            fill(ph, c, post_n[post_off[c]], pre_n.data() + pre_off[c], pre_n.data() + pre_off[c + 1]);
    } else if (all_multi_many) {   // ALL-REDUCE = reduce to root(c), then copy from root(c)
        P.mode = 2;
        P.phases.resize(2);
        Phase &r = P.phases[0], &g = P.phases[1];
        r.transposed = true;
        r.cond_src.resize(C); g.cond_src.resize(C);
        r.dest_off.assign((size_t)C + 1, 0); g.dest_off.assign((size_t)C + 1, 0);
        std::vector<uint32_t> I;
        for (uint32_t c = 0; c < C; ++c) {
            const uint32_t *pb = pre_n.data() + pre_off[c], *pe = pre_n.data() + pre_off[c + 1];
            const uint32_t *qb = post_n.data() + post_off[c], *qe = post_n.data() + post_off[c + 1];
            I.clear();
            std::set_intersection(pb, pe, qb, qe, std::back_inserter(I));
            if (I.empty()) I.assign(qb, qe);
            const uint32_t root = I[c % I.size()];
            fill(r, c, root, pb, pe);
            fill(g, c, root, qb, qe);
        }
    } else {
        return PCCL_ERR_UNSUPPORTED;
    }
    for (Phase& ph : P.phases) finish_phase(ph, N);
    return PCCL_OK;
}

int phase_upload(Phase& ph, uint32_t N, bool sync = true) {
    if (ph.blob) return PCCL_OK;
    const size_t C = ph.cond_src.size(), ND = ph.dests.size(), NS = ph.sources.size();
    Carver c;
    const size_t o_cs = c.take(C * 4), o_d = c.take(ND * 4), o_dc = c.take(ND * 4), o_s = c.take(NS * 4), o_si = c.take((size_t)N * 4);
    const size_t NDS = ph.dsts.size();
    const size_t o_do = c.take((C + 1) * 8), o_ds = c.take(NDS * 4), o_di = c.take((size_t)N * 4);
    const size_t o_or = c.take(ph.orig.size() * 4), o_cl = c.take(ph.cls.size() * 4);
    // copied straight from the normaliser's arrays (pooled, page-locked when a device is there): no staging pass
    void* blob = nullptr;
    int rc = dev_alloc(c.cur ? c.cur : 256, &blob);
    if (rc) return rc;
    unsigned char* d = (unsigned char*)blob;
    cudaError_t e = cudaSuccess;
    auto up = [&](size_t off, const void* src, size_t bytes) {
        if (bytes && e == cudaSuccess) e = cudaMemcpyAsync(d + off, src, bytes, cudaMemcpyHostToDevice, G.stream);
    };
    up(o_do, ph.dest_off.data(), (C + 1) * 8);
    up(o_ds, ph.dsts.data(), NDS * 4);
    up(o_di, ph.didx.data(), (size_t)N * 4);
    up(o_cs, ph.cond_src.data(), C * 4);
    up(o_d, ph.dests.data(), ND * 4);
    up(o_dc, ph.dchunk.data(), ND * 4);
    up(o_s, ph.sources.data(), NS * 4);
    up(o_si, ph.sidx.data(), (size_t)N * 4);
    up(o_or, ph.orig.data(), ph.orig.size() * 4);
    up(o_cl, ph.cls.data(), ph.cls.size() * 4);
    // (sync == false: the caller's next work is on the same stream and it synchronises before the arrays can go away)
    if (e == cudaSuccess && sync) e = cudaStreamSynchronize(G.stream);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        (void)cudaStreamSynchronize(G.stream);
        (void)cudaGetLastError();
        dev_free(blob);
        return PCCL_ERR_CUDA;
    }
    unsigned char* b = (unsigned char*)blob;
    ph.blob = blob;
    ph.d_cond_src = (uint32_t*)(b + o_cs); ph.d_dests = (uint32_t*)(b + o_d); ph.d_dchunk = (uint32_t*)(b + o_dc);
    ph.d_sources = (uint32_t*)(b + o_s); ph.d_sidx = (uint32_t*)(b + o_si);
    ph.d_dest_off = (uint64_t*)(b + o_do); ph.d_dsts = (uint32_t*)(b + o_ds); ph.d_didx = (uint32_t*)(b + o_di);
    ph.d_orig = ph.orig.empty() ? nullptr : (uint32_t*)(b + o_or);
    ph.d_cls = ph.cls.empty() ? nullptr : (uint32_t*)(b + o_cl);
    return PCCL_OK;
}

}  // namespace

extern "C" int pccl_problem_create(const pccl_topology_t* topo, const uint32_t* group_members,
                                   uint32_t n_members, const pccl_condition_t* pre,
                                   const pccl_condition_t* post, uint64_t chunk_bytes,
                                   pccl_problem_t** out) {
    if (!out) return PCCL_ERR_INVALID;
    pccl_problem* P = new (std::nothrow) pccl_problem();
    if (!P) return PCCL_ERR_NOMEM;
    int rc;
    try {
        rc = normalise(topo, group_members, n_members, pre, post, chunk_bytes, *P);
    } catch (const std::bad_alloc&) {
        rc = PCCL_ERR_NOMEM;
    }
    if (rc) { delete P; return rc; }
    *out = P;
    return PCCL_OK;
}

extern "C" void pccl_problem_destroy(pccl_problem_t* P) {
    SERIALISE;
    if (!P) return;
    for (Phase& ph : P->phases) dev_free(ph.blob);
    for (Phase& ph : P->prio_phases) dev_free(ph.blob);
    delete P;
}

// sync == false: the copies are only enqueued (from the problem's own page-locked arrays); the caller goes on working
// on the same stream and synchronises it before it returns
static int problem_upload(pccl_problem_t* P, bool sync) {
    SERIALISE;
    if (!P) return PCCL_ERR_INVALID;
    if (P->uploaded) return PCCL_OK;
    int rc = topo_upload(const_cast<pccl_topology*>(P->topo));
    if (rc) return rc;
    try {
        for (Phase& ph : P->phases) { rc = phase_upload(ph, P->topo->N, sync); if (rc) return rc; }
    } catch (const std::bad_alloc&) {
        return PCCL_ERR_NOMEM;
    }
    P->uploaded = true;
    return PCCL_OK;
}
extern "C" int pccl_problem_upload(pccl_problem_t* P) { return problem_upload(P, true); }

extern "C" int pccl_problem_mode(const pccl_problem_t* P) { return P ? P->mode : PCCL_ERR_INVALID; }
extern "C" uint32_t pccl_problem_n_chunks(const pccl_problem_t* P) { return P ? P->C : 0; }
extern "C" int64_t pccl_problem_condition(const pccl_problem_t* P, uint32_t phase, uint32_t chunk,
                                          uint32_t* src, uint32_t* dests, uint64_t cap) {
    if (!P || phase >= P->phases.size() || chunk >= P->C) return PCCL_ERR_INVALID;
    const Phase& ph = P->phases[phase];
    if (src) *src = ph.cond_src[chunk];
    const uint64_t b = ph.dest_off[chunk], e = ph.dest_off[chunk + 1];
    for (uint64_t i = b; i < e && (i - b) < cap && dests; ++i) dests[i - b] = ph.dests[i];
    return (int64_t)(e - b);
}

// -----------------------------------------------------------------------------------------
// one phase on the device: steps A..E (setup kernels + the persistent event loop)
// -----------------------------------------------------------------------------------------
namespace {

struct Work {   // device workspace of one phase
    void* blob = nullptr;
    uint64_t *w = nullptr, *D = nullptr, *have = nullptr, *wants = nullptr, *free_t = nullptr, *matchbits = nullptr;
    uint32_t *wants_cnt = nullptr, *inflight = nullptr, *have_epoch = nullptr, *empty_epoch = nullptr;
    LoopCtrl* ctrl = nullptr;
    uint64_t *hsum = nullptr, *wsum = nullptr;
    uint32_t *gcnt = nullptr, *gtot = nullptr;
    uint64_t* best = nullptr;
    uint32_t *hold_cnt = nullptr, *hold = nullptr;   // dynamic rule with kept counts: holders of each chunk
    uint32_t* drow = nullptr;                        // dynamic rule: Dto row of each (chunk, dest) pair
    uint64_t* st_free = nullptr;
    uint32_t* st_inf = nullptr;
    uint32_t Wp = 0, S = 0, nLw = 0, SWp = 0;
    size_t zero_off = 0, zero_bytes = 0;   // have + wants + wants_cnt + ctrl are cleared per run
    // barrier-free loop (pccl_loop2.cuh): plan arrays and its control block; the large arrays are allocated per phase
    unsigned long long *nbase = nullptr, *poff = nullptr, *loff = nullptr;
    uint32_t* soff = nullptr;
    A2Ctrl* a2ctrl = nullptr;
    bool a2_planned = false;               // phase_setup ran the plan kernel; a2 holds its results
    A2Ctrl a2;                             // host copy
    uint32_t a2_grid = 0, a2_wpc = 0;
};

size_t loop_smem_bytes(uint32_t S, uint32_t nbt = NB) {
    return (size_t)((nbt * S + 3u) & ~3u) * 4 + (size_t)LIST_CAP * 4;
}

int work_alloc(const pccl_problem& P, Work& W) {
    const size_t N = P.topo->N, L = P.topo->L, C = P.C;
    size_t max_sources = 0;   // one workspace serves every phase
    size_t max_pairs = 0;
    for (const Phase& ph : P.phases) {
        max_sources = std::max(max_sources, std::max(ph.sources.size(), ph.dsts.size()));   // D also holds the to-dest rows
        max_pairs = std::max(max_pairs, ph.dests.size());
    }
    const size_t words = (C + 63) / 64;
    W.Wp = (uint32_t)std::max<size_t>(16, align_up(words, 16));   // rows are multiples of 128 bytes
    W.S = (W.Wp / 2 + SEG_U4 - 1) / SEG_U4;
    W.nLw = (uint32_t)((L + 63) / 64);
    W.SWp = (uint32_t)align_up((W.Wp / 4 + 63) / 64, 2);          // one summary bit per 4-word sector
    if (loop_smem_bytes(W.S) > 200 * 1024) return PCCL_ERR_UNSUPPORTED;
    Carver c;
    const size_t o_drow = c.take(max_pairs * 4);
    const size_t o_best = c.take(max_pairs * 8), o_sf = c.take(L * 2 * 8), o_si = c.take(L * 2 * 4);
    const size_t o_w = c.take(L * 8), o_D = c.take(max_sources * N * 8), o_free = c.take(L * 8),
                 o_mb = c.take((size_t)3 * W.nLw * 8), o_inf = c.take(L * 4), o_he = c.take(N * 4), o_ee = c.take(L * 4),
                 o_gc = c.take(L * W.S * 4), o_gt = c.take(L * 4), o_hold = c.take(C * HOLD_ROW * 4);
    const size_t o_nb = c.take((N + 1) * 8), o_po = c.take((N + 1) * 8), o_lo = c.take((L + 1) * 8), o_so = c.take(N * 4);
    W.zero_off = c.cur;
    const size_t o_have = c.take(N * W.Wp * 8), o_wants = c.take(N * W.Wp * 8), o_hs = c.take(N * W.SWp * 8),
                 o_ws = c.take(N * W.SWp * 8), o_wc = c.take(N * 4), o_hc = c.take(C * 4), o_ctrl = c.take(sizeof(LoopCtrl)),
                 o_a2 = c.take(sizeof(A2Ctrl));
    W.zero_bytes = c.cur - W.zero_off;
    int rc = dev_alloc(c.cur, &W.blob);
    if (rc) return rc;
    unsigned char* b = (unsigned char*)W.blob;
    W.w = (uint64_t*)(b + o_w); W.D = (uint64_t*)(b + o_D); W.free_t = (uint64_t*)(b + o_free);
    W.matchbits = (uint64_t*)(b + o_mb); W.inflight = (uint32_t*)(b + o_inf); W.have_epoch = (uint32_t*)(b + o_he);
    W.empty_epoch = (uint32_t*)(b + o_ee); W.have = (uint64_t*)(b + o_have); W.wants = (uint64_t*)(b + o_wants);
    W.hsum = (uint64_t*)(b + o_hs); W.wsum = (uint64_t*)(b + o_ws);
    W.gcnt = (uint32_t*)(b + o_gc); W.gtot = (uint32_t*)(b + o_gt);
    W.best = (uint64_t*)(b + o_best); W.drow = (uint32_t*)(b + o_drow);
    W.hold = (uint32_t*)(b + o_hold); W.hold_cnt = (uint32_t*)(b + o_hc);
    W.st_free = (uint64_t*)(b + o_sf); W.st_inf = (uint32_t*)(b + o_si);
    W.wants_cnt = (uint32_t*)(b + o_wc); W.ctrl = (LoopCtrl*)(b + o_ctrl);
    W.nbase = (unsigned long long*)(b + o_nb); W.poff = (unsigned long long*)(b + o_po);
    W.loff = (unsigned long long*)(b + o_lo); W.soff = (uint32_t*)(b + o_so); W.a2ctrl = (A2Ctrl*)(b + o_a2);
    return PCCL_OK;
}

struct PhaseView {   // link tables in the synthesized direction
    const uint32_t *esrc, *edst, *in_off, *in_link, *out_link, *out_far, *lo_off, *lo_deg, *out_off, *in_far;
};
PhaseView view_of(const pccl_topology* t, bool transposed) {
    if (!transposed)
        return {t->d_src, t->d_dst, t->d_in_off, t->d_in_link, t->d_out_link, t->d_out_far, t->d_lo_off_n, t->d_lo_deg_n,
                t->d_out_off, t->d_in_far};
    return {t->d_dst, t->d_src, t->d_out_off, t->d_out_link, t->d_in_link, t->d_in_far, t->d_lo_off_t, t->d_lo_deg_t,
            t->d_in_off, t->d_out_far};
}

// steps A..C; on return the wants total is in *M (synchronises the stream)
int phase_setup(const pccl_problem& P, const Phase& ph, Work& W, uint64_t seed, uint64_t* M, bool dynamic = false,
                bool plan_async = false) {
    const pccl_topology* t = P.topo;
    const uint32_t N = t->N, L = t->L, C = P.C;
    const PhaseView pv = view_of(t, ph.transposed);
    const uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
    cudaStream_t st = G.stream;
    CU(cudaMemsetAsync((unsigned char*)W.blob + W.zero_off, 0, W.zero_bytes, st));
    if (L) k_link_cost<<<(L + 255) / 256, 256, 0, counted(st)>>>(t->d_alpha, t->d_bpp, L, P.chunk_bytes, W.w);
    if (dynamic) {
        // reading Q18: distances TO every distinct dest (Bellman-Ford on the reversed links), best = dist(src -> dest),
        // wants = every node strictly closer to some dest than the source
        const uint32_t NDS = (uint32_t)ph.dsts.size();
        const uint64_t NP = ph.dests.size();
        const size_t smem = (size_t)N * 8;
        if (smem > 200 * 1024) return PCCL_ERR_UNSUPPORTED;
        if (smem > 48 * 1024) CU(cudaFuncSetAttribute(k_distances, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (NDS) k_distances<<<NDS, 512, smem, counted(st)>>>(pv.edst, pv.esrc, W.w, N, L, ph.d_dsts, W.D);
        if (NP) k_best_init<<<(unsigned)((NP + 255) / 256), 256, 0, counted(st)>>>(ph.d_cond_src, ph.d_dests, ph.d_dchunk, NP, ph.d_didx,
                                                                         W.D, N, W.best, W.drow, &W.ctrl->err);
        if (C) k_have<<<(C + 255) / 256, 256, 0, counted(st)>>>(ph.d_cond_src, C, W.Wp, W.SWp, W.have, W.hsum);
        const uint64_t nth = (uint64_t)N * ((C + 63) / 64);   // warps: one per (node, 64-chunk word)
        if (nth > (0x7FFFFFFFull << 2)) return PCCL_ERR_UNSUPPORTED;
        if (nth) k_wants_dyn_init<<<(unsigned)((nth * 32 + 127) / 128), 128, 0, counted(st)>>>(ph.d_dest_off, ph.d_dests, ph.d_didx, W.D, W.best, N,
                                                                                C, W.Wp, W.SWp, W.wants, W.wsum, W.wants_cnt);
        k_sum_u32<<<1, 1024, 0, counted(st)>>>(W.wants_cnt, N, &W.ctrl->wants_total);
        CU(cudaGetLastError());
        LoopCtrl* mbx = (LoopCtrl*)G.mailbox;
        CU(cudaMemcpyAsync(mbx, W.ctrl, sizeof(LoopCtrl), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        if (mbx->err & 1u) return PCCL_ERR_UNREACHABLE;
        if (mbx->err) return PCCL_ERR_INTERNAL;
        *M = mbx->wants_total;
        return PCCL_OK;
    }
    const uint32_t NS = (uint32_t)ph.sources.size();
    if (NS) {
        const size_t smem = (size_t)N * 8;
        if (smem > 200 * 1024) return PCCL_ERR_UNSUPPORTED;
        if (smem > 48 * 1024) CU(cudaFuncSetAttribute(k_distances, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        k_distances<<<NS, 512, smem, counted(st)>>>(pv.esrc, pv.edst, W.w, N, L, ph.d_sources, W.D);
    }
    if (C) k_have<<<(C + 255) / 256, 256, 0, counted(st)>>>(ph.d_cond_src, C, W.Wp, W.SWp, W.have, W.hsum);
    const uint64_t ND = ph.dests.size();
    if (ND) {
        const size_t wants_smem = (size_t)N * 8 <= 32 * 1024 ? (size_t)N * 8 : 0;   // the staged distance row (k_wants)
        k_wants<<<(unsigned)((ND + 127) / 128), 128, wants_smem, counted(st)>>>(ph.d_cond_src, ph.d_dests, ph.d_dchunk, ND, pv.esrc, pv.in_off,
                                                          pv.in_link, W.w, ph.d_sidx, W.D, N, W.Wp, k0, k1, W.wants,
                                                          &W.ctrl->err, ph.d_orig, wants_smem ? 1u : 0u);
        k_wants_finish<<<N, 256, 0, counted(st)>>>(W.wants, W.Wp, W.SWp, W.wsum, W.wants_cnt);
    }
    k_sum_u32<<<1, 1024, 0, counted(st)>>>(W.wants_cnt, N, &W.ctrl->wants_total);
    W.a2_planned = false;
    if (plan_async) {
        // barrier-free loop: one warp per destination, ceil(N / SMs) destinations per CTA, one CTA per SM
        W.a2_wpc = std::max(1u, (N + (uint32_t)G.sm_count - 1) / (uint32_t)G.sm_count);
        W.a2_grid = (N + W.a2_wpc - 1) / W.a2_wpc;
        A2Args pa;
        memset(&pa, 0, sizeof(pa));
        pa.N = N; pa.L = L; pa.grid = W.a2_grid; pa.wpc = W.a2_wpc; pa.ncls = ph.ncls;
        pa.esrc = pv.esrc; pa.in_off = pv.in_off; pa.w = W.w; pa.wants_cnt = W.wants_cnt;
        pa.nbase = W.nbase; pa.poff = W.poff; pa.loff = W.loff; pa.soff = W.soff; pa.ctrl = W.a2ctrl;
        k_a2_plan<<<1, 1024, 0, counted(st)>>>(pa);
    }
    CU(cudaGetLastError());
    LoopCtrl* mb = (LoopCtrl*)G.mailbox;
    A2Ctrl* mb2 = (A2Ctrl*)((unsigned char*)G.mailbox + 1024);
    static_assert(sizeof(LoopCtrl) <= 1024 && sizeof(A2Ctrl) <= 1024, "mailbox quarters");
    CU(cudaMemcpyAsync(mb, W.ctrl, sizeof(LoopCtrl), cudaMemcpyDeviceToHost, st));
    if (plan_async) CU(cudaMemcpyAsync(mb2, W.a2ctrl, sizeof(A2Ctrl), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (mb->err & 1u) return PCCL_ERR_UNREACHABLE;
    if (mb->err) return PCCL_ERR_INTERNAL;
    *M = mb->wants_total;
    if (plan_async) { W.a2 = *mb2; W.a2_planned = true; }
    return PCCL_OK;
}

// row a5 as a streaming kernel (pccl_sweep.cuh): candidate counts of every link; seeds the kept counts of the barrier
// loops.  Rows staged by bulk asynchronous copies unless PCCL_FLAG_LSU_SWEEP asks for the per-lane 128-bit loads.
int launch_count_sweep(const LoopArgs& a, uint32_t flags) {
    if (a.N == 0 || a.L == 0) return PCCL_OK;
    cudaStream_t st = G.stream;
    const bool tma = !(flags & PCCL_FLAG_LSU_SWEEP);
    const void* kern = tma ? (const void*)k_count_sweep<true> : (const void*)k_count_sweep<false>;
    const size_t smem = tma ? (size_t)SW_STAGES * SW_ROWS * SW_SLICE_U4 * 16 : 0;
    if (smem > 48 * 1024) CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, SW_THREADS, smem));
    if (occ < 1) return PCCL_ERR_CUDA;
    // (the kernel can cut a row into parts to balance the CTAs; measured on B200 the restart of the copy pipeline per part
    // costs the TMA form more than the balance gains -- 70 -> 77 us on the 28x28 workload -- so rows stay whole)
    const uint32_t resident = (uint32_t)occ * (uint32_t)G.sm_count;
    const uint32_t parts = 1;
    LoopArgs b = a;
    b.flags = parts;                                           // (the sweep kernel reads its parts count here)
    if (parts > 1) CU(cudaMemsetAsync(a.gtot, 0, (size_t)a.L * 4, st));
    const uint32_t grid = (uint32_t)std::min<uint64_t>((uint64_t)a.N * parts, resident);
    if (tma) k_count_sweep<true><<<grid, SW_THREADS, smem, counted(st)>>>(b);
    else k_count_sweep<false><<<grid, SW_THREADS, smem, counted(st)>>>(b);
    CU(cudaGetLastError());
    return PCCL_OK;
}

struct LoopResult {
    uint64_t total, tmax, events, rows, links, slow, bytes;
    uint32_t grid;
};

// A phase of the call: an NVTX range (setup / loop / emit, visible in Nsight Systems and ncu --nvtx) and, with
// PCCL_FLAG_TIME_LOOP, a pair of CUDA events around every segment of it (read once at the end of the call: recording
// does not synchronise).
struct Timer {
    const char* name;
    bool on = false, open = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> seg;
    explicit Timer(const char* n) : name(n) {}
    void init(bool enable) { on = enable; }
    void start() {
        if (open) return;
        nvtxRangePushA(name);
        open = true;
        if (!on) return;
        cudaEvent_t a = nullptr, b = nullptr;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) {
            (void)cudaGetLastError();
            if (a) cudaEventDestroy(a);
            on = false;
            return;
        }
        try {
            seg.emplace_back(a, b);
        } catch (const std::bad_alloc&) {
            cudaEventDestroy(a); cudaEventDestroy(b);
            on = false;
            return;
        }
        cudaEventRecord(a, G.stream);
    }
    void stop() {
        if (!open) return;
        nvtxRangePop();
        open = false;
        if (on && !seg.empty()) cudaEventRecord(seg.back().second, G.stream);
    }
    float total() {   // milliseconds over all segments (waits for the last event of each)
        float acc = 0.f;
        for (auto& p : seg) {
            float ms = 0.f;
            if (cudaEventSynchronize(p.second) == cudaSuccess && cudaEventElapsedTime(&ms, p.first, p.second) == cudaSuccess) acc += ms;
            else (void)cudaGetLastError();
        }
        return acc;
    }
    ~Timer() {
        if (open) nvtxRangePop();
        for (auto& p : seg) { cudaEventDestroy(p.first); cudaEventDestroy(p.second); }
    }
};
struct Timers {
    Timer setup{"pccl:setup"}, loop{"pccl:loop"}, emit{"pccl:emit"};
};

// stable LSD radix sort / reduce emitter, defined below
int reverse_sorted(Rec* raw, uint64_t M, uint64_t T, uint32_t L, Rec* out, bool reverse, uint64_t shift);

// steps D..E without a grid barrier (pccl_loop2.cuh): setup of the per-destination entry lists and translation
// tables, the loop, and the ranking of the logged claims into canonical order.  `raw_only`: leave the records in log
// order (a transposed phase sorts them after the reversal anyway).
// host_out (optional, pinned, out_cap records): the emitter's windows run on a second stream while the loop is going
// and this thread copies the finished prefix of the records there meanwhile; *streamed says whether all of them went.
int phase_loop_async(const pccl_problem& P, const Phase& ph, const Work& W, uint64_t seed, uint32_t flags, Rec* out,
                     uint64_t out_cap, uint64_t t_offset, bool raw_only, LoopResult* res, Timers* tm,
                     Rec* host_out = nullptr, bool* streamed = nullptr) {
    const pccl_topology* t = P.topo;
    const PhaseView pv = view_of(t, ph.transposed);
    const uint32_t N = t->N, L = t->L;
    const uint64_t M = out_cap;
    cudaStream_t st = G.stream;
    A2Args a;
    memset(&a, 0, sizeof(a));
    a.N = N; a.L = L; a.Wp = W.Wp; a.nLw = W.nLw;
    a.k0 = (uint32_t)(seed & 0xFFFFFFFFull); a.k1 = (uint32_t)(seed >> 32);
    a.grid = W.a2_grid; a.wpc = W.a2_wpc;
    a.ncls = ph.ncls; a.cls = ph.d_cls; a.orig = ph.d_orig;
    a.esrc = pv.esrc; a.edst = pv.edst; a.psrc = t->d_src; a.pdst = t->d_dst; a.in_off = pv.in_off; a.in_link = pv.in_link;
    a.w = W.w; a.wants = W.wants; a.wants_cnt = W.wants_cnt; a.csrc = ph.d_cond_src;
    a.nbase = W.nbase; a.poff = W.poff; a.loff = W.loff; a.soff = W.soff; a.ctrl = W.a2ctrl; a.abort_flag = &W.ctrl->err;
    a.tcap = 1u << 16;
    a.ecap = (uint32_t)std::min<uint64_t>(16384, std::max<uint64_t>(64, ((uint64_t)64 << 20) / ((uint64_t)std::max(W.nLw, 1u) * 12)));
    a.out = out; a.out_cap = out_cap; a.t_offset = t_offset;
    Carver c;
    const size_t o_ids = c.take(M * 4), o_rp = c.take((size_t)N * W.Wp * 4), o_xm = c.take(W.a2.xmap_total * 4),
                 o_pr = c.take(W.a2.priv_total * 4), o_hdr = c.take((size_t)N * 16 * A2_HDR_STRIDE), o_es = c.take(M * 4),
                 o_us = c.take((size_t)a.ecap * 4), o_cs = c.take((size_t)a.ecap * 4), o_eb = c.take((size_t)a.ecap * 8),
                 o_wb = c.take((size_t)a.ecap * W.nLw * 4), o_tr = c.take((size_t)a.tcap * 4);
    const size_t o_ff = c.cur;                                   // filled with 0xFF: the log and the time keys
    const size_t o_log = c.take(M * 16 * A2_LOG_STRIDE), o_tk = c.take((size_t)a.tcap * 8);
    const size_t o_zero = c.cur;                                 // cleared
    const size_t o_tc = c.take((size_t)a.tcap * 4), o_tf = c.take((size_t)a.tcap * 4), o_bm = c.take((size_t)a.ecap * W.nLw * 8);
    const size_t o_wc = c.take((size_t)N * 4), o_wn = c.take((size_t)N * 4), o_win = c.take(sizeof(A2Win));
    void* blob = nullptr;
    int rc = dev_alloc(c.cur, &blob);
    if (rc) return rc;
    struct Guard { void* p; ~Guard() { dev_free(p); } } guard{blob};
    unsigned char* b = (unsigned char*)blob;
    a.ids = (uint32_t*)(b + o_ids); a.rowpre = (uint32_t*)(b + o_rp); a.xmap = (uint32_t*)(b + o_xm);
    a.priv = (uint32_t*)(b + o_pr); a.hdr = (U128*)(b + o_hdr); a.eslot = (uint32_t*)(b + o_es);
    a.used = (uint32_t*)(b + o_us); a.cnt_sorted = (uint32_t*)(b + o_cs); a.ebase = (unsigned long long*)(b + o_eb);
    a.wbase = (uint32_t*)(b + o_wb); a.trank = (uint32_t*)(b + o_tr); a.log = (U128*)(b + o_log);
    a.tkey = (unsigned long long*)(b + o_tk); a.tcnt = (uint32_t*)(b + o_tc); a.tflag = (uint32_t*)(b + o_tf);
    a.bm = (unsigned long long*)(b + o_bm);
    a.wcur = (uint32_t*)(b + o_wc); a.wnext = (uint32_t*)(b + o_wn); a.win = (A2Win*)(b + o_win);
    a.progress = nullptr;
    CU(cudaMemsetAsync(b + o_ff, 0xFF, o_zero - o_ff, st));
    CU(cudaMemsetAsync(b + o_zero, 0, c.cur - o_zero, st));
    // entries, translation tables, private images (once per phase)
    if (tm) tm->setup.start();
    k_a2_entries<<<N, 256, 0, counted(st)>>>(a);
    // the translation tables and the private images only depend on the entry lists: side by side on two streams
    // (config 4: 45 + 36 us one after the other)
    CU(cudaEventRecord(G.loop_done, st));
    CU(cudaStreamWaitEvent(G.emit_stream, G.loop_done, 0));
    k_a2_priv<<<N, 128, 0, counted(G.emit_stream)>>>(a);
    CU(cudaEventRecord(G.win_done, G.emit_stream));
    if (L) k_a2_xmap<<<L, 128, 0, counted(st)>>>(a);
    CU(cudaStreamWaitEvent(st, G.win_done, 0));
    const size_t smem = (size_t)W.a2.smem_need;
    const int threads = (int)W.a2_wpc * 32;
    const void* kloop2 = ph.ncls ? (const void*)k_loop2<true> : (const void*)k_loop2<false>;
    if (smem > 48 * 1024) CU(cudaFuncSetAttribute(kloop2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kloop2, threads, smem));
    if (occ < 1 || (uint64_t)occ * (uint64_t)G.sm_count < W.a2_grid) return PCCL_ERR_INTERNAL;   // (checked by the caller's plan)
    void* args[] = {(void*)&a};
    // one window of the emitter (pccl_loop2.cuh): the claims that start before the global virtual time -- or all that
    // are left (final) -- ranked and written behind the records of the earlier windows
    // `pad` bytes of (unused) dynamic shared memory keep a window's CTAs off the SMs where a CTA of the loop is resident:
    // beside the loop's latency-bound warps they cost it 0.18 ms at config 4 (measured); on the SMs the loop leaves free
    // they cost it nothing
    auto window = [&](cudaStream_t s, int final, size_t pad, uint32_t wgrid) -> cudaError_t {
        k_win_begin<<<1, 1024, pad, counted(s)>>>(a, final);
        k_win_times<<<wgrid, 256, pad, counted(s)>>>(a);
        if (!raw_only) {
            k_win_rank<<<(a.ecap + 255) / 256, 256, pad, counted(s)>>>(a);
            k_win_base<<<1, 1024, pad, counted(s)>>>(a);
            k_win_bits<<<wgrid, 256, pad, counted(s)>>>(a);
            k_win_wbase<<<std::min<uint32_t>((a.ecap + 7) / 8, 256u), 256, pad, counted(s)>>>(a);
            k_win_write<<<wgrid, 256, pad, counted(s)>>>(a);
            k_win_end<<<1, 1, 0, counted(s)>>>(a);
        } else {
            k_emit_raw<<<N, 256, 0, counted(s)>>>(a);
        }
        return cudaGetLastError();
    };
    // streaming: the progress word lives in the pinned mailbox (mapped: k_win_end stores to it directly)
    volatile unsigned long long* progress = (volatile unsigned long long*)((unsigned char*)G.mailbox + 2048);
    // Early windows -- the emitter running on a second stream while the loop is going -- in two cases.  (i) The records
    // leave for the host: the download then overlaps the loop.  (ii) They stay on the device and the loop leaves SMs free
    // (config 4: 128 CTAs on 148 SMs): what is left for the window after the loop is only the tail of the schedule.
    // Window CTAs resident BESIDE the loop's latency-bound warps cost it 0.1-0.18 ms at config 4 (measured).  When the
    // loop leaves at least 16 SMs free, an early window is therefore launched with only as many CTAs as fit on those SMs
    // (8 of 256 threads each; the block scheduler fills idle SMs first) striding over the nodes, and 24 KB of unused
    // dynamic shared memory per CTA keeps it at 8 per SM: loop + emit 2.52 -> 2.41 ms at config 4 with the records kept
    // on the device, end to end 3.8 -> 3.7 ms in the same process.  (One CTA per free SM, forced by a 216 KB pad, is too
    // slow: the windows fall behind the download, 3.4 -> 4.1 ms.)  With fewer free SMs (config 5: one) case (i) uses the
    // full grid and case (ii) has no early windows.
    const bool stream_out = !raw_only && out_cap > 0 && host_out != nullptr;
    const uint32_t free_sms = (uint32_t)G.sm_count > W.a2_grid ? (uint32_t)G.sm_count - W.a2_grid : 0u;
    const bool shielded = !raw_only && out_cap > 0 && free_sms >= 16u;
    const size_t win_pad = shielded ? 24 * 1024 : 0;
    const uint32_t wgrid_early = shielded ? std::min<uint32_t>(N, free_sms * 8u) : N;
    const bool early = stream_out || shielded;
    uint64_t copied = 0;
    struct Drain {   // whatever happens, nothing of this call is left running on the side streams
        bool on;
        ~Drain() {
            if (!on) return;
            (void)cudaStreamSynchronize(G.emit_stream);
            (void)cudaStreamSynchronize(G.copy_stream);
            (void)cudaGetLastError();
        }
    } drain{early};
    if (early) {
        if (stream_out) {
            *progress = 0;
            void* dp = nullptr;
            CU(cudaHostGetDevicePointer(&dp, (void*)progress, 0));
            a.progress = (unsigned long long*)dp;
        }
        CU(cudaEventRecord(G.pre_loop, st));                      // headers, logs and tables are initialised
        CU(cudaStreamWaitEvent(G.emit_stream, G.pre_loop, 0));
    }
    if (tm) { tm->setup.stop(); tm->loop.start(); }
    DBGT("  a2 setup enqueued");
    CU(cudaLaunchCooperativeKernel(kloop2, dim3(W.a2_grid), dim3(threads), args, smem, counted(st)));
    if (tm) tm->loop.stop();
    DBGT("  loop launched");
    if (early) {
        // windows on the emit stream while the loop runs (it never waits for them; they read headers and logs only);
        // finished records leave in pieces of >= 2 MB on the copy stream.  Both streams are drained before anything
        // can fail or return.
        constexpr uint64_t PIECE = 1u << 16;
        bool in_flight = false, any = false;
        cudaError_t e = cudaEventRecord(G.loop_done, st), q = cudaErrorNotReady;
        while (e == cudaSuccess && (q = cudaEventQuery(G.loop_done)) == cudaErrorNotReady) {
            if (in_flight && cudaEventQuery(G.win_done) != cudaErrorNotReady) in_flight = false;
            if (in_flight) continue;
            const uint64_t p = stream_out ? std::min<uint64_t>(*progress, out_cap) : 0;
            if (p >= copied + PIECE) {
                e = cudaMemcpyAsync(host_out + copied, out + copied, (p - copied) * sizeof(Rec), cudaMemcpyDeviceToHost,
                                    G.copy_stream);
                copied = p;
            }
            if (e == cudaSuccess) e = window(G.emit_stream, 0, win_pad, wgrid_early);
            if (e == cudaSuccess) e = cudaEventRecord(G.win_done, G.emit_stream);
            in_flight = any = true;
        }
        if (e == cudaSuccess && q != cudaSuccess) e = q;
        if (e == cudaSuccess && any) e = cudaStreamWaitEvent(st, G.win_done, 0);   // the last window before the final one
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            (void)cudaStreamSynchronize(G.emit_stream);
            (void)cudaStreamSynchronize(G.copy_stream);
            (void)cudaStreamSynchronize(st);
            (void)cudaGetLastError();
            return PCCL_ERR_CUDA;
        }
    }
    DBGT("  loop done (polling)");
    if (tm) tm->emit.start();
    {
        const cudaError_t e = window(st, 1, 0, N);
        if (e != cudaSuccess) {
            (void)cudaStreamSynchronize(G.copy_stream);
            (void)cudaStreamSynchronize(st);
            (void)cudaGetLastError();
            return PCCL_ERR_CUDA;
        }
    }
    if (tm) tm->emit.stop();
    LoopCtrl* mb = (LoopCtrl*)G.mailbox;
    A2Ctrl* mb2 = (A2Ctrl*)((unsigned char*)G.mailbox + 1024);
    CU(cudaMemcpyAsync(mb, W.ctrl, sizeof(LoopCtrl), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(mb2, W.a2ctrl, sizeof(A2Ctrl), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    DBGT("  final window synced");
#ifdef PCCL_A2_PROFILE
    fprintf(stderr, "[a2 profile] actions %llu polls %llu | cycles per action: philox %.0f poll %.0f apply %.0f pick %.0f commit %.0f next %.0f | per poll: load wait %.0f evaluate %.0f\n",
            mb2->actions, mb2->polls, (double)mb2->prof[0] / mb2->actions, (double)mb2->prof[1] / mb2->actions,
            (double)mb2->prof[2] / mb2->actions, (double)mb2->prof[3] / mb2->actions, (double)mb2->prof[4] / mb2->actions,
            (double)mb2->prof[5] / mb2->actions, (double)mb2->prof[6] / mb2->polls, (double)mb2->prof[7] / mb2->polls);
#endif
    if (mb->err) return PCCL_ERR_INTERNAL;
    if (mb2->err & 2u) return PCCL_ERR_NOMEM;
    if (!raw_only && (mb2->err & 1u)) {
        // more distinct event times than the time table or the per-event bitmaps hold: records in log order, then the
        // general sort by (t_start, link)
        Rec* tmp = nullptr;
        rc = dev_alloc(std::max<uint64_t>(M, 1) * sizeof(Rec), (void**)&tmp);
        if (rc) return rc;
        A2Args a2 = a;
        a2.out = tmp; a2.t_offset = 0;
        k_emit_raw<<<N, 256, 0, counted(st)>>>(a2);
        if (tm) tm->emit.start();
        rc = reverse_sorted(tmp, mb2->total, mb2->tmax, L, out, false, t_offset);
        if (tm) tm->emit.stop();
        cudaError_t e = cudaStreamSynchronize(st);
        dev_free(tmp);
        if (rc) return rc;
        if (e != cudaSuccess) { (void)cudaGetLastError(); return PCCL_ERR_CUDA; }
    }
    if (stream_out && !(mb2->err & 1u) && mb2->total <= out_cap) {   // the tail (after a fall-back sort nothing was streamed)
        if (mb2->total > copied)
            CU(cudaMemcpyAsync(host_out + copied, out + copied, (mb2->total - copied) * sizeof(Rec), cudaMemcpyDeviceToHost,
                               G.copy_stream));
        CU(cudaStreamSynchronize(G.copy_stream));
        DBGT("  tail copy synced");
        if (streamed) *streamed = true;
    }
    res->total = mb2->total; res->tmax = mb2->tmax;
    res->events = (uint64_t)mb2->n_end + 1;   // event times = {0} and every distinct t_end (each free time is visited)
    res->rows = mb2->actions; res->links = mb2->picks; res->slow = mb2->slow; res->bytes = mb2->bytes;
    res->grid = W.a2_grid;
    return PCCL_OK;
}

// steps D..E: the event loop; records go to `out` (capacity M) in canonical order
// host_out (optional, pinned, out_cap records): with the one-barrier loop the records are copied there while the
// loop runs (the kernel publishes how many are final, this thread issues the copies); *streamed says whether
int phase_loop(const pccl_problem& P, const Phase& ph, const Work& W, uint64_t seed, uint32_t flags, Rec* out,
               uint64_t out_cap, uint64_t t_offset, LoopResult* res, Timers* tm, std::vector<uint64_t>* trace = nullptr,
               Rec* host_out = nullptr, bool* streamed = nullptr) {
    const bool dynamic = (flags & PCCL_FLAG_DYNAMIC_RELAY) != 0;
    if (W.a2_planned && out_cap > 0 && out_cap <= 0xFFFFFFFFull && W.a2.smem_need <= 220 * 1024 &&
        ((flags & (PCCL_FLAG_ASYNC | PCCL_FLAG_DIST_PICK)) || W.a2.w_max / 16 <= W.a2.w_min))
        return phase_loop_async(P, ph, W, seed, flags, out, out_cap, t_offset, ph.transposed, res, tm, host_out, streamed);
    if ((flags & PCCL_FLAG_DIST_PICK) && out_cap > 0) return PCCL_ERR_UNSUPPORTED;   // the c.dist pick lives in the barrier-free loop
    // the dynamic rule keeps the counts current too: wants bits are only dropped where a neighbour holds the chunk
    // (holder lists, dyn_shrink_wants); DENSE_SWEEP / RESCAN recount instead and drop every bit at once
    const pccl_topology* t = P.topo;
    const PhaseView pv = view_of(t, ph.transposed);
    LoopArgs a;
    a.N = t->N; a.L = t->L; a.Wp = W.Wp; a.S = W.S; a.nLw = W.nLw; a.SWp = W.SWp; a.flags = flags;
    a.k0 = (uint32_t)(seed & 0xFFFFFFFFull); a.k1 = (uint32_t)(seed >> 32);
    a.esrc = pv.esrc; a.edst = pv.edst; a.psrc = t->d_src; a.pdst = t->d_dst;
    a.in_off = pv.in_off; a.in_link = pv.in_link; a.w = W.w; a.have = W.have; a.wants = W.wants;
    a.hsum = W.hsum; a.wsum = W.wsum;
    const bool rescan = (flags & (PCCL_FLAG_RESCAN | PCCL_FLAG_DENSE_SWEEP)) != 0;
    a.gcnt = rescan ? nullptr : W.gcnt; a.gtot = rescan ? nullptr : W.gtot;
    a.out_link = pv.out_link; a.out_far = pv.out_far; a.lo_off = pv.lo_off; a.lo_deg = pv.lo_deg;
    a.wants_cnt = W.wants_cnt; a.free_t = W.free_t; a.inflight = W.inflight; a.have_epoch = W.have_epoch;
    a.empty_epoch = W.empty_epoch; a.matchbits = W.matchbits; a.ctrl = W.ctrl; a.out = out; a.t_offset = t_offset;
    a.out_cap = out_cap;
    // dynamic rule with kept counts: a tightened best revisits only the out-neighbours of the chunk's holders
    const bool lazy = dynamic && !(flags & (PCCL_FLAG_RESCAN | PCCL_FLAG_DENSE_SWEEP));
    a.csrc = ph.d_cond_src; a.out_off = pv.out_off; a.drow = W.drow; a.in_far = pv.in_far;
    a.hold = lazy ? W.hold : nullptr; a.hold_cnt = lazy ? W.hold_cnt : nullptr;
    a.best = dynamic ? W.best : nullptr; a.Dto = W.D; a.didx = ph.d_didx; a.dest_off = ph.d_dest_off; a.dests = ph.d_dests;
    cudaStream_t st = G.stream;
    a.trace = nullptr; a.trace_cap = 0;
    void* trace_dev = nullptr;
    if ((flags & PCCL_FLAG_TRACE) && trace) {
        a.trace_cap = 1u << 14;
        const size_t tb = (size_t)a.trace_cap * TRACE_SLOTS * 8;
        int rc = dev_alloc(tb, &trace_dev);
        if (rc) return rc;
        if (cudaMemsetAsync(trace_dev, 0, tb, st) != cudaSuccess) { (void)cudaGetLastError(); dev_free(trace_dev); return PCCL_ERR_CUDA; }
        a.trace = (uint64_t*)trace_dev;
    }
    struct TraceGuard { void* p; ~TraceGuard() { dev_free(p); } } trace_guard{trace_dev};
    const uint32_t n_init = std::max(std::max(a.L, a.N), std::max(3 * a.nLw, 1u));
    // one warp per in-link of a sweep: destinations with at most 4 in-links run in 128-thread CTAs (8 per SM),
    // so that twice as many destinations are resident at once
    const uint32_t max_deg = ph.transposed ? t->max_out : t->max_in;
    const bool small = max_deg <= 4;
    int threads = small ? 128 : 256;
    size_t smem = loop_smem_bytes(W.S, small ? 4 : 8);
    // the one-barrier loop (pccl_loop1.cuh): kept counts, <= 8 in-links per node, <= 128 segments per row,
    // at most DEST_CACHE destinations per CTA; everything else runs the two-barrier loop
    bool fast = !rescan && !dynamic && !(flags & PCCL_FLAG_TWO_BARRIERS) && max_deg <= 8 && W.S <= 128;
    const void* kern = nullptr;
    uint32_t grid = 0;
    for (int attempt = 0; attempt < 2; ++attempt) {
        // one-barrier loop: teams of 4 warps are paired in 256-thread CTAs (half as many CTAs at the barrier)
        kern = fast ? (small ? (const void*)k_loop1<4, 2> : (const void*)k_loop1<8, 1>)
                    : (dynamic ? (small ? (const void*)k_loop<4, true> : (const void*)k_loop<8, true>)
                               : (small ? (const void*)k_loop<4, false> : (const void*)k_loop<8, false>));
        const int teams = (fast && small) ? 2 : 1;
        threads = (small ? 128 : 256) * teams;
        smem = loop_smem_bytes(W.S, small ? 4 : 8) * teams;
        if (smem > 48 * 1024) CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int occ = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem));
        if (occ < 1) return PCCL_ERR_CUDA;
        const uint32_t max_grid = (uint32_t)occ * (uint32_t)G.sm_count;
        const uint32_t want = std::max(std::max((a.N + teams - 1) / teams, (a.L + threads - 1) / threads), 1u);
        grid = std::min(max_grid, want);
        if (fast && (uint64_t)a.N > (uint64_t)DEST_CACHE * grid * teams) { fast = false; continue; }
        break;
    }
    a.st_free = fast ? W.st_free : nullptr;
    a.st_inf = fast ? W.st_inf : nullptr;
    // the progress word lives in the second half of the pinned mailbox (mapped: the kernel stores to it directly)
    static_assert(sizeof(LoopCtrl) <= 2048, "mailbox halves");
    volatile unsigned long long* progress = (volatile unsigned long long*)((unsigned char*)G.mailbox + 2048);
    const bool stream_out = fast && host_out != nullptr && out_cap > 0;
    a.progress = nullptr;
    if (stream_out) {
        *progress = 0;
        void* dp = nullptr;
        CU(cudaHostGetDevicePointer(&dp, (void*)progress, 0));
        a.progress = (unsigned long long*)dp;
    }
    if (tm) tm->setup.start();
    k_loop_init<<<(n_init + 255) / 256, 256, 0, counted(st)>>>(a);
    if (a.gcnt != nullptr && a.L) { const int rcs = launch_count_sweep(a, flags); if (rcs) return rcs; }
    void* args[] = {(void*)&a};
    if (tm) { tm->setup.stop(); tm->loop.start(); }
    CU(cudaLaunchCooperativeKernel(kern, dim3(grid), dim3(threads), args, smem, counted(st)));
    if (tm) tm->loop.stop();
    LoopCtrl* mb = (LoopCtrl*)G.mailbox;
    CU(cudaMemcpyAsync(mb, W.ctrl, sizeof(LoopCtrl), cudaMemcpyDeviceToHost, st));
    if (stream_out) {
        // copy finished records in pieces of >= 2 MB on the copy stream while the loop is still running; the tail
        // follows once the loop is done.  The copy stream is drained before anything can fail or return.
        constexpr uint64_t PIECE = 1u << 16;
        uint64_t copied = 0;
        cudaError_t e = cudaEventRecord(G.loop_done, st), q = cudaErrorNotReady;
        while (e == cudaSuccess && (q = cudaEventQuery(G.loop_done)) == cudaErrorNotReady) {
            const uint64_t p = stream_out ? std::min<uint64_t>(*progress, out_cap) : 0;
            if (p >= copied + PIECE) {
                e = cudaMemcpyAsync(host_out + copied, out + copied, (p - copied) * sizeof(Rec), cudaMemcpyDeviceToHost,
                                    G.copy_stream);
                copied = p;
            }
        }
        if (e == cudaSuccess && q != cudaSuccess) e = q;
        if (e == cudaSuccess && mb->err == 0 && mb->total <= out_cap && mb->total > copied)
            e = cudaMemcpyAsync(host_out + copied, out + copied, (mb->total - copied) * sizeof(Rec), cudaMemcpyDeviceToHost,
                                G.copy_stream);
        const cudaError_t e2 = cudaStreamSynchronize(G.copy_stream);
        if (e != cudaSuccess || e2 != cudaSuccess) {
            (void)cudaGetLastError();
            (void)cudaStreamSynchronize(st);
            (void)cudaGetLastError();
            return PCCL_ERR_CUDA;
        }
        if (streamed) *streamed = true;
    } else {
        CU(cudaStreamSynchronize(st));
    }
    if (mb->err & 32u) { res->total = mb->total; return PCCL_ERR_NOMEM; }   // more transfers than the record buffer holds
    if (mb->err) return PCCL_ERR_INTERNAL;
    res->total = mb->total; res->tmax = mb->tmax; res->events = mb->events;
    res->rows = mb->rows_scanned; res->links = mb->links_scanned; res->slow = mb->slow_picks;
    res->bytes = mb->bytes_requested;
    res->grid = grid;
    if (a.trace) {
        const size_t n = (size_t)std::min<uint64_t>(res->events, a.trace_cap) * TRACE_SLOTS;
        try {
            trace->assign(n, 0);
        } catch (const std::bad_alloc&) {
            return PCCL_ERR_NOMEM;
        }
        CU(cudaMemcpyAsync(trace->data(), a.trace, n * 8, cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    return PCCL_OK;
}

// stable LSD radix sort of (key, value) pairs on the low `bits` bits; returns which of the two buffers holds the result
int radix_sort_pairs(uint64_t* keys[2], uint32_t* vals[2], uint64_t n, uint32_t bits, uint32_t* ghist, uint32_t nblocks,
                     int cur) {
    cudaStream_t st = G.stream;
    for (uint32_t shift = 0; shift < bits; shift += 8) {
        k_sort_hist<<<nblocks, SORT_THREADS, 0, counted(st)>>>(keys[cur], n, shift, ghist, nblocks);
        k_sort_scan<<<1, 1024, 0, counted(st)>>>(ghist, (uint64_t)256 * nblocks);
        k_sort_scatter<<<nblocks, SORT_THREADS, 0, counted(st)>>>(keys[cur], vals[cur], keys[cur ^ 1], vals[cur ^ 1], n, shift, ghist, nblocks);
        cur ^= 1;
    }
    return cur;
}

// a9 for reductions: raw (transposed-broadcast) records -> reversed, sorted by (t_start, link), into out
// (reverse = false: only sorted, times shifted by `shift`; T then only bounds the key width)
int reverse_sorted(Rec* raw, uint64_t M, uint64_t T, uint32_t L, Rec* out, bool reverse, uint64_t shift) {
    if (M == 0) return PCCL_OK;
    cudaStream_t st = G.stream;
    uint32_t link_bits = 1;
    while ((1ull << link_bits) < (uint64_t)L) ++link_bits;
    uint32_t t_bits = 1;
    while (t_bits < 64 && (T >> t_bits)) ++t_bits;
    if (t_bits + link_bits > 64 || M > 0xFFFFFFFFull) return PCCL_ERR_UNSUPPORTED;
    const uint32_t nblocks = (uint32_t)((M + SORT_TILE - 1) / SORT_TILE);
    Carver c;
    const size_t o_k0 = c.take(M * 8), o_k1 = c.take(M * 8), o_v0 = c.take(M * 4), o_v1 = c.take(M * 4),
                 o_h = c.take((size_t)256 * nblocks * 4);
    void* blob = nullptr;
    int rc = dev_alloc(c.cur, &blob);
    if (rc) return rc;
    unsigned char* b = (unsigned char*)blob;
    uint64_t* keys[2] = {(uint64_t*)(b + o_k0), (uint64_t*)(b + o_k1)};
    uint32_t* vals[2] = {(uint32_t*)(b + o_v0), (uint32_t*)(b + o_v1)};
    uint32_t* ghist = (uint32_t*)(b + o_h);
    const unsigned g256 = (unsigned)((M + 255) / 256);
    k_reverse_keys<<<g256, 256, 0, counted(st)>>>(raw, M, T, link_bits, keys[0], vals[0], reverse);
    const int cur = radix_sort_pairs(keys, vals, M, t_bits + link_bits, ghist, nblocks, 0);
    k_gather_shift<<<g256, 256, 0, counted(st)>>>(raw, vals[cur], M, shift, out);
    cudaError_t e = cudaGetLastError();
    dev_free(blob);   // stream-ordered: freed after the kernels above
    return e == cudaSuccess ? PCCL_OK : PCCL_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------
// PCCL_FLAG_BFS: one phase of the paper's own synthesizer (pccl_bfs.cuh).  On return *out_recs
// holds the M records in canonical order (reversed in direction and time for a transposed
// phase, shifted by t_shift otherwise); the caller owns it.
// ---------------------------------------------------------------------------------------
// PCCL_FLAG_DIST_PICK: the phases of P with their chunks relabelled in (descending c.dist, ascending chunk id) order, so
// that "the candidates with the largest c.dist" are the candidates of the lowest class of labels and ascending label =
// ascending chunk id inside a class.  c.dist and the order are computed on the device (link costs, distances, k_cdist,
// stable radix sort); the host only re-indexes the condition arrays with that order.  Cached in the problem.
int prio_prepare(pccl_problem& P) {
    if (!P.prio_phases.empty()) return PCCL_OK;
    const pccl_topology* t = P.topo;
    const uint32_t N = t->N, L = t->L, C = P.C;
    cudaStream_t st = G.stream;
    std::vector<Phase> out;
    try {
        for (const Phase& ph : P.phases) {
            const PhaseView pv = view_of(t, ph.transposed);
            const uint32_t NS = (uint32_t)ph.sources.size();
            const uint32_t nblocks = (uint32_t)((C + SORT_TILE - 1) / SORT_TILE);
            Carver c;
            const size_t o_w = c.take((size_t)L * 8), o_D = c.take((size_t)NS * N * 8), o_cd = c.take((size_t)C * 8),
                         o_k0 = c.take((size_t)C * 8), o_k1 = c.take((size_t)C * 8), o_v0 = c.take((size_t)C * 4),
                         o_v1 = c.take((size_t)C * 4), o_h = c.take((size_t)256 * std::max(nblocks, 1u) * 4);
            void* blob = nullptr;
            int rc = dev_alloc(c.cur, &blob);
            if (rc) return rc;
            struct Guard { void* p; ~Guard() { dev_free(p); } } guard{blob};
            unsigned char* b = (unsigned char*)blob;
            uint64_t* keys[2] = {(uint64_t*)(b + o_k0), (uint64_t*)(b + o_k1)};
            uint32_t* vals[2] = {(uint32_t*)(b + o_v0), (uint32_t*)(b + o_v1)};
            std::vector<uint64_t> h_cd(C);
            std::vector<uint32_t> h_order(C);
            if (C) {
                if (L) k_link_cost<<<(L + 255) / 256, 256, 0, counted(st)>>>(t->d_alpha, t->d_bpp, L, P.chunk_bytes, (uint64_t*)(b + o_w));
                if (NS) {
                    const size_t smem = (size_t)N * 8;
                    if (smem > 200 * 1024) return PCCL_ERR_UNSUPPORTED;
                    if (smem > 48 * 1024) CU(cudaFuncSetAttribute(k_distances, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                    k_distances<<<NS, 512, smem, counted(st)>>>(pv.esrc, pv.edst, (uint64_t*)(b + o_w), N, L, ph.d_sources, (uint64_t*)(b + o_D));
                }
                k_cdist<<<(C + 255) / 256, 256, 0, counted(st)>>>(ph.d_cond_src, ph.d_dest_off, ph.d_dests, C, ph.d_sidx, (uint64_t*)(b + o_D), N,
                                                                  (uint64_t*)(b + o_cd), keys[0], vals[0]);
                const int cur = radix_sort_pairs(keys, vals, C, 64, (uint32_t*)(b + o_h), nblocks, 0);
                CU(cudaGetLastError());
                CU(cudaMemcpyAsync(h_cd.data(), b + o_cd, (size_t)C * 8, cudaMemcpyDeviceToHost, st));
                CU(cudaMemcpyAsync(h_order.data(), vals[cur], (size_t)C * 4, cudaMemcpyDeviceToHost, st));
                CU(cudaStreamSynchronize(st));
            }
            // re-index the conditions with the device's order (no arithmetic of the method here)
            Phase pp;
            pp.transposed = ph.transposed;
            pp.sources = ph.sources; pp.sidx = ph.sidx; pp.dsts = ph.dsts; pp.didx = ph.didx;
            pp.cond_src.resize(C); pp.dest_off.resize((size_t)C + 1); pp.dests.resize(ph.dests.size()); pp.dchunk.resize(ph.dests.size());
            pp.orig.resize(C); pp.cls.resize(C);
            uint64_t nd = 0;
            uint32_t cls = 0;
            pp.dest_off[0] = 0;
            for (uint32_t i = 0; i < C; ++i) {
                const uint32_t c0 = h_order[i];
                if (i > 0 && h_cd[c0] != h_cd[h_order[i - 1]]) ++cls;
                pp.orig[i] = c0; pp.cls[i] = cls;
                pp.cond_src[i] = ph.cond_src[c0];
                for (uint64_t k = ph.dest_off[c0]; k < ph.dest_off[c0 + 1]; ++k) { pp.dests[nd] = ph.dests[k]; pp.dchunk[nd] = i; ++nd; }
                pp.dest_off[i + 1] = nd;
            }
            pp.ncls = C ? cls + 1 : 0;
            int rc2 = phase_upload(pp, N);
            if (rc2) return rc2;
            out.push_back(std::move(pp));
        }
    } catch (const std::bad_alloc&) {
        for (Phase& ph : out) dev_free(ph.blob);
        return PCCL_ERR_NOMEM;
    }
    P.prio_phases = std::move(out);
    return PCCL_OK;
}

struct BfsResult {
    uint64_t M, tmax, conditions, searches, relax, rounds;
    uint32_t grid;
};

// pre / n_pre / t_pre (pipelined All-Reduce, Q26): the reduce phase's records in forward time (device) and their
// largest t_end -- they pre-occupy the links, and a chunk's search starts when its root has received the last of them
int bfs_phase(const pccl_problem& P, const Phase& ph, uint64_t seed, uint64_t t_shift, Rec** out_recs, BfsResult* res,
              Timer& t_setup, Timer& t_loop, Timer& t_emit, const Rec* pre = nullptr, uint64_t n_pre = 0, uint64_t t_pre = 0) {
    const pccl_topology* t = P.topo;
    const uint32_t N = t->N, L = t->L, C = P.C;
    const PhaseView pv = view_of(t, ph.transposed);
    cudaStream_t st = G.stream;
    *out_recs = nullptr;
    memset(res, 0, sizeof(*res));
    if (C == 0 || ph.dests.empty()) return PCCL_OK;
    if (L == 0) return PCCL_ERR_UNREACHABLE;
    uint32_t link_bits = 1;
    while ((1ull << link_bits) < (uint64_t)L) ++link_bits;
    const size_t smem_base = align_up((size_t)N * 20 + ((size_t)N + 1) * 4, 16);
    if (smem_base > 200 * 1024) return PCCL_ERR_UNSUPPORTED;
    // the out-link table and entry 0 of every busy-run row live in shared memory when they fit (32 bytes per link)
    const bool os_in_smem = smem_base + (size_t)L * 32 <= 200 * 1024;
    const size_t smem = smem_base + (os_in_smem ? (size_t)L * 32 : 0);

    // ---- order (Alg. 3 lines 1-7) ----
    t_setup.start();
    const uint32_t NS = (uint32_t)ph.sources.size();
    const uint32_t sort_blocks = (uint32_t)((C + SORT_TILE - 1) / SORT_TILE);
    Carver c;
    const size_t o_w = c.take((size_t)L * 8), o_D = c.take((size_t)NS * N * 8), o_cd = c.take((size_t)C * 8),
                 o_k0 = c.take((size_t)C * 8), o_k1 = c.take((size_t)C * 8), o_v0 = c.take((size_t)C * 4),
                 o_v1 = c.take((size_t)C * 4), o_h = c.take((size_t)256 * sort_blocks * 4), o_ctrl = c.take(sizeof(BfsCtrl)),
                 o_os = c.take((size_t)L * 16);
    const uint32_t pre_blocks = (uint32_t)((n_pre + SORT_TILE - 1) / SORT_TILE);
    const size_t o_rdy = c.take(pre ? (size_t)C * 8 : 0), o_pk0 = c.take(n_pre * 8), o_pk1 = c.take(n_pre * 8),
                 o_pv0 = c.take(n_pre * 4), o_pv1 = c.take(n_pre * 4), o_ph = c.take((size_t)256 * pre_blocks * 4);
    void* blob = nullptr;
    int rc = dev_alloc(c.cur, &blob);
    if (rc) return rc;
    struct Guard { void* p[4] = {nullptr, nullptr, nullptr, nullptr}; ~Guard() { for (void* q : p) dev_free(q); } } guard;
    guard.p[0] = blob;
    unsigned char* b = (unsigned char*)blob;
    uint64_t* d_w = (uint64_t*)(b + o_w);
    uint64_t* d_D = (uint64_t*)(b + o_D);
    uint64_t* d_cdist = (uint64_t*)(b + o_cd);
    uint64_t* keys[2] = {(uint64_t*)(b + o_k0), (uint64_t*)(b + o_k1)};
    uint32_t* vals[2] = {(uint32_t*)(b + o_v0), (uint32_t*)(b + o_v1)};
    uint32_t* ghist = (uint32_t*)(b + o_h);
    BfsCtrl* ctrl = (BfsCtrl*)(b + o_ctrl);
    CU(cudaMemsetAsync(ctrl, 0, sizeof(BfsCtrl), st));
    k_link_cost<<<(L + 255) / 256, 256, 0, counted(st)>>>(t->d_alpha, t->d_bpp, L, P.chunk_bytes, d_w);
    uint4* d_oslot = (uint4*)(b + o_os);
    k_bfs_pack<<<(L + 255) / 256, 256, 0, counted(st)>>>(pv.out_link, pv.edst, d_w, L, d_oslot);
    if (NS) {
        const size_t ds = (size_t)N * 8;
        if (ds > 48 * 1024) CU(cudaFuncSetAttribute(k_distances, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ds));
        k_distances<<<NS, 256, ds, counted(st)>>>(pv.esrc, pv.edst, d_w, N, L, ph.d_sources, d_D);
    }
    const uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
    const unsigned gC = (C + 255) / 256;
    k_bfs_keys<<<gC, 256, 0, counted(st)>>>(ph.d_cond_src, ph.d_dest_off, ph.d_dests, C, ph.d_sidx, d_D, N, k0, k1, d_cdist, keys[0],
                                   vals[0], ctrl);
    int cur = radix_sort_pairs(keys, vals, C, 64, ghist, sort_blocks, 0);          // by (draw, chunk)
    k_bfs_keys2<<<gC, 256, 0, counted(st)>>>(d_cdist, vals[cur], C, keys[cur ^ 1], vals[cur ^ 1]);
    cur = radix_sort_pairs(keys, vals, C, 64, ghist, sort_blocks, cur ^ 1);         // stable, by descending c.dist
    const uint32_t* d_order = vals[cur];
    // pipelined All-Reduce: ready times and the reduce phase's records sorted by (link, t_start)
    unsigned long long* d_ready = nullptr;
    const uint64_t* d_pkeys = nullptr;
    const uint32_t* d_pidx = nullptr;
    uint32_t pre_tbits = 1;
    if (pre && n_pre) {
        while (pre_tbits < 64 && (t_pre >> pre_tbits)) ++pre_tbits;
        if (pre_tbits + link_bits > 64 || n_pre > 0xFFFFFFFFull) return PCCL_ERR_UNSUPPORTED;
        d_ready = (unsigned long long*)(b + o_rdy);
        CU(cudaMemsetAsync(d_ready, 0, (size_t)C * 8, st));
        uint64_t* pk[2] = {(uint64_t*)(b + o_pk0), (uint64_t*)(b + o_pk1)};
        uint32_t* pvv[2] = {(uint32_t*)(b + o_pv0), (uint32_t*)(b + o_pv1)};
        k_bfs_ready<<<(unsigned)((n_pre + 255) / 256), 256, 0, counted(st)>>>(pre, n_pre, ph.d_cond_src, d_ready, pre_tbits, pk[0], pvv[0]);
        const int pc = radix_sort_pairs(pk, pvv, n_pre, pre_tbits + link_bits, (uint32_t*)(b + o_ph), pre_blocks, 0);
        d_pkeys = pk[pc]; d_pidx = pvv[pc];
    }
    CU(cudaGetLastError());
    BfsCtrl* mb = (BfsCtrl*)G.mailbox;
    CU(cudaMemcpyAsync(mb, ctrl, sizeof(BfsCtrl), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (mb->err & 1u) return PCCL_ERR_UNREACHABLE;
    if (mb->err) return PCCL_ERR_INTERNAL;
    const uint32_t nact = mb->nact;
    t_setup.stop();
    if (nact == 0) return PCCL_OK;

    // ---- window size = co-resident CTAs ----
    const void* kbfs = !t->buf_limit.empty() ? (const void*)k_bfs<true> : (const void*)k_bfs<false>;
    if (smem > 40 * 1024) CU(cudaFuncSetAttribute(kbfs, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kbfs, (int)BFS_THREADS, smem));
    if (occ < 1) return PCCL_ERR_CUDA;
    // switch model: per limited node a sorted table of the stays committed so far; conditions are then
    // routed strictly one after another (a one-condition window), so a search sees every earlier stay
    const bool sw_model = !t->buf_limit.empty();
    std::vector<uint32_t> h_swidx;
    uint32_t n_lim = 0;
    if (sw_model) {
        try {
            h_swidx.assign(N, NONE32);
        } catch (const std::bad_alloc&) {
            return PCCL_ERR_NOMEM;
        }
        for (uint32_t v = 0; v < N; ++v)
            if (t->buf_limit[v] != 0xFFFFFFFFu) h_swidx[v] = n_lim++;
        if ((uint64_t)std::max(n_lim, 1u) * nact * 16 > ((uint64_t)1 << 30)) return PCCL_ERR_UNSUPPORTED;
    }
    uint32_t Bwant = (uint32_t)G.sm_count;   // one 1024-thread CTA per SM
    if (const uint64_t o = G.opt_bfs_window) Bwant = (uint32_t)std::min<uint64_t>((uint64_t)occ * (uint64_t)G.sm_count, o);
    const uint32_t B = sw_model ? 1u : std::max(1u, std::min(Bwant, nact));

    // ---- record capacity: a tree has at most N - 1 transfers; retried with the exact count if short ----
    uint64_t cap = 0;
    for (uint32_t ci = 0; ci < C; ++ci) {
        const uint64_t nd = ph.dest_off[ci + 1] - ph.dest_off[ci];
        cap += std::min<uint64_t>((uint64_t)N - 1, nd * 32);
    }
    // busy runs per link row: 256 (4 KB), more when many conditions share few links (<= 4096 and <= 1 GB in all);
    // a full row makes the kernel stop and the phase is rerun with 4 R
    uint32_t R = 256;
    while (R < 4096 && R < nact / std::max(L, 1u) && (size_t)L * (R * 2) * 16 <= ((size_t)1 << 30)) R *= 2;
    if (const uint64_t o = G.opt_bfs_rows) R = (uint32_t)std::min<uint64_t>(std::max<uint64_t>(8, o), 1u << 20);   // (tests: force the rerun)
    for (int attempt = 0; attempt < 8; ++attempt) {
        Carver w2;
        const size_t o_runs = w2.take((size_t)L * R * 16), o_rn = w2.take((size_t)L * 4), o_rs = w2.take((size_t)L * B * 8),
                     o_rp = w2.take((size_t)L * B * 4), o_tl = w2.take((size_t)B * N * 4), o_ts = w2.take((size_t)B * N * 8);
        const size_t nl1 = std::max(n_lim, 1u);
        const size_t o_swi = w2.take(sw_model ? (size_t)N * 4 : 0), o_swl = w2.take(sw_model ? (size_t)N * 4 : 0),
                     o_swm = w2.take(sw_model ? (size_t)N : 0), o_sba = w2.take(sw_model ? nl1 * nact * 8 : 0),
                     o_sbr = w2.take(sw_model ? nl1 * nact * 8 : 0), o_sbn = w2.take(sw_model ? nl1 * 4 : 0),
                     o_sta = w2.take(sw_model ? nl1 * B * 8 : 0), o_str = w2.take(sw_model ? nl1 * B * 8 : 0);
        void* ws = nullptr;
        rc = dev_alloc(w2.cur, &ws);
        if (rc) return rc;
        guard.p[1] = ws;
        Rec* raw = nullptr;
        rc = dev_alloc(std::max<uint64_t>(cap, 1) * sizeof(Rec), (void**)&raw);
        if (rc) return rc;
        guard.p[2] = raw;
        unsigned char* q = (unsigned char*)ws;
        BfsArgs a;
        a.N = N; a.L = L; a.R = R; a.B = B; a.link_bits = link_bits; a.nact = nact;
        a.os_in_smem = os_in_smem ? 1u : 0u; a.os_smem_off8 = (uint32_t)(smem_base / 8);
        {
            const uint32_t md = std::max(1u, ph.transposed ? t->max_in : t->max_out);
            a.deg_shift = 0;
            while ((1u << a.deg_shift) < md && a.deg_shift < 5) ++a.deg_shift;
        }
        a.out_off = ph.transposed ? t->d_in_off : t->d_out_off; a.oslot = d_oslot;
        a.esrc = pv.esrc; a.edst = pv.edst; a.psrc = t->d_src; a.pdst = t->d_dst; a.w = d_w;
        a.cond_src = ph.d_cond_src; a.dest_off = ph.d_dest_off; a.dests = ph.d_dests; a.order = d_order;
        a.runs = (ulonglong2*)(q + o_runs); a.rl_n = (uint32_t*)(q + o_rn); a.rl_start = (uint64_t*)(q + o_rs);
        a.rl_pos = (uint32_t*)(q + o_rp); a.tr_link = (uint32_t*)(q + o_tl); a.tr_start = (uint64_t*)(q + o_ts);
        a.out = raw; a.out_cap = cap; a.t_offset = 0; a.ctrl = ctrl;
        a.t_ready = d_ready;
        a.swidx = nullptr; a.buf_limit = nullptr; a.no_mcast = nullptr; a.n_lim = 0; a.sb_cap = 0;
        a.sb_arr = a.sb_rel = a.st_arr = a.st_rel = nullptr; a.sb_n = nullptr;
        if (sw_model) {
            a.swidx = (uint32_t*)(q + o_swi); a.buf_limit = (uint32_t*)(q + o_swl); a.no_mcast = (unsigned char*)(q + o_swm);
            a.n_lim = n_lim; a.sb_cap = nact;
            a.sb_arr = (unsigned long long*)(q + o_sba); a.sb_rel = (unsigned long long*)(q + o_sbr); a.sb_n = (uint32_t*)(q + o_sbn);
            a.st_arr = (unsigned long long*)(q + o_sta); a.st_rel = (unsigned long long*)(q + o_str);
            CU(cudaMemcpyAsync(q + o_swi, h_swidx.data(), (size_t)N * 4, cudaMemcpyHostToDevice, st));
            CU(cudaMemcpyAsync(q + o_swl, t->buf_limit.data(), (size_t)N * 4, cudaMemcpyHostToDevice, st));
            CU(cudaMemcpyAsync(q + o_swm, t->no_mcast.data(), (size_t)N, cudaMemcpyHostToDevice, st));
        }
        t_loop.start();
        k_bfs_init<<<(std::max(std::max(L, n_lim), 1u) + 255) / 256, 256, 0, counted(st)>>>(a);
        if (d_pkeys) k_bfs_preoccupy<<<(L + 127) / 128, 128, 0, counted(st)>>>(a, pre, n_pre, d_pkeys, d_pidx, pre_tbits);
        void* args[] = {(void*)&a};
        CU(cudaLaunchCooperativeKernel(kbfs, dim3(B), dim3(BFS_THREADS), args, smem, counted(st)));
        CU(cudaMemcpyAsync(mb, ctrl, sizeof(BfsCtrl), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        t_loop.stop();
        const uint32_t err = mb->err;
        if (err & 1u) return PCCL_ERR_UNREACHABLE;
        if (err & 2u) return PCCL_ERR_UNSUPPORTED;          // times do not fit beside the link id in 64 bits
        if (err & 16u) return PCCL_ERR_INTERNAL;
        if (err & (4u | 8u)) {                              // a busy-run row or the record buffer was too small
            if (err & 4u) R *= 4;
            if (err & 8u) cap = mb->nrec;
            dev_free(ws); dev_free(raw);
            guard.p[1] = guard.p[2] = nullptr;
            CU(cudaMemsetAsync(&ctrl->err, 0, 4, st));
            continue;
        }
#ifdef PCCL_BFS_PROFILE
        fprintf(stderr, "[pccl bfs] rounds %llu searches %llu sweeps %llu relax %llu | CTA 0: search %.2f ms check %.2f ms commit %.2f ms | "
                        "per search: sweeps %.2f us filter %.2f us | R %u B %u\n",
                mb->rounds, mb->searches, mb->iters, mb->relax, mb->ns_search * 1e-6, mb->ns_check * 1e-6, mb->ns_commit * 1e-6,
                mb->searches ? mb->ns_sweeps * 1e-3 / mb->searches : 0.0, mb->searches ? mb->ns_filter * 1e-3 / mb->searches : 0.0, R, B);
#endif
        const uint64_t M = mb->nrec;
        res->M = M; res->tmax = mb->tmax; res->conditions = nact; res->searches = mb->searches; res->relax = mb->relax;
        res->rounds = mb->rounds; res->grid = B;
        dev_free(ws);
        guard.p[1] = nullptr;
        if (M == 0) return PCCL_OK;
        Rec* sorted = nullptr;
        rc = dev_alloc(M * sizeof(Rec), (void**)&sorted);
        if (rc) return rc;
        t_emit.start();
        rc = reverse_sorted(raw, M, mb->tmax, L, sorted, ph.transposed, ph.transposed ? 0 : t_shift);
        if (rc) { dev_free(sorted); return rc; }
        t_emit.stop();
        *out_recs = sorted;
        return PCCL_OK;
    }
    return PCCL_ERR_NOMEM;
}

}  // namespace

extern "C" int pccl_problem_synthesize(pccl_problem_t* P, uint64_t seed, uint32_t flags, pccl_schedule_t** out) {
    SERIALISE;
    if (!P || !out) return PCCL_ERR_INVALID;
    int rc = problem_upload(P, false);
    DBGT("upload enqueued");
    if (rc) return rc;
    pccl_schedule* S = new (std::nothrow) pccl_schedule();
    if (!S) { if (cudaStreamSynchronize(G.stream) != cudaSuccess) (void)cudaGetLastError(); return PCCL_ERR_NOMEM; }
    memset(&S->stats, 0, sizeof(S->stats));
    S->stats.mode = (uint32_t)P->mode;
    Timers tm;
    Timer &t_setup = tm.setup, &t_loop = tm.loop, &t_emit = tm.emit;
    const bool timed = (flags & PCCL_FLAG_TIME_LOOP) != 0;
    t_setup.init(timed); t_loop.init(timed); t_emit.init(timed);

    Work W;
    Rec* out_recs = nullptr;   // final records
    Rec* raw = nullptr;        // raw records of a reduce phase
    Rec* stage1 = nullptr;     // sorted phase-1 records of an all-reduce
    uint64_t M1 = 0, T1 = 0;
    auto fail = [&](int code) {
        dev_free(W.blob); dev_free(out_recs); dev_free(raw); dev_free(stage1);
        if (cudaStreamSynchronize(G.stream) != cudaSuccess) (void)cudaGetLastError();
        pinned_put(S->h_recs, S->h_bytes);
        delete S;
        return code;
    };
    const uint32_t L = P->topo->L;
    const bool dist_pick = (flags & PCCL_FLAG_DIST_PICK) != 0;
    if (dist_pick) {
        if (flags & (PCCL_FLAG_BFS | PCCL_FLAG_DYNAMIC_RELAY | PCCL_FLAG_RESCAN | PCCL_FLAG_DENSE_SWEEP | PCCL_FLAG_TWO_BARRIERS |
                     PCCL_FLAG_BARRIER_LOOP | PCCL_FLAG_TRACE)) return fail(PCCL_ERR_UNSUPPORTED);
        rc = prio_prepare(*P);
        if (rc) return fail(rc);
    }
    for (size_t pi = 0; pi < P->phases.size(); ++pi) {
        const Phase& ph = dist_pick ? P->prio_phases[pi] : P->phases[pi];
        const bool last = pi + 1 == P->phases.size();
        if (flags & PCCL_FLAG_BFS) {   // the paper's per-condition search instead of the matching loop
            BfsResult br;
            Rec* recs = nullptr;
            // All-Reduce with PCCL_FLAG_PIPELINE: the copy phase is routed against the reduce phase's intervals, each chunk
            // from the time its root is complete (Q26) -- no shift, the two record lists are merged afterwards
            const bool pipelined = (flags & PCCL_FLAG_PIPELINE) && pi == 1 && stage1 != nullptr;
            if ((flags & PCCL_FLAG_PIPELINE) && P->mode == 2 && !P->topo->buf_limit.empty()) return fail(PCCL_ERR_UNSUPPORTED);
            const uint64_t toff = (pi == 0 || pipelined) ? 0 : T1;
            rc = pipelined ? bfs_phase(*P, ph, seed, 0, &recs, &br, t_setup, t_loop, t_emit, stage1, M1, T1)
                           : bfs_phase(*P, ph, seed, toff, &recs, &br, t_setup, t_loop, t_emit);
            if (rc) return fail(rc);
            S->stats.wants_total += br.M;
            S->stats.events += br.conditions;
            S->stats.rows_scanned += br.searches;
            S->stats.links_scanned += br.relax;
            S->stats.slow_picks += br.rounds;
            S->stats.grid_blocks = br.grid;
            if (ph.transposed) {
                if (last) { out_recs = recs; S->M = br.M; S->T = br.tmax; } else stage1 = recs;
                M1 = br.M; T1 = br.tmax;
                S->stats.time_phase1_ps = br.tmax;
            } else {
                const uint64_t base = (pi == 0) ? 0 : M1;
                if (base) {
                    rc = dev_alloc((base + br.M) * sizeof(Rec), (void**)&out_recs);
                    if (rc) { dev_free(recs); return fail(rc); }
                    if (cudaMemcpyAsync(out_recs, stage1, base * sizeof(Rec), cudaMemcpyDeviceToDevice, G.stream) != cudaSuccess ||
                        (br.M && cudaMemcpyAsync(out_recs + base, recs, br.M * sizeof(Rec), cudaMemcpyDeviceToDevice, G.stream) !=
                                     cudaSuccess)) {
                        (void)cudaGetLastError();
                        dev_free(recs);
                        return fail(PCCL_ERR_CUDA);
                    }
                    dev_free(recs);
                    if (pipelined && br.M) {   // the phases overlap in time: one sort of the concatenation by (t_start, link)
                        Rec* merged = nullptr;
                        rc = dev_alloc((base + br.M) * sizeof(Rec), (void**)&merged);
                        if (rc) return fail(rc);
                        t_emit.start();
                        rc = reverse_sorted(out_recs, base + br.M, std::max(T1, br.tmax), L, merged, false, 0);
                        t_emit.stop();
                        if (rc) { dev_free(merged); return fail(rc); }
                        dev_free(out_recs);
                        out_recs = merged;
                    }
                } else {
                    out_recs = recs;
                }
                S->M = base + br.M;
                S->T = pipelined ? std::max(T1, br.tmax) : toff + br.tmax;
            }
            continue;
        }
        if (!P->topo->buf_limit.empty()) return fail(PCCL_ERR_UNSUPPORTED);   // the switch model belongs to PCCL_FLAG_BFS
        if ((flags & PCCL_FLAG_PIPELINE) && P->mode == 2) return fail(PCCL_ERR_UNSUPPORTED);   // and so does the pipelined All-Reduce
        if (!W.blob) { rc = work_alloc(*P, W); if (rc) return fail(rc); }
        uint64_t M = 0;
        t_setup.start();
        const bool dynamic = (flags & PCCL_FLAG_DYNAMIC_RELAY) != 0;
        // the barrier-free loop applies to the static thin relay tree with kept counts, at most 8 in-links per node and
        // one warp per destination resident (pccl_loop2.cuh); everything else runs the barrier loops
        const uint32_t deg_view = ph.transposed ? P->topo->max_out : P->topo->max_in;
        const bool plan_async = !dynamic && !(flags & (PCCL_FLAG_RESCAN | PCCL_FLAG_DENSE_SWEEP | PCCL_FLAG_TWO_BARRIERS |
                                                      PCCL_FLAG_BARRIER_LOOP | PCCL_FLAG_TRACE)) &&
                                deg_view <= A2_MAX_IN && P->topo->N <= (uint32_t)G.sm_count * A2_MAX_WARPS;
        uint64_t M_thin = 0;
        if (dynamic) {   // the thin relay tree's transfer count sizes the dynamic rule's record buffer (below)
            rc = phase_setup(*P, ph, W, seed, &M_thin, false, false);
            if (rc) return fail(rc);
        }
        DBGT("before phase_setup");
        rc = phase_setup(*P, ph, W, seed, &M, dynamic, plan_async);
        DBGT("phase_setup (synced)");
        if (rc) return fail(rc);
        t_setup.stop();
        S->stats.wants_total += M;
        // thin relay tree: exactly M transfers.  dynamic rule: at most M (a (node, chunk) pair is claimed at most once),
        // in practice a little more than the thin tree's count (config 4: 58 M initial wants, 1.573 M thin-tree transfers,
        // 1.579 M with the rule): the record buffer holds 1.25 x the thin tree's count and, if that is short, the phase
        // is rerun with the exact count the first run reports
        uint64_t cap = dynamic ? std::min<uint64_t>(M, M_thin + M_thin / 4 + P->topo->N + 1024) : M;
        if (dynamic && G.opt_dyn_records) cap = std::min<uint64_t>(M, G.opt_dyn_records);   // (tests: force the rerun)
        LoopResult lr;
        memset(&lr, 0, sizeof(lr));
        for (int attempt = 0;; ++attempt) {
            if (attempt > 0) {   // rerun: steps A..C again (the loop consumed the wants), exact capacity
                if (cap > (1ull << 31)) return fail(PCCL_ERR_NOMEM);
                uint64_t M2 = 0;
                rc = phase_setup(*P, ph, W, seed, &M2, dynamic, false);
                if (rc) return fail(rc);
            }
            if (ph.transposed) {
                rc = dev_alloc(cap * sizeof(Rec), (void**)&raw);
                if (rc) return fail(rc);
                rc = phase_loop(*P, ph, W, seed, flags, raw, cap, 0, &lr, &tm, &S->trace);
                if (rc == PCCL_ERR_NOMEM && dynamic && attempt == 0 && lr.total > cap && lr.total <= M) {
                    dev_free(raw); raw = nullptr;
                    cap = lr.total;
                    continue;
                }
                if (rc) return fail(rc);
                if (dynamic ? lr.total > M : lr.total != M) return fail(PCCL_ERR_INTERNAL);
                M = lr.total;
                Rec* dst = nullptr;
                rc = dev_alloc(M * sizeof(Rec), (void**)&dst);
                if (rc) return fail(rc);
                if (last) out_recs = dst; else stage1 = dst;
                t_emit.start();
                rc = reverse_sorted(raw, M, lr.tmax, L, dst, true, 0);
                if (rc) return fail(rc);
                t_emit.stop();
                dev_free(raw);
                raw = nullptr;
                M1 = M; T1 = lr.tmax;
                if (last) { S->M = M; S->T = lr.tmax; }
                S->stats.time_phase1_ps = lr.tmax;
            } else {
                const uint64_t base = (pi == 0) ? 0 : M1;
                const uint64_t toff = (pi == 0) ? 0 : T1;
                rc = dev_alloc((base + cap) * sizeof(Rec), (void**)&out_recs);
                if (rc) return fail(rc);
                if (base) {
                    if (cudaMemcpyAsync(out_recs, stage1, base * sizeof(Rec), cudaMemcpyDeviceToDevice, G.stream) != cudaSuccess) {
                        (void)cudaGetLastError();
                        return fail(PCCL_ERR_CUDA);
                    }
                }
                // a schedule that goes to the host anyway is streamed out while the loop runs (single copy phase)
                bool streamed = false;
                if (base == 0 && last && !dynamic && cap && !(flags & PCCL_FLAG_KEEP_ON_DEVICE)) {
                    S->h_bytes = cap * sizeof(Rec);
                    S->h_recs = pinned_get(S->h_bytes);   // null: no streaming, the download reports the failure
                }
                DBGT("before phase_loop");
                rc = phase_loop(*P, ph, W, seed, flags, out_recs + base, cap, toff, &lr, &tm, &S->trace, (Rec*)S->h_recs, &streamed);
                DBGT("phase_loop returns");
                if (rc == PCCL_ERR_NOMEM && dynamic && attempt == 0 && lr.total > cap && lr.total <= M) {
                    dev_free(out_recs); out_recs = nullptr;
                    cap = lr.total;
                    continue;
                }
                if (rc) return fail(rc);
                if (dynamic ? lr.total > M : lr.total != M) return fail(PCCL_ERR_INTERNAL);
                M = lr.total;
                S->M = base + M;
                S->T = toff + lr.tmax;
                S->downloaded = streamed;
            }
            break;
        }
        S->stats.events += lr.events;
        S->stats.rows_scanned += lr.rows;
        S->stats.links_scanned += lr.links;
        S->stats.slow_picks += lr.slow;
        S->stats.bytes_requested += lr.bytes;
        S->stats.grid_blocks = lr.grid;
        S->stats.row_bytes = (uint64_t)W.Wp * 8;
    }
    dev_free(W.blob); W.blob = nullptr;
    dev_free(stage1); stage1 = nullptr;
    S->d_recs = out_recs;
    S->n_links = P->topo->L;
    S->n_npus = P->topo->N;
    S->stats.loop_ms = t_loop.total(); S->stats.setup_ms = t_setup.total(); S->stats.emit_ms = t_emit.total();
    if (!(flags & PCCL_FLAG_KEEP_ON_DEVICE)) {
        if (S->M && !pccl_schedule_transfers(S)) { pccl_schedule_destroy(S); return PCCL_ERR_CUDA; }
    }
    *out = S;
    return PCCL_OK;
}

extern "C" int pccl_synthesize(const pccl_topology_t* topo, const uint32_t* group_members, uint32_t n_members,
                               const pccl_condition_t* pre, const pccl_condition_t* post, uint64_t chunk_bytes,
                               uint64_t seed, pccl_schedule_t** out) {
    if (!out) return PCCL_ERR_INVALID;
    DBGT("-- pccl_synthesize");
    pccl_problem_t* P = nullptr;
    int rc = pccl_problem_create(topo, group_members, n_members, pre, post, chunk_bytes, &P);
    DBGT("problem_create (normalise)");
    if (rc) return rc;
    pccl_schedule_t* S = nullptr;
    rc = pccl_problem_synthesize(P, seed, 0, &S);
    DBGT("problem_synthesize returns");
    pccl_problem_destroy(P);
    DBGT("problem_destroy");
    if (rc) return rc;
    *out = S;
    return PCCL_OK;
}

// -----------------------------------------------------------------------------------------
// schedule accessors
// -----------------------------------------------------------------------------------------
extern "C" uint64_t pccl_schedule_time(const pccl_schedule_t* s) { return s ? s->T : 0; }
extern "C" uint64_t pccl_schedule_size(const pccl_schedule_t* s) { return s ? s->M : 0; }
extern "C" const pccl_transfer_t* pccl_schedule_transfers(pccl_schedule_t* s) {
    SERIALISE;
    if (!s || s->M == 0) return nullptr;
    if (!s->downloaded) {
        if (!s->d_recs) return nullptr;
        const size_t bytes = s->M * sizeof(Rec);
        if (!s->h_recs) { s->h_recs = pinned_get(bytes); s->h_bytes = bytes; }
        if (!s->h_recs) return nullptr;
        if (cudaMemcpyAsync(s->h_recs, s->d_recs, bytes, cudaMemcpyDeviceToHost, G.stream) != cudaSuccess ||
            cudaStreamSynchronize(G.stream) != cudaSuccess) {
            (void)cudaGetLastError();
            return nullptr;
        }
        s->downloaded = true;
    }
    return (const pccl_transfer_t*)s->h_recs;
}
extern "C" const pccl_transfer_t* pccl_schedule_transfers_device(const pccl_schedule_t* s) {
    return s ? (const pccl_transfer_t*)s->d_recs : nullptr;
}
extern "C" void pccl_schedule_destroy(pccl_schedule_t* s) {
    SERIALISE;
    if (!s) return;
    dev_free(s->d_recs);
    pinned_put(s->h_recs, s->h_bytes);
    delete s;
}
static_assert(sizeof(pccl_op_t) == sizeof(Op), "op layout");

extern "C" int pccl_schedule_programs(pccl_schedule_t* s, uint64_t* offsets, pccl_op_t* ops) {
    SERIALISE;
    if (!s || !offsets || (s->M && !ops)) return PCCL_ERR_INVALID;
    const uint32_t N = s->n_npus;
    const uint64_t M = s->M, n = 2 * M;
    if (M == 0) {
        for (uint32_t v = 0; v <= N; ++v) offsets[v] = 0;
        return PCCL_OK;
    }
    if (!s->d_recs) return PCCL_ERR_INVALID;
    uint32_t link_bits = 1;
    while ((1ull << link_bits) < (uint64_t)s->n_links) ++link_bits;
    uint32_t t_bits = 1;
    while (t_bits < 64 && (s->T >> t_bits)) ++t_bits;
    uint32_t node_bits = 1;
    while ((1ull << node_bits) < (uint64_t)N) ++node_bits;
    if (t_bits + 1 + link_bits > 64 || n > 0xFFFFFFFFull) return PCCL_ERR_UNSUPPORTED;
    cudaStream_t st = G.stream;
    const uint32_t nblocks = (uint32_t)((n + SORT_TILE - 1) / SORT_TILE);
    Carver c;
    const size_t o_k0 = c.take(n * 8), o_k1 = c.take(n * 8), o_v0 = c.take(n * 4), o_v1 = c.take(n * 4),
                 o_h = c.take((size_t)256 * nblocks * 4), o_ops = c.take(n * sizeof(Op)), o_off = c.take(((size_t)N + 1) * 8);
    void* blob = nullptr;
    int rc = dev_alloc(c.cur, &blob);
    if (rc) return rc;
    unsigned char* b = (unsigned char*)blob;
    uint64_t* keys[2] = {(uint64_t*)(b + o_k0), (uint64_t*)(b + o_k1)};
    uint32_t* vals[2] = {(uint32_t*)(b + o_v0), (uint32_t*)(b + o_v1)};
    uint32_t* ghist = (uint32_t*)(b + o_h);
    const unsigned g256 = (unsigned)((n + 255) / 256);
    // stable LSD order: first by (time, kind, link), then by node
    k_ops_keys<<<g256, 256, 0, counted(st)>>>(s->d_recs, M, link_bits, keys[0], vals[0]);
    int cur = radix_sort_pairs(keys, vals, n, t_bits + 1 + link_bits, ghist, nblocks, 0);
    k_ops_nodes<<<g256, 256, 0, counted(st)>>>(s->d_recs, M, vals[cur], keys[cur]);
    cur = radix_sort_pairs(keys, vals, n, node_bits, ghist, nblocks, cur);
    k_ops_gather<<<g256, 256, 0, counted(st)>>>(s->d_recs, M, vals[cur], (Op*)(b + o_ops));
    k_ops_offsets<<<(N + 1 + 255) / 256, 256, 0, counted(st)>>>(keys[cur], n, N, (uint64_t*)(b + o_off));
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(ops, b + o_ops, n * sizeof(Op), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(offsets, b + o_off, ((size_t)N + 1) * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    dev_free(blob);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return PCCL_ERR_CUDA; }
    return PCCL_OK;
}

extern "C" int64_t pccl_schedule_trace(const pccl_schedule_t* s, uint64_t* out, uint64_t cap) {
    if (!s || (cap && !out)) return PCCL_ERR_INVALID;
    const uint64_t n = s->trace.size();
    if (n && cap) memcpy(out, s->trace.data(), (size_t)std::min(n, cap) * 8);
    return (int64_t)n;
}
extern "C" int pccl_schedule_stats(const pccl_schedule_t* s, pccl_stats_t* out) {
    if (!s || !out) return PCCL_ERR_INVALID;
    *out = s->stats;
    return PCCL_OK;
}

// -----------------------------------------------------------------------------------------
// single rows for parity tests
// -----------------------------------------------------------------------------------------
extern "C" int pccl_device_philox(const uint32_t* ctr, uint64_t n, const uint32_t key[2], uint32_t* out) {
    SERIALISE;
    if ((n && (!ctr || !out)) || !key) return PCCL_ERR_INVALID;
    if (n == 0) return PCCL_OK;
    int rc = ensure_device();
    if (rc) return rc;
    void* d = nullptr;
    rc = dev_alloc(n * 32, &d);
    if (rc) return rc;
    uint32_t* dc = (uint32_t*)d;
    uint32_t* dout = dc + 4 * n;
    cudaStream_t st = G.stream;
    cudaError_t e = cudaMemcpyAsync(dc, ctr, n * 16, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        k_philox<<<(unsigned)((n + 255) / 256), 256, 0, counted(st)>>>(dc, n, key[0], key[1], dout);
        e = cudaMemcpyAsync(out, dout, n * 16, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    dev_free(d);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return PCCL_ERR_CUDA; }
    return PCCL_OK;
}

extern "C" int pccl_device_link_costs(pccl_topology_t* t, uint64_t chunk_bytes, uint64_t* out) {
    SERIALISE;
    if (!t || !out || chunk_bytes == 0) return PCCL_ERR_INVALID;
    int rc = topo_upload(t);
    if (rc) return rc;
    if (t->L == 0) return PCCL_OK;
    void* d = nullptr;
    rc = dev_alloc((size_t)t->L * 8, &d);
    if (rc) return rc;
    cudaStream_t st = G.stream;
    k_link_cost<<<(t->L + 255) / 256, 256, 0, counted(st)>>>(t->d_alpha, t->d_bpp, t->L, chunk_bytes, (uint64_t*)d);
    cudaError_t e = cudaMemcpyAsync(out, d, (size_t)t->L * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    dev_free(d);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return PCCL_ERR_CUDA; }
    return PCCL_OK;
}

extern "C" int pccl_device_distances(pccl_topology_t* t, uint64_t chunk_bytes, uint32_t src, int transposed,
                                     uint64_t* out) {
    SERIALISE;
    if (!t || !out || chunk_bytes == 0 || src >= t->N) return PCCL_ERR_INVALID;
    int rc = topo_upload(t);
    if (rc) return rc;
    const size_t N = t->N, L = t->L;
    if (N * 8 > 200 * 1024) return PCCL_ERR_UNSUPPORTED;
    Carver c;
    const size_t o_w = c.take(L * 8), o_D = c.take(N * 8), o_s = c.take(4);
    void* d = nullptr;
    rc = dev_alloc(c.cur, &d);
    if (rc) return rc;
    unsigned char* b = (unsigned char*)d;
    cudaStream_t st = G.stream;
    const PhaseView pv = view_of(t, transposed != 0);
    cudaError_t e = cudaMemcpyAsync(b + o_s, &src, 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && N * 8 > 48 * 1024)
        e = cudaFuncSetAttribute(k_distances, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(N * 8));
    if (e == cudaSuccess) {
        if (L) k_link_cost<<<(unsigned)((L + 255) / 256), 256, 0, counted(st)>>>(t->d_alpha, t->d_bpp, (uint32_t)L, chunk_bytes, (uint64_t*)(b + o_w));
        k_distances<<<1, 256, N * 8, counted(st)>>>(pv.esrc, pv.edst, (uint64_t*)(b + o_w), (uint32_t)N, (uint32_t)L, (uint32_t*)(b + o_s), (uint64_t*)(b + o_D));
        e = cudaMemcpyAsync(out, b + o_D, N * 8, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    dev_free(d);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return PCCL_ERR_CUDA; }
    return PCCL_OK;
}

extern "C" int64_t pccl_device_wants(pccl_problem_t* P, uint32_t phase, uint64_t seed, pccl_pair_t* out, uint64_t cap) {
    SERIALISE;
    if (!P || phase >= P->phases.size() || (cap && !out)) return PCCL_ERR_INVALID;
    int rc = pccl_problem_upload(P);
    if (rc) return rc;
    const Phase& ph = P->phases[phase];
    Work W;
    rc = work_alloc(*P, W);
    if (rc) return rc;
    uint64_t M = 0;
    rc = phase_setup(*P, ph, W, seed, &M);
    if (rc) { dev_free(W.blob); return rc; }
    const uint32_t N = P->topo->N;
    // node bases from wants_cnt (host exclusive scan; accessor only)
    std::vector<uint32_t> wc;
    std::vector<uint64_t> base;
    try {
        wc.assign(N, 0);
        base.assign((size_t)N + 1, 0);
    } catch (const std::bad_alloc&) {
        dev_free(W.blob);
        return PCCL_ERR_NOMEM;
    }
    cudaStream_t st = G.stream;
    cudaError_t e = cudaMemcpyAsync(wc.data(), W.wants_cnt, (size_t)N * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { (void)cudaGetLastError(); dev_free(W.blob); return PCCL_ERR_CUDA; }
    for (uint32_t v = 0; v < N; ++v) base[v + 1] = base[v] + wc[v];
    const uint64_t n_out = std::min<uint64_t>(M, cap);
    void* d = nullptr;
    Carver c;
    const size_t o_b = c.take(((size_t)N + 1) * 8), o_p = c.take(n_out * 8);
    rc = dev_alloc(c.cur, &d);
    if (rc) { dev_free(W.blob); return rc; }
    unsigned char* b = (unsigned char*)d;
    e = cudaMemcpyAsync(b + o_b, base.data(), ((size_t)N + 1) * 8, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && N) {
        k_wants_pairs<<<(N + 3) / 4, 128, 0, counted(st)>>>(W.wants, N, W.Wp, (const uint64_t*)(b + o_b), (uint32_t*)(b + o_p), n_out);
        if (n_out) e = cudaMemcpyAsync(out, b + o_p, n_out * 8, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    dev_free(d);
    dev_free(W.blob);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return PCCL_ERR_CUDA; }
    return (int64_t)M;
}

// a5: candidate counts |have[src_l] & wants[dst_l]| of every link at t = 0 by the streaming sweep kernel, timed alone
extern "C" int pccl_device_candidate_sweep(pccl_problem_t* P, uint32_t phase, uint64_t seed, uint32_t flags, uint32_t iters,
                                           float* ms_per_sweep, uint64_t* bytes_per_sweep, uint32_t* totals) {
    SERIALISE;
    if (!P || phase >= P->phases.size() || iters == 0) return PCCL_ERR_INVALID;
    int rc = pccl_problem_upload(P);
    if (rc) return rc;
    const Phase& ph = P->phases[phase];
    Work W;
    rc = work_alloc(*P, W);
    if (rc) return rc;
    struct Guard { void* p; ~Guard() { dev_free(p); } } guard{W.blob};
    uint64_t M = 0;
    rc = phase_setup(*P, ph, W, seed, &M);
    if (rc) return rc;
    const pccl_topology* t = P->topo;
    const PhaseView pv = view_of(t, ph.transposed);
    LoopArgs a;
    memset(&a, 0, sizeof(a));
    a.N = t->N; a.L = t->L; a.Wp = W.Wp; a.S = W.S;
    a.esrc = pv.esrc; a.edst = pv.edst; a.in_off = pv.in_off; a.in_link = pv.in_link;
    a.have = W.have; a.wants = W.wants; a.gcnt = W.gcnt; a.gtot = W.gtot;
    cudaStream_t st = G.stream;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        (void)cudaGetLastError();
        if (e0) cudaEventDestroy(e0);
        return PCCL_ERR_CUDA;
    }
    struct EvGuard { cudaEvent_t a, b; ~EvGuard() { cudaEventDestroy(a); cudaEventDestroy(b); } } evg{e0, e1};
    rc = launch_count_sweep(a, flags);                       // warm-up (and the result)
    if (rc) return rc;
    CU(cudaEventRecord(e0, st));
    for (uint32_t i = 0; i < iters; ++i) { rc = launch_count_sweep(a, flags); if (rc) return rc; }
    CU(cudaEventRecord(e1, st));
    CU(cudaEventSynchronize(e1));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    if (ms_per_sweep) *ms_per_sweep = ms / (float)iters;
    // algorithmic bytes of one sweep: one wants row per node with in-links and one have row per link
    if (bytes_per_sweep) {
        uint64_t rows = t->L;
        for (uint32_t v = 0; v < t->N; ++v) {
            const uint32_t deg = ph.transposed ? t->out_off[v + 1] - t->out_off[v] : t->in_off[v + 1] - t->in_off[v];
            rows += (deg + NB - 1) / NB;
        }
        *bytes_per_sweep = rows * (uint64_t)W.Wp * 8;
    }
    if (totals && t->L) {
        CU(cudaMemcpyAsync(totals, W.gtot, (size_t)t->L * 4, cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    return PCCL_OK;
}

// sequential 128-bit read of a `bytes`-sized device buffer, `iters` times: ms per pass (the measured ceiling of L2 when the
// buffer fits there, of HBM when it does not, for the access pattern of the bitmap sweeps)
extern "C" int pccl_device_read_bandwidth(uint64_t bytes, uint32_t iters, float* ms_per_pass) {
    SERIALISE;
    if (bytes < 16 || iters == 0 || !ms_per_pass) return PCCL_ERR_INVALID;
    int rc = ensure_device();
    if (rc) return rc;
    void* d = nullptr;
    rc = dev_alloc(bytes + 256, &d);
    if (rc) return rc;
    struct Guard { void* p; ~Guard() { dev_free(p); } } guard{d};
    cudaStream_t st = G.stream;
    CU(cudaMemsetAsync(d, 0x5A, bytes, st));
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_read_sweep, SW_THREADS, 0));
    const uint32_t grid = (uint32_t)std::max(1, occ) * (uint32_t)G.sm_count;
    uint32_t* sink = (uint32_t*)((unsigned char*)d + (bytes & ~(uint64_t)15));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        (void)cudaGetLastError();
        if (e0) cudaEventDestroy(e0);
        return PCCL_ERR_CUDA;
    }
    struct EvGuard { cudaEvent_t a, b; ~EvGuard() { cudaEventDestroy(a); cudaEventDestroy(b); } } evg{e0, e1};
    for (int i = 0; i < 2; ++i) k_read_sweep<<<grid, SW_THREADS, 0, counted(st)>>>((const uint4*)d, bytes / 16, sink);
    CU(cudaEventRecord(e0, st));
    for (uint32_t i = 0; i < iters; ++i) k_read_sweep<<<grid, SW_THREADS, 0, counted(st)>>>((const uint4*)d, bytes / 16, sink);
    CU(cudaEventRecord(e1, st));
    CU(cudaEventSynchronize(e1));
    CU(cudaGetLastError());
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    *ms_per_pass = ms / (float)iters;
    return PCCL_OK;
}

// -----------------------------------------------------------------------------------------
// The entry point that allocates nothing (include/pccl.h: pccl_candidate_totals_static).
//
// Row a5 on the caller's bitmaps by k_count_sweep<true>, its scratch in a fixed array of the device image instead of
// the per-call workspace.  Layout of the part a call uses:  [n_links][S] u32 segment counts (gcnt), then [n_links] u32
// whole-row sums (gtot); the totals handed to the caller are summed from the segment counts by k_static_totals, so
// the result goes THROUGH the array.  In host code `g_static_scratch` is only a stand-in for the symbol: the device
// address comes from cudaGetSymbolAddress, once per device, with that device current.
// -----------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_scratch[PCCL_STATIC_SCRATCH_BYTES];

namespace {

// totals[l] = sum over segments of gcnt[l][s]; one warp per link
__global__ void __launch_bounds__(256) k_static_totals(const uint32_t* __restrict__ gcnt, const uint32_t* __restrict__ gtot,
                                                       uint32_t L, uint32_t S, uint32_t* __restrict__ totals) {
    const uint32_t l = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (l >= L) return;
    uint32_t t = 0;
    for (uint32_t s = lane; s < S; s += 32) t += gcnt[(size_t)l * S + s];
    t = __reduce_add_sync(0xFFFFFFFFu, t);
    // (the whole-row sum is the kernel's own second tally of the same row: a mismatch marks the total as invalid)
    if (lane == 0) totals[l] = (t == gtot[l]) ? t : 0xFFFFFFFFu;
}

constexpr int STATIC_MAX_DEV = 64;
struct StaticDev {
    bool ready = false;
    unsigned char* scratch = nullptr;   // device address of g_static_scratch on this device
    uint32_t resident = 0;              // CTAs of k_count_sweep<true> the device holds at once
};
StaticDev g_static_dev[STATIC_MAX_DEV];
std::mutex g_static_mu;

// once per device, with that device current: the array's device address, the kernel's shared-memory attribute, the
// resident grid.  None of these allocates.
int static_setup(const StaticDev** out) {
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEV) return PCCL_ERR_INVALID;
    std::lock_guard<std::mutex> lk(g_static_mu);
    StaticDev& d = g_static_dev[dev];
    if (!d.ready) {
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return PCCL_ERR_CUDA;
        const void* kern = (const void*)k_count_sweep<true>;
        const size_t smem = (size_t)SW_STAGES * SW_ROWS * SW_SLICE_U4 * 16;
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int occ = 0, sms = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, SW_THREADS, smem));
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        if (occ < 1 || sms < 1) return PCCL_ERR_CUDA;
        d.scratch = (unsigned char*)p;
        d.resident = (uint32_t)occ * (uint32_t)sms;
        d.ready = true;
    }
    *out = &d;
    return PCCL_OK;
}

}  // namespace

extern "C" int pccl_candidate_totals_static(const uint64_t* have, const uint64_t* wants, uint32_t n_npus, uint32_t n_links,
                                            uint32_t words_per_row, const uint32_t* link_src, const uint32_t* in_off,
                                            const uint32_t* in_link, uint32_t* totals, void* stream) {
    if (n_npus == 0 || n_links == 0) return PCCL_OK;
    if (!have || !wants || !link_src || !in_off || !in_link || !totals) return PCCL_ERR_INVALID;
    if (words_per_row == 0 || (words_per_row & 1u)) return PCCL_ERR_INVALID;
    if ((((uintptr_t)have) | ((uintptr_t)wants)) & 15u) return PCCL_ERR_INVALID;
    const uint32_t S = (words_per_row / 2 + SEG_U4 - 1) / SEG_U4;
    const uint64_t need = (uint64_t)n_links * ((uint64_t)S + 1) * 4;
    if (need > (uint64_t)PCCL_STATIC_SCRATCH_BYTES) return PCCL_ERR_TOO_LARGE;
    const StaticDev* d = nullptr;
    int rc = static_setup(&d);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    uint32_t* gcnt = reinterpret_cast<uint32_t*>(d->scratch);
    uint32_t* gtot = gcnt + (size_t)n_links * S;
    // the array keeps the last call's contents: what this call uses starts at zero
    CU(cudaMemsetAsync(d->scratch, 0, (size_t)need, st));
    LoopArgs a;
    memset(&a, 0, sizeof(a));
    a.N = n_npus; a.L = n_links; a.Wp = words_per_row; a.S = S;
    a.esrc = link_src; a.in_off = in_off; a.in_link = in_link;
    a.have = const_cast<uint64_t*>(have); a.wants = const_cast<uint64_t*>(wants);
    a.gcnt = gcnt; a.gtot = gtot;
    a.flags = 1;                                               // (rows whole: the sweep kernel reads its parts count here)
    const size_t smem = (size_t)SW_STAGES * SW_ROWS * SW_SLICE_U4 * 16;
    const uint32_t grid = std::min<uint32_t>(n_npus, d->resident);
    k_count_sweep<true><<<grid, SW_THREADS, smem, counted(st)>>>(a);
    CU(cudaGetLastError());
    k_static_totals<<<(n_links + 7) / 8, 256, 0, counted(st)>>>(gcnt, gtot, n_links, S, totals);
    CU(cudaGetLastError());
    return PCCL_OK;
}
