/* =========================================================================================
 * pccl.h -- C-ABI boundary of the B200-native link-chunk matching synthesizer.
 *
 * What the library computes: a collective-communication schedule for one or several
 * process groups on an arbitrary topology, by per-event link-chunk matching over the
 * time-expanded network (TEN).  The problem statement is the paper's:
 *   - topology with per-link latency alpha and bandwidth 1/beta ...... PAPER.md:334 (sec 4.6)
 *   - collective as NPU-centric pre/postcondition ...................... PAPER.md:76  (sec 2.1)
 *   - process group = the NPUs that take part; others only relay ...... PAPER.md:84  (sec 2.2),
 *                                                                        :298-300, :320, :422
 *   - result: which chunk crosses which link during which interval .... PAPER.md:149-156 (sec 3.5)
 * The matching procedure itself (steps R, A..F) is written out in DESIGN.md.
 *
 * Conventions
 *   - Every function that returns int returns PCCL_OK (0) or a negative pccl_error; on error
 *     every `out` pointer is left untouched.  No function throws or aborts.
 *   - "host" / "device" in a parameter comment says which address space the pointer is in.
 *     Input arrays are BORROWED for the duration of the call only.
 *   - Handles are opaque, owned by the library, released by the matching *_destroy
 *     (NULL is accepted and ignored).
 *   - All times are unsigned 64-bit integer picoseconds.  No floating point anywhere.
 *   - n_npus counts ALL nodes of the network: NPUs and switch nodes alike (PAPER.md:256,
 *     :348).  A switch is a node that is never listed in group_members.
 *   - Link id = index into the `links` array.  Parallel links are legal.
 *   - Several concurrent process groups go in ONE call: group_members is their union, chunk
 *     ids are globally unique.
 *   - Device work is enqueued on the stream set with pccl_set_stream (default: the legacy
 *     default stream) and is synchronised before a function returns host-visible results.
 *     The library binds to the CUDA device that is current at its first device call; a later
 *     call made with another device current returns PCCL_ERR_INVALID.
 *   - Calls on distinct handles may come from different threads: the entry points that touch the
 *     device serialise themselves (one runs at a time; they share a control mailbox, a copy
 *     stream and the stream below).  A single handle must not be used from two threads at once.
 *     The process-wide settings (stream, allocator) are set once, before any other thread calls.
 *   - There is NO CPU fallback: without a CUDA device every compute entry point returns
 *     PCCL_ERR_CUDA.
 * ========================================================================================= */
#ifndef PCCL_H_
#define PCCL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PCCL_VERSION 100 /* 0.1.0 */

typedef enum pccl_error {
    PCCL_OK = 0,
    PCCL_ERR_INVALID = -1,     /* null pointer; src/dst >= n_npus; self-loop; bytes_per_ps == 0;
                                  chunk_bytes == 0; duplicate or out-of-range group member; a
                                  pair whose NPU is not a group member; chunk id >= n_chunks; a
                                  chunk with no pre-holder or no post-holder; pre.n_chunks !=
                                  post.n_chunks */
    PCCL_ERR_UNSUPPORTED = -2, /* copy and reduction chunks mixed in one call (DESIGN.md step R);
                                  sizes beyond the limits listed in DESIGN.md */
    PCCL_ERR_UNREACHABLE = -3, /* some destination cannot be reached from its chunk's source */
    PCCL_ERR_CUDA = -4,        /* any CUDA runtime failure, including "no device" */
    PCCL_ERR_NOMEM = -5,       /* host or device allocation failed */
    PCCL_ERR_INTERNAL = -6,    /* a post-run invariant failed (never expected) */
    PCCL_ERR_TOO_LARGE = -7    /* pccl_candidate_totals_static: the problem needs more than PCCL_STATIC_SCRATCH_BYTES */
} pccl_error;

/* A directed physical link, cost alpha_ps + ceil(chunk_bytes / bytes_per_ps) picoseconds
 * (alpha-beta model; integer ceiling = DESIGN.md reading Q7). */
typedef struct pccl_link {
    uint32_t src, dst;
    uint64_t alpha_ps, bytes_per_ps;
} pccl_link_t;

/* "npu holds chunk" -- one element of an NPU-centric pre- or postcondition. */
typedef struct pccl_pair {
    uint32_t npu, chunk;
} pccl_pair_t;

typedef struct pccl_condition {
    uint32_t n_chunks;        /* chunk ids are 0 .. n_chunks-1 */
    uint64_t n_pairs;
    const pccl_pair_t* pairs; /* host; any order; duplicates are ignored */
} pccl_condition_t;

/* One transfer of the schedule: `chunk` occupies physical link `link` (src -> dst) during
 * [t_start_ps, t_end_ps).  32 bytes, no padding. */
typedef struct pccl_transfer {
    uint32_t chunk, src, dst, link;
    uint64_t t_start_ps, t_end_ps;
} pccl_transfer_t;

typedef struct pccl_topology pccl_topology_t;
typedef struct pccl_problem pccl_problem_t;
typedef struct pccl_schedule pccl_schedule_t;

/* ---------------------------------------------------------------------------------------
 * Process-wide plumbing (PyTorch supplies these through the Python binding).
 * ------------------------------------------------------------------------------------- */

/* cuda_stream: a cudaStream_t (NULL = legacy default stream).  All later device work of the
 * library is enqueued on it. */
void pccl_set_stream(void* cuda_stream);

/* Device allocator hooks.  alloc(bytes, cuda_stream, user) returns a device pointer aligned
 * to >= 256 bytes or NULL; release(ptr, user) gives it back.  Both NULL restores the
 * built-in stream-ordered allocator (cudaMallocAsync / cudaFreeAsync).  The library makes
 * O(1) allocations per call (one workspace, one result buffer). */
typedef void* (*pccl_alloc_fn)(size_t bytes, void* cuda_stream, void* user);
typedef void (*pccl_free_fn)(void* device_ptr, void* user);
void pccl_set_allocator(pccl_alloc_fn alloc, pccl_free_fn release, void* user);

const char* pccl_strerror(int err);
int pccl_version(void);

/* Process-wide tuning options (everything is an argument of the C-ABI: the library reads no environment variables
 * and no files).  value 0 restores the default.  Errors: INVALID (unknown option). */
typedef enum pccl_option {
    PCCL_OPT_BFS_WINDOW = 1,   /* PCCL_FLAG_BFS: conditions searched optimistically per round (default: one per SM) */
    PCCL_OPT_BFS_ROWS = 2,     /* PCCL_FLAG_BFS: initial capacity of a link's busy-run row, in runs (default: 256 or
                                  more; a full row reruns the phase with 4x longer rows) */
    PCCL_OPT_DYNAMIC_RECORDS = 3 /* PCCL_FLAG_DYNAMIC_RELAY: initial capacity of the record buffer (default: 1.25 x the
                                  static relay tree's transfer count; a short buffer reruns the phase with the exact
                                  count) */
} pccl_option;
int pccl_set_option(int option, uint64_t value);
uint64_t pccl_get_option(int option);

/* Number of CUDA kernels the library has launched in this process so far (every launch is counted where it is
 * issued).  The difference across a region is the library's own count of its GPU work there. */
uint64_t pccl_launch_count(void);

/* ---------------------------------------------------------------------------------------
 * Topology store (DESIGN.md row a0 and the link/in-link tables).
 * links: host array of n_links directed links.  Validates endpoints, builds the per-node
 * in-link and out-link tables in ascending link id on the host; the device copy is made on
 * first use.  Errors: INVALID, NOMEM.
 * ------------------------------------------------------------------------------------- */
int pccl_topology_create(uint32_t n_npus, const pccl_link_t* links, uint32_t n_links,
                         pccl_topology_t** out);
/* Switch model of PAPER.md:348 (section 4.7), per node; used by PCCL_FLAG_BFS (the other modes return UNSUPPORTED
 * while a model is set).  buffer_limit: host, n_npus u32, chunks the node may buffer at once (0xFFFFFFFF: no limit) --
 * a chunk is buffered at a node it is forwarded from, from its arrival until the end of the last transfer that forwards
 * it, and a visit of the node at time t is skipped while the conditions routed before hold that many chunks there at t
 * (Q23, Q24).  no_multicast: host, n_npus bytes, non-zero: the node forwards over its out-links one transfer
 * at a time, in ascending link id (Q25).  Either may be NULL; both NULL (or all unlimited / zero) removes the model.
 * With a model the conditions are routed strictly one after another (a one-condition window).
 * Errors: INVALID, NOMEM. */
int pccl_topology_set_switch_model(pccl_topology_t* topo, const uint32_t* buffer_limit, const uint8_t* no_multicast);
void pccl_topology_destroy(pccl_topology_t* topo);
uint32_t pccl_topology_n_npus(const pccl_topology_t* topo);
uint32_t pccl_topology_n_links(const pccl_topology_t* topo);

/* ---------------------------------------------------------------------------------------
 * pccl_synthesize -- the whole path with HOST buffers (the paper's problem statement,
 * PAPER.md:149-156): normalise (step R), upload, run steps A..F on the GPU, download.
 * group_members: host, n_members distinct node ids.  precondition / postcondition: which
 * group NPU holds which chunk before / after.  |pre(c)| = 1 for every chunk
 * means a copy collective (All-Gather, All-to-All(v), Broadcast ...); |pre(c)| > 1 with
 * |post(c)| = 1 a reduction (Reduce, Reduce-Scatter); |pre(c)| > 1 with |post(c)| > 1
 * All-Reduce = Reduce-Scatter then All-Gather.  seed keys the
 * deterministic tie-breaks (Philox4x32-10).  The schedule's transfers are in host memory
 * on return.  Errors: INVALID, UNSUPPORTED, UNREACHABLE, CUDA, NOMEM, INTERNAL.
 * ------------------------------------------------------------------------------------- */
int pccl_synthesize(const pccl_topology_t* topo, const uint32_t* group_members,
                    uint32_t n_members, const pccl_condition_t* precondition,
                    const pccl_condition_t* postcondition, uint64_t chunk_bytes, uint64_t seed,
                    pccl_schedule_t** out);

/* ---------------------------------------------------------------------------------------
 * Prepared problem: step R done once (host), conditions resident in HBM; then any number of
 * seeds can be synthesized with no host input traffic (best-of-K seed sweeps).
 * pccl_problem_create borrows topo for the lifetime of the problem (destroy the problem
 * first).  It validates and normalises on the host only; the device copy is made by the
 * first pccl_problem_synthesize (or pccl_problem_upload).
 * ------------------------------------------------------------------------------------- */
int pccl_problem_create(const pccl_topology_t* topo, const uint32_t* group_members,
                        uint32_t n_members, const pccl_condition_t* precondition,
                        const pccl_condition_t* postcondition, uint64_t chunk_bytes,
                        pccl_problem_t** out);
void pccl_problem_destroy(pccl_problem_t* problem);
int pccl_problem_upload(pccl_problem_t* problem); /* Errors: CUDA, NOMEM */

/* 0 copy, 1 reduce / reduce-scatter, 2 all-reduce (DESIGN.md step R) */
int pccl_problem_mode(const pccl_problem_t* problem);
uint32_t pccl_problem_n_chunks(const pccl_problem_t* problem);
/* Chunk-centric condition of `chunk` in `phase` (0: the only phase of a
 * copy or reduce problem, or the reduce phase of all-reduce; 1: the copy phase of
 * all-reduce).  *src = the source (copy) or root (reduce); returns the number of dests and
 * writes up to cap of them, ascending, to dests (host; may be NULL when cap == 0).
 * Returns a negative pccl_error for a bad chunk / phase. */
int64_t pccl_problem_condition(const pccl_problem_t* problem, uint32_t phase, uint32_t chunk,
                               uint32_t* src, uint32_t* dests, uint64_t cap);

/* flags for pccl_problem_synthesize.  None of them changes the result except DYNAMIC_RELAY (a different relay
 * rule); the others select how the same schedule is computed, for measurement and cross-checks. */
#define PCCL_FLAG_KEEP_ON_DEVICE 1u  /* do not download the transfers until they are asked for */
#define PCCL_FLAG_NO_IDLE_SKIP 2u    /* recount modes: rescan idle links every event */
#define PCCL_FLAG_TIME_LOOP 4u       /* record CUDA events around setup / event loop / emitter (stats) */
#define PCCL_FLAG_TRACE 8u           /* record per-event phase timestamps (pccl_schedule_trace) */
#define PCCL_FLAG_DENSE_SWEEP 16u    /* recount every free link's candidates at every event by sweeping whole
                                        bitmap rows: the plain memory-bound scan (two-barrier loop) */
#define PCCL_FLAG_RESCAN 32u         /* recount at every event, but only the 32-byte sectors whose summary bits
                                        are set in both rows (sector work list; two-barrier loop) */
#define PCCL_FLAG_DYNAMIC_RELAY 64u  /* relay rule of DESIGN.md Q18 instead of the static thin relay tree: a node
                                        takes a chunk iff it is strictly closer to some destination than the
                                        source and every node that claimed the chunk at an earlier event (fewer
                                        link-times, a few unused deliveries; kept counts with per-chunk holder
                                        lists unless DENSE_SWEEP or RESCAN is given) */
#define PCCL_FLAG_KEPT_COUNTS 128u   /* with DYNAMIC_RELAY: keep the candidate counts current (its default; the
                                        flag is accepted for compatibility) */
#define PCCL_FLAG_TWO_BARRIERS 256u  /* run the two-barrier event loop even where the one-barrier loop applies */
#define PCCL_FLAG_BFS 512u           /* the paper's own synthesizer instead of the matching loop (Alg. 1-3,
                                        :332-344 section 4.6; Q19-Q22): conditions in descending c.dist
                                        (ties: Philox(seed; chunk, tag 2), then chunk id), each routed by an
                                        earliest-arrival search over the whole network against the busy intervals of
                                        the conditions before it (lowest link id on equal arrivals), only the paths to
                                        its dests kept, their intervals then busy.  The other mode flags are ignored.
                                        Statistics: events = conditions routed, wants_total = transfers,
                                        rows_scanned = searches run (a condition is searched again when a condition
                                        ahead of it took an interval it used), links_scanned = link relaxations,
                                        slow_picks = commit rounds.  UNSUPPORTED if a time does not fit in
                                        64 - ceil(log2(n_links)) bits or n_npus > 8,500. */

#define PCCL_FLAG_BARRIER_LOOP 1024u  /* run the barrier loops (one grid barrier per event where that loop applies, else
                                        two) even where the barrier-free loop applies */
#define PCCL_FLAG_ASYNC 2048u        /* run the barrier-free loop (one warp per destination, pairwise synchronisation
                                        through per-node claim logs) even when the link costs differ
                                        by more than 16x -- its lookahead is the cheapest in-link of a node, so idle
                                        regions then advance in small time steps.  It is the default for the static
                                        relay tree when every node has at most 8 in-links, at most 16 x SM-count nodes,
                                        and link costs within 16x of each other */

#define PCCL_FLAG_LSU_SWEEP 4096u    /* the streaming candidate sweep (row a5: seeds the kept counts of the barrier loops;
                                        pccl_device_candidate_sweep) loads its rows with per-lane 128-bit loads instead of
                                        staging them in shared memory by bulk asynchronous copies (TMA) */

#define PCCL_FLAG_PIPELINE 8192u     /* with PCCL_FLAG_BFS, on an All-Reduce problem: the copy phase of a chunk starts as soon
                                        as its root holds the complete sum (the end of the last transfer of the chunk into
                                        the root) instead of after the whole reduce phase; it is routed against the link
                                        intervals the reduce phase took (Q26; PAPER.md:330 composes the phases).
                                        Other collectives: no effect.  UNSUPPORTED without PCCL_FLAG_BFS or with a switch
                                        model.  time_phase1_ps = end of the reduce phase, schedule time = the later end */

#define PCCL_FLAG_DIST_PICK 16384u   /* pick policy of the matching loop (Q27; Alg. 3's order, as a
                                        priority): a link takes one of its candidates with the LARGEST c.dist = max over dests
                                        of the alpha-beta shortest path from the chunk's source, ties by the seeded draw (the
                                        k-th tied candidate in ascending chunk id).  Runs in the barrier-free loop on chunks
                                        relabelled in (c.dist, id) order; UNSUPPORTED where that loop does not apply (a node
                                        with more than 8 in-links) and with the other mode flags */

/* Steps A..F on the GPU for one seed.  Errors: UNREACHABLE, CUDA, NOMEM, INTERNAL. */
int pccl_problem_synthesize(pccl_problem_t* problem, uint64_t seed, uint32_t flags,
                            pccl_schedule_t** out);

/* ---------------------------------------------------------------------------------------
 * Schedule.  Transfers are in canonical order: ascending (t_start_ps, link).
 * ------------------------------------------------------------------------------------- */
uint64_t pccl_schedule_time(const pccl_schedule_t* s); /* max t_end_ps; 0 if empty */
uint64_t pccl_schedule_size(const pccl_schedule_t* s); /* number of transfers */
/* host pointer, valid until the schedule is destroyed; downloads on first use when the
 * schedule was kept on the device; NULL if empty or on a CUDA failure */
const pccl_transfer_t* pccl_schedule_transfers(pccl_schedule_t* s);
/* device pointer to the same records (NULL once released or if empty) */
const pccl_transfer_t* pccl_schedule_transfers_device(const pccl_schedule_t* s);
void pccl_schedule_destroy(pccl_schedule_t* s);

/* Translation (section 4.8): the schedule as one program per node.  Every transfer gives
 * two operations: kind 0 = its destination RECEIVES `chunk` from `peer` over `link`, complete at time_ps =
 * t_end; kind 1 = its source SENDS `chunk` to `peer` over `link`, starting at time_ps = t_start.  A node's
 * program lists its operations by (time_ps, kind, link) -- a receive precedes a send at the same instant
 * (store-and-forward).  offsets: host, n_npus + 1 entries; the program of node v is
 * ops[offsets[v] .. offsets[v+1]).  ops: host, 2 * pccl_schedule_size(s) entries.  Built on the GPU (two
 * stable radix sorts) from the device copy of the transfers.  Errors: INVALID, UNSUPPORTED, CUDA, NOMEM. */
typedef struct pccl_op {
    uint32_t kind, peer, chunk, link;
    uint64_t time_ps;
} pccl_op_t;
int pccl_schedule_programs(pccl_schedule_t* s, uint64_t* offsets, pccl_op_t* ops);

/* Counters of the run that produced the schedule. */
typedef struct pccl_stats {
    uint64_t events;         /* event times processed (both phases of an all-reduce summed) */
    uint64_t wants_total;    /* popcount(wants) after step C == number of transfers */
    uint64_t rows_scanned;   /* bitmap rows the match kernel swept (have + wants rows): the dense,
                                algorithmic count -- rows_scanned * row_bytes = bytes a sweep without the
                                sector summaries would request */
    uint64_t bytes_requested;/* bytes the match kernel actually requested: bitmap sectors whose summary
                                bits were set in both rows, the summary rows, the segments re-read by picks */
    uint64_t row_bytes;      /* bytes of one (padded) bitmap row */
    uint64_t links_scanned;  /* active in-links whose candidates were counted */
    uint64_t slow_picks;     /* picks that took the serial re-pick path */
    uint64_t time_phase1_ps; /* all-reduce: time of the reduce phase */
    float loop_ms;           /* event-loop kernel time (PCCL_FLAG_TIME_LOOP), else 0 */
    float setup_ms;          /* steps A..D kernels (PCCL_FLAG_TIME_LOOP), else 0 */
    float emit_ms;           /* emitter kernels (PCCL_FLAG_TIME_LOOP), else 0 */
    uint32_t mode;           /* 0 copy, 1 reduce, 2 all-reduce */
    uint32_t grid_blocks;    /* CTAs of the persistent event-loop kernel */
} pccl_stats_t;
int pccl_schedule_stats(const pccl_schedule_t* s, pccl_stats_t* out);

/* Diagnostic trace (PCCL_FLAG_TRACE): for each event time of the last phase, PCCL_TRACE_SLOTS
 * %globaltimer stamps (ns) taken by CTA 0 of the event-loop kernel: loop top, end of the
 * links phase (emit + arrivals), end of grid barrier 1, in-link list built, candidates
 * counted, picks made, destination done, end of grid barrier 2.  Returns the number of u64
 * values available (events * PCCL_TRACE_SLOTS) and writes up to cap of them to out (host). */
#define PCCL_TRACE_SLOTS 12
int64_t pccl_schedule_trace(const pccl_schedule_t* s, uint64_t* out, uint64_t cap);

/* ---------------------------------------------------------------------------------------
 * Single rows of the path, exposed for parity tests against the oracle.  Each runs the
 * same device code the full path uses.
 * ------------------------------------------------------------------------------------- */
/* a6: Philox4x32-10 evaluated on the GPU for n counters.  ctr: host n*4 u32, key: host 2
 * u32, out: host n*4 u32. */
int pccl_device_philox(const uint32_t* ctr, uint64_t n, const uint32_t key[2], uint32_t* out);
/* a0: link costs, out: host n_links u64. */
int pccl_device_link_costs(pccl_topology_t* topo, uint64_t chunk_bytes, uint64_t* out);
/* a1: alpha-beta shortest distances from src (transposed != 0: on the reversed links),
 * out: host n_npus u64, UINT64_MAX = unreachable. */
int pccl_device_distances(pccl_topology_t* topo, uint64_t chunk_bytes, uint32_t src,
                          int transposed, uint64_t* out);
/* a2: wants relation of `phase` after step C for `seed`, as (node, chunk) pairs sorted by
 * (node, chunk).  Returns the pair count (may exceed cap; only cap are written) or a
 * negative pccl_error.  out: host. */
int64_t pccl_device_wants(pccl_problem_t* problem, uint32_t phase, uint64_t seed,
                          pccl_pair_t* out, uint64_t cap);

/* a5: the candidate bitmap of every link, cand(l) = have[src_l] & wants[dst_l], at t = 0 (after steps A..C for `seed`),
 * by the streaming sweep kernel alone: (N + L) bitmap rows per sweep, rows staged in shared memory by bulk asynchronous
 * copies (PCCL_FLAG_LSU_SWEEP: per-lane 128-bit loads).  Runs `iters` sweeps between two CUDA events.
 * ms_per_sweep, bytes_per_sweep (algorithmic bytes of one sweep: rows x padded row bytes) and totals (host, n_links u32:
 * |cand(l)|) may each be NULL.  Errors: INVALID, UNREACHABLE, CUDA, NOMEM. */
int pccl_device_candidate_sweep(pccl_problem_t* problem, uint32_t phase, uint64_t seed, uint32_t flags, uint32_t iters,
                                float* ms_per_sweep, uint64_t* bytes_per_sweep, uint32_t* totals);
/* Measurement aid: reads a device buffer of `bytes` bytes sequentially with the sweeps' access pattern (128-bit
 * ld.global.cg, grid-stride) `iters` times and reports the milliseconds per pass: the measured ceiling of L2 when the
 * buffer fits there, of HBM when it does not.  Errors: INVALID, CUDA, NOMEM. */
int pccl_device_read_bandwidth(uint64_t bytes, uint32_t iters, float* ms_per_pass);

/* ---------------------------------------------------------------------------------------
 * The entry point that allocates nothing.
 *
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): row a5 -- |cand(l)| = popcount(have[src_l] & wants[dst_l]) of every link (one chunk per link and
 * step; north star: per-link candidate bitmap) -- on bitmaps the CALLER holds on the device, by the same streaming
 * sweep kernel as pccl_device_candidate_sweep.  The kernel's scratch (per-link, per-4096-chunk segment counts and the
 * whole-row sums it keeps beside them) lives in a fixed array of PCCL_STATIC_SCRATCH_BYTES inside the library's device
 * image: every GPU that loads the library holds it until the process exits.  The call makes no cudaMalloc / cudaFree /
 * cudaMallocAsync / cudaHostAlloc and calls no allocating library routine; it enqueues one memset, two kernels.
 *
 *   have, wants     device, n_npus rows of words_per_row u64 each (bit c of row v = chunk c at / wanted by node v);
 *                   16-byte aligned, words_per_row even and > 0 (rows are copied in 16-byte units)
 *   link_src        device, n_links u32: source node of link l
 *   in_off, in_link device, CSR by destination: the in-links of node v are in_link[in_off[v] .. in_off[v+1]),
 *                   n_npus + 1 and n_links u32; every link appears once
 *   totals          device, n_links u32, written: |cand(l)|
 *   stream          a cudaStream_t (NULL = the default stream); the work is enqueued there, the call does not wait
 *
 * Limit: n_links * (ceil(words_per_row / 64) + 1) * 4 bytes <= PCCL_STATIC_SCRATCH_BYTES, else PCCL_ERR_TOO_LARGE
 * (nothing is enqueued).  Other errors: INVALID (null / misaligned pointer, odd or zero words_per_row), CUDA.
 * n_npus == 0 or n_links == 0: PCCL_OK, nothing enqueued.
 *
 * Every call on a device shares the one array, which keeps the previous call's contents: the part a call uses is
 * cleared on `stream` first.  Two calls whose work overlaps on the GPU (different streams, or threads) RACE on it --
 * order them.  The first call on each device looks the array's device address up (cudaGetSymbolAddress) and sets the
 * kernel's shared-memory attribute: make it outside stream capture.  The caller owns all buffers. */
#define PCCL_STATIC_SCRATCH_BYTES (4u << 20)
int pccl_candidate_totals_static(const uint64_t* have, const uint64_t* wants, uint32_t n_npus, uint32_t n_links,
                                 uint32_t words_per_row, const uint32_t* link_src, const uint32_t* in_off,
                                 const uint32_t* in_link, uint32_t* totals, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* PCCL_H_ */
