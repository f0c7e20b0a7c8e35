// =========================================================================================
// pccl_loop2.cuh -- the event loop WITHOUT a grid barrier (default for the static thin relay tree).
//
// k_loop / k_loop1 advance all destinations in lockstep: one (two) grid barriers per event time and a global
// atomicMin for the next time.  Here every destination is its own process -- ONE WARP per destination, no block
// or grid barrier at all -- and the processes synchronise pairwise, as a conservative parallel discrete-event
// simulation with the link cost as lookahead:
//
//   * a destination v acts only at its own event times (an in-link of v becomes free, or a chunk
//     arrives at one of its sources).  At any other global event time the oracle's sweep finds
//     nothing for v (candidates only appear at arrivals, links only free at their free times), so the schedule
//     is the same, bit for bit;
//   * v publishes every claim it makes -- (t_start, entry, in-link) -- in an append-only per-node LOG
//     (write-once 16-byte entries, self-validating against the 0xFF fill), and a 16-byte HEADER
//     (LVT_v, count): "all my claims that start before LVT_v are log entries [0, count)".  Both are written and
//     read with single 128-bit relaxed gpu-scope accesses (atomic), so no fence is needed anywhere: a reader
//     that sees a header waits until it holds valid copies of the entries the header counts;
//   * v may act at time t once every source u has LVT_u + wmin_u > t (wmin_u = cheapest in-link of u: a claim
//     u has not published yet cannot arrive at u before that).  It then consumes u's log entries with
//     t_start + wmin_u <= t (at most one per in-link of u stays pending), applies the arrivals with t_end = t,
//     matches, and publishes its next event time (a lower bound of it) as LVT_v.  The node with the smallest
//     time can always proceed, so there is no deadlock; a node whose wants are exhausted publishes LVT = inf
//     and leaves.
//
// State.  The wants row of v is static here (k_wants' output, never modified).  Its set bits, in ascending chunk
// id, are v's ENTRIES 0 .. W_v-1.  Per in-link j the warp keeps, in shared memory, a candidate bitmap over the
// entries (bit e: entry e still wanted AND source of j holds its chunk), counts per group of 1024 entries and
// the total n_j: a5's  have[src] & wants[dst]  kept incrementally, the pick (a6) is the k-th set bit by
// popcount / __fns, a claim (a7, a8) clears the entry's bit in every in-link's bitmap.  An arrival of source
// u's entry e_u is translated by one load from a precomputed table  xmap[link][e_u] -> entry of v (or none).
// Nothing in the loop touches the NPU x chunk bitmaps; per event a destination reads <= 8 headers and the few
// new log entries of its sources (one L2 round trip), the table words of the arrivals (a second one), and
// stores its own claims and header.
//
// The records are ranked after the fact (k_win_*), in windows of start times behind the global virtual time -- on a
// second stream while the loop runs when the host is streaming them out, else in one window after it: start times
// are hashed into a small table, the distinct ones ranked, and a per-event link bitmap gives the position
// base(event) + rank(link)  -- the same canonical (t_start, link) order the barrier loops emit.
// =========================================================================================
#pragma once
#include "pccl_device.cuh"

namespace pccl {

struct __align__(16) U128 { unsigned long long lo, hi; };

__device__ __forceinline__ U128 ld128(const U128* p) {
    U128 r;
    asm volatile("{\n .reg .b128 t;\n ld.relaxed.gpu.global.b128 t, [%2];\n mov.b128 {%0, %1}, t;\n}"
                 : "=l"(r.lo), "=l"(r.hi) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st128(U128* p, unsigned long long lo, unsigned long long hi) {
    asm volatile("{\n .reg .b128 t;\n mov.b128 t, {%1, %2};\n st.relaxed.gpu.global.b128 [%0], t;\n}"
                 :: "l"(p), "l"(lo), "l"(hi) : "memory");
}

// two predicated 128-bit loads issued back to back (a lane's two poll items); an item that is not loaded reads as all ones
__device__ __forceinline__ void ld128x2(const U128* p0, bool on0, const U128* p1, bool on1, U128& r0, U128& r1) {
    asm volatile("{\n .reg .b128 t0, t1;\n .reg .pred q0, q1;\n"
                 " setp.ne.u32 q0, %6, 0;\n setp.ne.u32 q1, %7, 0;\n"
                 " mov.b128 t0, {%8, %8};\n mov.b128 t1, {%8, %8};\n"
                 " @q0 ld.relaxed.gpu.global.b128 t0, [%4];\n"
                 " @q1 ld.relaxed.gpu.global.b128 t1, [%5];\n"
                 " mov.b128 {%0, %1}, t0;\n mov.b128 {%2, %3}, t1;\n}"
                 : "=l"(r0.lo), "=l"(r0.hi), "=l"(r1.lo), "=l"(r1.hi)
                 : "l"(p0), "l"(p1), "r"((uint32_t)on0), "r"((uint32_t)on1), "l"(0xFFFFFFFFFFFFFFFFull)
                 : "memory");
}

constexpr int A2_MAX_IN = 8;         // in-links per node (one quad of lanes each)
#ifndef A2_HDR_STRIDE
#define A2_HDR_STRIDE 8              // U128 units between two nodes' headers: one header per 128-byte line
#endif
#define A2_HDR(a, v) ((a).hdr + (size_t)(v) * A2_HDR_STRIDE)
#ifndef A2_LOG_STRIDE
#define A2_LOG_STRIDE 1              // U128 units between two log entries (a sector or a line per entry was tried: no gain)
#endif
#define A2_LOG(a, i) ((a).log + (size_t)(i) * A2_LOG_STRIDE)
constexpr int A2_MAX_WARPS = 16;     // destinations per CTA

struct A2Ctrl {                      // read back once by the host after the plan kernel / after the loop
    unsigned long long xmap_total;   // entries of the translation tables
    unsigned long long priv_total;   // u32 words of all private images
    unsigned long long smem_need;    // dynamic shared memory of the largest CTA, bytes
    unsigned long long w_min, w_max; // link costs (lookahead quality)
    unsigned long long actions, polls, picks, slow, bytes;   // loop statistics
    // emit
    unsigned long long total, tmax;
    uint32_t n_start, n_end;         // distinct start times / end times
    uint32_t err;                    // 1 table or bitmap capacity exceeded (the host falls back to the radix sort)
    uint32_t pad;
    unsigned long long prof[8];      // -DPCCL_A2_PROFILE: SM cycles per phase, summed over the warps
};

// state of the windowed emitter (device memory, cleared before the first window)
struct A2Win {
    unsigned long long gvt;           // this window takes the claims that start before gvt
    unsigned long long emitted;       // records written by the earlier windows
    unsigned long long emitted_next;  //   ... and by this one
    uint32_t used0, pad;              // this window's distinct start times are used[used0 .. n_start)
};

// per-destination fixed part of the warp's shared memory
struct A2Fixed {
    uint32_t nin, nsrc, W, Wd, G, pad0[3];
    uint32_t link[A2_MAX_IN];
    uint32_t sidx[A2_MAX_IN];                 // in-link -> index of its source among the distinct sources
    unsigned long long w[A2_MAX_IN];
    uint32_t s_node[A2_MAX_IN], s_W[A2_MAX_IN], s_mask[A2_MAX_IN], s_pad[A2_MAX_IN];
    unsigned long long s_wmin[A2_MAX_IN], s_logbase[A2_MAX_IN], s_xbase[A2_MAX_IN];
    unsigned long long hop_w[A2_MAX_IN * 8];  // [s * 8 + i]: cost of in-link i of source s
    uint32_t cur[A2_MAX_IN];                  // next log entry of source s to consume
    uint32_t pend_e[A2_MAX_IN * 8];           // in flight towards source s over its in-link i: entry of v (NONE32: not wanted)
    unsigned long long pend_te[A2_MAX_IN * 8];//   ... and its arrival time (T_INF: nothing pending)
    unsigned long long free_te[A2_MAX_IN];
    uint32_t n[A2_MAX_IN];                    // candidates of in-link j
    uint32_t pad1[A2_MAX_IN];
};
static_assert(sizeof(A2Fixed) % 16 == 0, "alignment of the arrays that follow");

// ncls > 0 (PCCL_FLAG_DIST_PICK): the image ends with the destination's class boundaries in entry space,
// [nb][bnd[0 .. ncls]]: bnd[i] = first entry of the i-th c.dist class present among the entries, bnd[nb] = W
__host__ __device__ __forceinline__ uint32_t a2_priv_words(uint32_t W, uint32_t nin, uint32_t ncls) {
    const uint32_t Wd = (W + 31) >> 5, G = (Wd + 31) >> 5;
    return Wd * (1 + nin) + nin * G + (ncls ? ncls + 2 : 0);   // live[Wd], cb[nin][Wd], grp[nin][G], boundaries
}
__host__ __device__ __forceinline__ uint32_t a2_warp_bytes(uint32_t W, uint32_t nin, uint32_t ncls) {
    return (uint32_t)sizeof(A2Fixed) + ((a2_priv_words(W, nin, ncls) * 4u + 15u) & ~15u);
}

struct A2Args {
    uint32_t N, L, Wp, nLw;
    uint32_t k0, k1;
    uint32_t grid, wpc;               // CTAs and warps per CTA of k_loop2 (destination v = cta + warp * grid)
    uint32_t ncls;                    // c.dist classes of the relabelled chunks (PCCL_FLAG_DIST_PICK), 0: uniform pick
    const uint32_t* cls;              // [C] class of each (relabelled) chunk
    const uint32_t* orig;             // [C] the caller's chunk id of each relabelled chunk, or null
    const uint32_t *esrc, *edst, *psrc, *pdst, *in_off, *in_link;
    const uint64_t* w;
    const uint64_t* wants;            // [N][Wp], static
    const uint32_t* wants_cnt;        // [N] = W_v
    const uint32_t* csrc;             // [C] source of each chunk
    unsigned long long* nbase;        // [N+1] first entry of node v in ids / log
    unsigned long long* poff;         // [N+1] first word of node v's private image
    unsigned long long* loff;         // [L+1] first word of link l's translation table
    uint32_t* soff;                   // [N] byte offset of node v's warp in its CTA's shared memory
    uint32_t* ids;                    // [M] chunk of each entry
    uint32_t* rowpre;                 // [N][Wp] entries of the row before each word
    uint32_t* xmap;                   // [xmap_total]
    uint32_t* priv;                   // [priv_total]
    U128* log;                        // [M]
    U128* hdr;                        // [N]
    A2Ctrl* ctrl;
    uint32_t* abort_flag;             // LoopCtrl::err of the phase: non-zero -> every warp leaves
    // emit
    unsigned long long* tkey;         // [tcap] hashed times (T_INF: empty)
    uint32_t *tcnt, *tflag, *trank;   // [tcap] records starting at the time; bit 0 is an end time, bit 1 is a start time; rank
    uint32_t* used;                   // [ecap] slots of the distinct start times
    uint32_t* cnt_sorted;             // [ecap] records per start time, in time order
    unsigned long long* ebase;        // [ecap] first record of each start time
    uint32_t* eslot;                  // [M] slot of each entry's start time
    unsigned long long* bm;           // [ecap][nLw] links matched at each start time
    uint32_t* wbase;                  // [ecap][nLw] matched links before each word
    uint32_t tcap, ecap;
    Rec* out;
    uint64_t out_cap, t_offset;
    // windows of the emitter
    A2Win* win;
    uint32_t *wcur, *wnext;           // [N] log entries of node v below wcur are emitted; the window ends at wnext
    unsigned long long* progress;     // mapped host word: records that are final (null: nobody is streaming them out)
};

// ---------------------------------------------------------------------------------------------------------------
// plan (one block): entry bases, private-image offsets, translation-table offsets, shared-memory layout
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long block_excl_scan_1024(unsigned long long x, unsigned long long* total, unsigned long long* sm) {
    // exclusive scan over the 1024 threads of the block; sm: 33 words of shared memory
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long y = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if ((int)lane >= o) incl += y;
    }
    __syncthreads();
    if (lane == 31) sm[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        const unsigned long long y = sm[lane];
        unsigned long long yi = y;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long z = __shfl_up_sync(0xFFFFFFFFu, yi, o);
            if ((int)lane >= o) yi += z;
        }
        sm[lane] = yi - y;
        if (lane == 31) sm[32] = yi;
    }
    __syncthreads();
    *total = sm[32];
    return sm[warp] + incl - x;
}

__global__ void __launch_bounds__(1024) k_a2_plan(A2Args a) {
    __shared__ unsigned long long sm[33];
    __shared__ unsigned long long s_max, s_wmin, s_wmax;
    const uint32_t tid = threadIdx.x;
    if (tid == 0) { s_max = 0; s_wmin = T_INF; s_wmax = 0; }
    unsigned long long carry = 0, tot;
    for (uint32_t b = 0; b < a.N; b += 1024) {                       // nbase
        const uint32_t v = b + tid;
        const unsigned long long x = v < a.N ? a.wants_cnt[v] : 0ull;
        const unsigned long long ex = block_excl_scan_1024(x, &tot, sm);
        if (v < a.N) a.nbase[v] = carry + ex;
        carry += tot;
    }
    if (tid == 0) a.nbase[a.N] = carry;
    carry = 0;
    for (uint32_t b = 0; b < a.N; b += 1024) {                       // poff
        const uint32_t v = b + tid;
        const unsigned long long x = v < a.N ? a2_priv_words(a.wants_cnt[v], a.in_off[v + 1] - a.in_off[v], a.ncls) : 0ull;
        const unsigned long long ex = block_excl_scan_1024(x, &tot, sm);
        if (v < a.N) a.poff[v] = carry + ex;
        carry += tot;
    }
    if (tid == 0) { a.poff[a.N] = carry; a.ctrl->priv_total = carry; }
    carry = 0;
    unsigned long long wmn = T_INF, wmx = 0;
    for (uint32_t b = 0; b < a.L; b += 1024) {                       // loff
        const uint32_t l = b + tid;
        const unsigned long long x = l < a.L ? a.wants_cnt[a.esrc[l]] : 0ull;
        if (l < a.L) { wmn = min(wmn, (unsigned long long)a.w[l]); wmx = max(wmx, (unsigned long long)a.w[l]); }
        const unsigned long long ex = block_excl_scan_1024(x, &tot, sm);
        if (l < a.L) a.loff[l] = carry + ex;
        carry += tot;
    }
    if (tid == 0) { a.loff[a.L] = carry; a.ctrl->xmap_total = carry; }
    atomicMin(&s_wmin, wmn);
    atomicMax(&s_wmax, wmx);
    unsigned long long mx = 0;
    for (uint32_t cta = tid; cta < a.grid; cta += 1024) {            // shared-memory layout of each CTA
        uint32_t off = 0;
        for (uint32_t wi = 0; wi < a.wpc; ++wi) {
            const uint32_t v = cta + wi * a.grid;
            if (v >= a.N) break;
            a.soff[v] = off;
            off += a2_warp_bytes(a.wants_cnt[v], a.in_off[v + 1] - a.in_off[v], a.ncls);
        }
        mx = max(mx, (unsigned long long)off);
    }
    atomicMax(&s_max, mx);
    __syncthreads();
    if (tid == 0) { a.ctrl->smem_need = s_max; a.ctrl->w_min = s_wmin; a.ctrl->w_max = s_wmax; }
}

// ---------------------------------------------------------------------------------------------------------------
// entries: ids[nbase[v] + e] = chunk of v's entry e (ascending), rowpre[v][word] = entries before the word.
// One 256-thread block per node: every warp takes a contiguous slice of the row.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_a2_entries(A2Args a) {
    const uint32_t v = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __shared__ uint32_t wsum[8];
    const uint64_t* row = a.wants + (size_t)v * a.Wp;
    const uint32_t per = ((a.Wp + 8 * 32 - 1) / (8 * 32)) * 32;       // words per warp, a multiple of 32
    const uint32_t w0 = warp * per, w1 = min(a.Wp, w0 + per);
    uint32_t s = 0;
    for (uint32_t wi = w0 + lane; wi < w1; wi += 32) s += __popcll(row[wi]);
    s = __reduce_add_sync(0xFFFFFFFFu, s);
    if (lane == 0) wsum[warp] = s;
    __syncthreads();
    uint32_t pos = 0;
    for (uint32_t k = 0; k < warp; ++k) pos += wsum[k];
    uint32_t* ids = a.ids + a.nbase[v];
    uint32_t* pre = a.rowpre + (size_t)v * a.Wp;
    for (uint32_t wb = w0; wb < w1; wb += 32) {
        const uint32_t wi = wb + lane;
        const uint64_t word = wi < w1 ? row[wi] : 0ull;
        const uint32_t pc = __popcll(word);
        const uint32_t incl = warp_incl_scan(pc, lane);
        uint32_t my = pos + incl - pc;
        if (wi < w1) pre[wi] = my;
        uint64_t x = word;
        while (x) {
            const int b = __ffsll((long long)x) - 1;
            x &= x - 1;
            ids[my++] = wi * 64 + b;
        }
        pos += __shfl_sync(0xFFFFFFFFu, incl, 31);
    }
}

// translation tables: xmap[loff[l] + e] = entry of edst[l] that holds the chunk of esrc[l]'s entry e (NONE32: not wanted)
__global__ void __launch_bounds__(128) k_a2_xmap(A2Args a) {
    const uint32_t l = blockIdx.x;
    const uint32_t u = a.esrc[l], x = a.edst[l];
    const uint32_t W = a.wants_cnt[u];
    const uint32_t* ids = a.ids + a.nbase[u];
    uint32_t* xm = a.xmap + a.loff[l];
    const uint64_t* row = a.wants + (size_t)x * a.Wp;
    const uint32_t* pre = a.rowpre + (size_t)x * a.Wp;
    for (uint32_t e = threadIdx.x; e < W; e += blockDim.x) {
        const uint32_t c = ids[e];
        const uint64_t word = row[c >> 6];
        uint32_t r = NONE32;
        if ((word >> (c & 63)) & 1ull) r = pre[c >> 6] + __popcll(word & ((1ull << (c & 63)) - 1ull));
        xm[e] = r;
    }
}

// private image of node v: live bits, candidate bits of every in-link at t = 0 (the source of the in-link is the
// chunk's source), group counts; header and (by the host's memset) log start empty
__global__ void __launch_bounds__(128) k_a2_priv(A2Args a) {
    const uint32_t v = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const uint32_t W = a.wants_cnt[v];
    const uint32_t e0 = a.in_off[v], nin = a.in_off[v + 1] - e0;
    if (threadIdx.x == 0) st128(A2_HDR(a, v), W ? 0ull : T_INF, 0ull);
    if (W == 0) return;
    const uint32_t Wd = (W + 31) >> 5, G = (Wd + 31) >> 5;
    uint32_t* live = a.priv + a.poff[v];
    uint32_t* cb = live + Wd;
    uint32_t* grp = cb + (size_t)nin * Wd;
    const uint32_t* ids = a.ids + a.nbase[v];
    __shared__ uint32_t s_src[A2_MAX_IN];
    if (threadIdx.x < nin && threadIdx.x < A2_MAX_IN) s_src[threadIdx.x] = a.esrc[a.in_link[e0 + threadIdx.x]];
    __syncthreads();
    for (uint32_t wd = warp; wd < Wd; wd += nw) {
        const uint32_t e = wd * 32 + lane;
        const bool valid = e < W;
        const uint32_t s = valid ? a.csrc[ids[e]] : NONE32;
        const uint32_t lv = __ballot_sync(0xFFFFFFFFu, valid);
        if (lane == 0) live[wd] = lv;
        for (uint32_t j = 0; j < nin && j < A2_MAX_IN; ++j) {
            const uint32_t b = __ballot_sync(0xFFFFFFFFu, valid && s == s_src[j]);
            if (lane == 0) cb[(size_t)j * Wd + wd] = b;
        }
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < nin * G; i += blockDim.x) {
        const uint32_t j = i / G, g = i - j * G;
        uint32_t s = 0;
        for (uint32_t wd = g * 32; wd < min(Wd, g * 32 + 32); ++wd) s += __popc(cb[(size_t)j * Wd + wd]);
        grp[i] = s;
    }
    if (a.ncls) {
        // entries ascend in (relabelled) chunk id, so their classes ascend too: the boundaries are the entries whose
        // class differs from the entry before; bnd[i] is written at the rank of its class among the present ones
        uint32_t* pb = grp + (size_t)nin * G;       // [nb][bnd ...]
        __shared__ uint32_t s_nb;
        if (threadIdx.x == 0) s_nb = 0;
        __syncthreads();
        for (uint32_t e = threadIdx.x; e < W; e += blockDim.x)
            if (e == 0 || a.cls[ids[e]] != a.cls[ids[e - 1]]) pb[1 + atomicAdd(&s_nb, 1u)] = e;
        __syncthreads();
        if (threadIdx.x == 0) {                     // few boundaries: insertion sort, then the sentinel
            const uint32_t nb = s_nb;
            uint32_t* B = pb + 1;
            for (uint32_t i = 1; i < nb; ++i) {
                const uint32_t x = B[i];
                uint32_t k = i;
                while (k > 0 && B[k - 1] > x) { B[k] = B[k - 1]; --k; }
                B[k] = x;
            }
            pb[0] = nb;
            B[nb] = W;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// the loop
// ---------------------------------------------------------------------------------------------------------------
// position of the k-th (0-based) set bit of w, k < popc(w)
__device__ __forceinline__ uint32_t a2_kth_bit32(uint32_t w, uint32_t k) {
    uint32_t pos = 0, c;
    c = __popc(w & 0xFFFFu); if (k >= c) { k -= c; pos += 16; w >>= 16; }
    c = __popc(w & 0xFFu);   if (k >= c) { k -= c; pos += 8;  w >>= 8; }
    c = __popc(w & 0xFu);    if (k >= c) { k -= c; pos += 4;  w >>= 4; }
    c = __popc(w & 0x3u);    if (k >= c) { k -= c; pos += 2;  w >>= 2; }
    if (k >= (w & 1u)) pos += 1;
    return pos;
}

// k-th (0-based) set bit of in-link row cbj (counts per 1024-entry group in grpj) by the four lanes q = 0..3 of a
// quad; `on` is quad-uniform.  Returns the entry index in every lane of the quad.
__device__ __forceinline__ uint32_t a2_quad_select(const uint32_t* cbj, const uint32_t* grpj, uint32_t Wd, uint32_t G,
                                                   uint32_t k, bool on, uint32_t q, uint32_t lane) {
    const uint32_t qbase = lane & ~3u;
    uint32_t g_sel = 0;
    if (G > 1 && G <= 4) {                                          // warp-uniform; every lane scans the few group counts itself
        uint32_t c[4];
#pragma unroll
        for (int g = 0; g < 4; ++g) c[g] = (on && (uint32_t)g < G) ? grpj[g] : 0u;
#pragma unroll
        for (int g = 0; g < 3; ++g)
            if (g_sel == (uint32_t)g && k >= c[g]) { k -= c[g]; g_sel = g + 1; }
    } else if (G > 4) {
        const uint32_t per = (G + 3) >> 2, g0 = q * per, g1 = min(G, g0 + per);
        uint32_t sum = 0;
        if (on) for (uint32_t g = g0; g < g1; ++g) sum += grpj[g];
        uint32_t incl = sum, y;
        y = __shfl_up_sync(0xFFFFFFFFu, incl, 1, 4); if (q >= 1) incl += y;
        y = __shfl_up_sync(0xFFFFFFFFu, incl, 2, 4); if (q >= 2) incl += y;
        const uint32_t excl = incl - sum;
        const bool mine = on && k >= excl && k < incl;
        uint32_t gs = 0, kr = 0;
        if (mine) {
            kr = k - excl;
            for (uint32_t g = g0; g < g1; ++g) {
                const uint32_t c = grpj[g];
                if (kr < c) { gs = g; break; }
                kr -= c;
            }
        }
        const uint32_t bal = (__ballot_sync(0xFFFFFFFFu, mine) >> qbase) & 0xFu;
        const uint32_t own = bal ? (uint32_t)(__ffs(bal) - 1) : 0u;
        g_sel = __shfl_sync(0xFFFFFFFFu, gs, qbase + own);
        k = __shfl_sync(0xFFFFFFFFu, kr, qbase + own);
    }
    const uint32_t w0 = g_sel * 32 + q * 8;
    uint32_t wv[8];
    uint32_t sum = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        wv[i] = (on && w0 + i < Wd) ? cbj[w0 + i] : 0u;
        sum += __popc(wv[i]);
    }
    uint32_t incl = sum, y;
    y = __shfl_up_sync(0xFFFFFFFFu, incl, 1, 4); if (q >= 1) incl += y;
    y = __shfl_up_sync(0xFFFFFFFFu, incl, 2, 4); if (q >= 2) incl += y;
    const uint32_t excl = incl - sum;
    const bool mine = on && k >= excl && k < incl;
    uint32_t e = NONE32;
    if (mine) {                                                      // the word first, then one select inside it
        uint32_t kr = k - excl, wsel = 0, wi = 0;
        bool found = false;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const uint32_t pc = __popc(wv[i]);
            if (!found) {
                if (kr < pc) { found = true; wsel = wv[i]; wi = (uint32_t)i; }
                else kr -= pc;
            }
        }
        e = (w0 + wi) * 32 + a2_kth_bit32(wsel, kr);
    }
    const uint32_t bal = (__ballot_sync(0xFFFFFFFFu, mine) >> qbase) & 0xFu;
    const uint32_t own = bal ? (uint32_t)(__ffs(bal) - 1) : 0u;
    return __shfl_sync(0xFFFFFFFFu, e, qbase + own);
}

// candidates of row cbj with an entry index below hi, by the quad (same layout as a2_quad_select)
__device__ __forceinline__ uint32_t a2_quad_rank(const uint32_t* cbj, const uint32_t* grpj, uint32_t Wd, uint32_t hi, bool on,
                                                 uint32_t q) {
    uint32_t sum = 0;
    const uint32_t gh = hi >> 10, wh = hi >> 5;
    if (on) {
        for (uint32_t g = q; g < gh; g += 4) sum += grpj[g];          // whole groups below hi
        const uint32_t w0 = gh * 32 + q * 8;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const uint32_t wi = w0 + i;
            if (wi < Wd && wi <= wh) {
                const uint32_t word = cbj[wi];
                sum += __popc(wi < wh ? word : (word & ((1u << (hi & 31)) - 1u)));
            }
        }
    }
    sum += __shfl_xor_sync(0xFFFFFFFFu, sum, 1);
    sum += __shfl_xor_sync(0xFFFFFFFFu, sum, 2);
    return sum;
}

// The pick of one in-link by its quad: the k-th candidate, k = (r * n) >> 32 -- over all n candidates, or (PRIO, reading
// Q27) over the candidates of the first candidate's c.dist class: the entries are in (class, chunk id) order, so those are
// the candidates below the class's end bnd[.] and the k-th of them is the k-th candidate overall.
template <bool PRIO>
__device__ __forceinline__ uint32_t a2_pick(const uint32_t* cbj, const uint32_t* grpj, uint32_t Wd, uint32_t G, uint32_t n,
                                            uint32_t r, bool on, uint32_t q, uint32_t lane, const uint32_t* pb, uint32_t W) {
    if (PRIO) {
        const uint32_t e0 = a2_quad_select(cbj, grpj, Wd, G, 0u, on, q, lane);
        uint32_t hi = W;
        if (on) {
            const uint32_t nb = pb[0];
            for (uint32_t i = q; i <= nb; i += 4) { const uint32_t b = pb[1 + i]; if (b > e0) hi = min(hi, b); }
        }
        hi = min(hi, __shfl_xor_sync(0xFFFFFFFFu, hi, 1));
        hi = min(hi, __shfl_xor_sync(0xFFFFFFFFu, hi, 2));
        n = a2_quad_rank(cbj, grpj, Wd, hi, on, q);
    }
    return a2_quad_select(cbj, grpj, Wd, G, __umulhi(r, n), on, q, lane);
}

// The quads whose `doit` is set claim their entry e for in-link j4 = lane / 4 at time t: the entry leaves every
// in-link's candidates (lane q of the quad serves rows q and q + 4), the link is busy until t + w,
// the claim goes to the log at position rank.  Entries of different quads are distinct.
__device__ __forceinline__ void a2_commit(A2Fixed& f, uint32_t* live, uint32_t* cb, uint32_t* grp, uint32_t nin, uint32_t Wd,
                                          uint32_t G, bool doit, uint32_t e, uint32_t j4, uint32_t q4, unsigned long long t,
                                          U128* slot) {   // slot == nullptr: the log entry is already written
    if (doit) {
        const uint32_t bit = 1u << (e & 31);
#pragma unroll
        for (int x = 0; x < 2; ++x) {
            const uint32_t r = q4 + 4 * x;
            if (r < nin && (cb[r * Wd + (e >> 5)] & bit)) {
                atomicAnd(&cb[r * Wd + (e >> 5)], ~bit);
                atomicSub(&grp[r * G + (e >> 10)], 1u);
                atomicSub(&f.n[r], 1u);
            }
        }
        if (q4 == 0) {
            atomicAnd(&live[e >> 5], ~bit);
            f.free_te[j4] = t + f.w[j4];
            if (slot != nullptr) st128(slot, t, (unsigned long long)e | ((unsigned long long)j4 << 32));
        }
    }
}

template <bool PRIO>
__global__ void __launch_bounds__(A2_MAX_WARPS * 32, 1) k_loop2(const A2Args a) {
    extern __shared__ __align__(16) unsigned char a2_smem[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t v = blockIdx.x + warp * gridDim.x;
    if (v >= a.N) return;                                            // (no block-wide barrier anywhere below)
    const uint32_t W = a.wants_cnt[v];
    if (W == 0) return;                                              // header = (inf, 0) since k_a2_priv
    A2Fixed& f = *reinterpret_cast<A2Fixed*>(a2_smem + a.soff[v]);
    uint32_t* live = reinterpret_cast<uint32_t*>(&f + 1);
    const uint32_t e0 = a.in_off[v], nin = a.in_off[v + 1] - e0;
    const uint32_t Wd = (W + 31) >> 5, G = (Wd + 31) >> 5;
    uint32_t* cb = live + Wd;
    uint32_t* grp = cb + nin * Wd;
    const uint32_t* pb = grp + nin * G;                              // class boundaries (PRIO)
    // ---- static tables (once) ----
    if (lane == 0) {
        f.nin = nin; f.W = W; f.Wd = Wd; f.G = G;
        uint32_t ns = 0;
        for (uint32_t j = 0; j < nin; ++j) {
            const uint32_t l = a.in_link[e0 + j], u = a.esrc[l];
            f.link[j] = l; f.w[j] = a.w[l]; f.free_te[j] = 0;
            uint32_t s = 0;
            while (s < ns && f.s_node[s] != u) ++s;
            if (s == ns) {
                f.s_node[s] = u; f.s_W[s] = a.wants_cnt[u]; f.s_mask[s] = 0; f.cur[s] = 0;
                f.s_logbase[s] = a.nbase[u]; f.s_xbase[s] = a.loff[l];
                const uint32_t u0 = a.in_off[u], un = a.in_off[u + 1] - u0;
                unsigned long long wm = T_INF;
                for (uint32_t i = 0; i < 8; ++i) {
                    const unsigned long long wi = i < un ? a.w[a.in_link[u0 + i]] : T_INF;
                    f.hop_w[s * 8 + i] = wi;
                    wm = min(wm, wi);
                }
                f.s_wmin[s] = wm;
                ++ns;
            }
            f.sidx[j] = s;
            f.s_mask[s] |= 1u << j;
        }
        f.nsrc = ns;
    }
    for (uint32_t h = lane; h < A2_MAX_IN * 8; h += 32) { f.pend_e[h] = NONE32; f.pend_te[h] = T_INF; }
    {
        const uint32_t* img = a.priv + a.poff[v];
        const uint32_t words = a2_priv_words(W, nin, a.ncls);
        for (uint32_t i = lane; i < words; i += 32) live[i] = img[i];
    }
    __syncwarp();
    if (lane < nin) {                                                // n_j = sum of the group counts
        uint32_t s = 0;
        for (uint32_t g = 0; g < G; ++g) s += grp[lane * G + g];
        f.n[lane] = s;
    }
    __syncwarp();
    const uint32_t nsrc = f.nsrc;
    const int nslots = nsrc > 4 ? 2 : 1;                             // sources 4..7 use the second item of every lane
    U128* mylog = A2_LOG(a, a.nbase[v]);
    const uint32_t my_link = lane < nin ? f.link[lane] : 0u;
    // the two items of this lane in a poll: (source s0 = lane / 8, k = lane % 8) and (source s0 + 4, k); k = 0 is the
    // source's header, k = 1..7 its log entries cur + k - 1.  Everything static about the two sources sits in registers.
    const uint32_t kq = lane & 7, gl = lane & ~7u;
    bool p_act[2];
    unsigned long long p_wmin[2];
    const U128* p_ptr[2];            // header (k = 0) or log entry cur = 0 of this lane's k
    const uint32_t* p_xm[2];
    uint32_t p_W[2], p_cur[2];
#pragma unroll
    for (int sl = 0; sl < 2; ++sl) {
        const uint32_t s = sl * 4 + (lane >> 3);
        p_act[sl] = s < nsrc;
        p_wmin[sl] = p_act[sl] ? f.s_wmin[s] : 1ull;
        p_W[sl] = p_act[sl] ? f.s_W[s] : 0u;
        p_cur[sl] = 0;
        p_xm[sl] = a.xmap + (p_act[sl] ? f.s_xbase[s] : 0ull);
        p_ptr[sl] = !p_act[sl] ? a.hdr : (kq == 0 ? A2_HDR(a, f.s_node[s]) : A2_LOG(a, f.s_logbase[s] + (kq - 1)));
    }
    unsigned long long t = 0;
    uint32_t cnt = 0, remaining = W;
    unsigned long long st_actions = 0, st_polls = 0, st_picks = 0, st_slow = 0, st_bytes = 0;
#ifdef PCCL_A2_PROFILE
    long long pc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, pt = clock64();
#define A2_TICK(i) { const long long now__ = clock64(); pc[i] += now__ - pt; pt = now__; }
#else
#define A2_TICK(i)
#endif
    for (;;) {
        A2_TICK(0)
        // ---- wait for the sources, consume their claims (a3) ----
        // Per source (a group of 8 lanes): lane 0 holds the header and decides, lanes 1..7 hold the next log entries.
        // An entry is consumed when it is visible and starts early enough to arrive by t (t_start + wmin <= t), in log
        // order.  The source is settled once its header allows time t (LVT + wmin > t) and every entry the header counts
        // is consumed or visible but too late; what it can still send arrives no earlier than lane_lb.
        unsigned long long lane_lb[2] = {T_INF, T_INF};
        uint32_t need = (1u << nsrc) - 1u;           // sources not settled yet
        uint32_t spins = 0, r_mine = 0;
        bool have_r = false;
        // what this lane saw in the last evaluated poll of this event: a header is identified by its time (every header a
        // node stores carries a later time than the one before), a log entry by its second word (write-once)
        unsigned long long seen0 = 0, seen1 = 0;
        bool have_seen = false;
        uint32_t xh[2] = {NONE32, NONE32}, xv[2] = {NONE32, NONE32};   // consumed entry whose table word is still in flight
        unsigned long long xte[2] = {0, 0};
        while (need) {
            U128 it[2];
            {
                const uint32_t s0 = lane >> 3, s1 = 4 + s0;
                const bool on0 = p_act[0] && ((need >> s0) & 1u) && (kq == 0 || p_cur[0] + kq - 1 < p_W[0]);
                const bool on1 = nslots == 2 && p_act[1] && ((need >> s1) & 1u) && (kq == 0 || p_cur[1] + kq - 1 < p_W[1]);
                ld128x2(p_ptr[0] + (kq == 0 ? 0u : p_cur[0] * A2_LOG_STRIDE), on0, p_ptr[1] + (kq == 0 ? 0u : p_cur[1] * A2_LOG_STRIDE), on1, it[0], it[1]);
            }
            if (!have_r) {   // the pick's draw depends on (t, link) only: computed while the loads are in flight
                if (lane < nin) r_mine = philox_draw((uint32_t)t, (uint32_t)(t >> 32), my_link, 0u, a.k0, a.k1);
                have_r = true;
            }
            ++st_polls;
            st_bytes += 128u * (uint32_t)__popc(need);
            {   // nothing new since the last poll (same sources polled, same words back): evaluating it again would change
                // nothing -- poll again at once, so that the change is seen a whole evaluation earlier
                const unsigned long long now0 = kq == 0 ? it[0].lo : it[0].hi, now1 = kq == 0 ? it[1].lo : it[1].hi;
                const bool same = have_seen && now0 == seen0 && now1 == seen1;
                seen0 = now0; seen1 = now1;
                if (__all_sync(0xFFFFFFFFu, same)) {
                    if ((++spins & 63u) == 0u) {
                        if (ldcg32(a.abort_flag) != 0u) return;
                        if (spins > (1u << 24)) { if (lane == 0) atomicOr(a.abort_flag, 64u); return; }
                    }
                    continue;
                }
                have_seen = true;
            }
#ifdef PCCL_A2_PROFILE
            const long long q0 = clock64();
            { const unsigned long long z = __shfl_sync(0xFFFFFFFFu, it[0].lo ^ it[1].lo, 0); if (z == 0x1234567ull) ++st_polls; }
            const long long q1 = clock64();
            pc[6] += q1 - q0;
#endif
            bool nd[2] = {false, false};
#pragma unroll
            for (int sl = 0; sl < 2; ++sl) {
                if (sl < nslots) {
                    const uint32_t s = sl * 4 + (lane >> 3);
                    const bool act = p_act[sl] && ((need >> s) & 1u);
                    const unsigned long long wmin = p_wmin[sl];
                    const bool entry = act && kq > 0, valid = entry && it[sl].hi != T_INF;
                    const bool early = valid && it[sl].lo + wmin <= t;
                    const uint32_t cbits = (__ballot_sync(0xFFFFFFFFu, early) >> gl) & 0xFEu;
                    const uint32_t vbits = (__ballot_sync(0xFFFFFFFFu, valid) >> gl) & 0xFEu;
                    const uint32_t m = (uint32_t)__ffs(~(cbits >> 1)) - 1u;      // leading consumable entries (0..7)
                    if (act) {
                        const uint32_t ncur = p_cur[sl] + m;
                        p_cur[sl] = ncur;
                        if (kq == 0) {
                            const unsigned long long lvt = it[sl].lo;
                            const uint32_t count = (uint32_t)it[sl].hi;
                            const bool time_ok = lvt == T_INF || lvt + wmin > t;
                            lane_lb[sl] = T_INF;
                            if (ncur >= count) {                      // everything the header counts is consumed
                                nd[sl] = !time_ok;
                                if (lvt != T_INF) lane_lb[sl] = lvt + wmin;
                            } else if (m == 7 || !((vbits >> (m + 1)) & 1u)) {
                                nd[sl] = true;                        // more entries than one poll loads, or counted but not visible yet
                            } else {
                                nd[sl] = !time_ok;                    // the next entry is visible and too late (its lane holds the bound)
                            }
                        } else if (kq <= m) {                         // consume
                            if (xh[sl] != NONE32) { f.pend_e[xh[sl]] = xv[sl]; f.pend_te[xh[sl]] = xte[sl]; }
                            const uint32_t e_u = (uint32_t)it[sl].hi, j_u = (uint32_t)(it[sl].hi >> 32) & 7u;
                            xh[sl] = s * 8 + j_u;
                            xv[sl] = __ldg(p_xm[sl] + e_u);
                            xte[sl] = it[sl].lo + f.hop_w[xh[sl]];
                            lane_lb[sl] = T_INF;
                        } else {
                            lane_lb[sl] = (valid && !early) ? it[sl].lo + wmin : T_INF;
                        }
                    }
                }
            }
            {   // the header lanes' verdicts -> sources to poll again
                const uint32_t b0 = __ballot_sync(0xFFFFFFFFu, nd[0]) & 0x01010101u;
                need = (b0 | (b0 >> 7) | (b0 >> 14) | (b0 >> 21)) & 0xFu;
                if (nslots == 2) {
                    const uint32_t b1 = __ballot_sync(0xFFFFFFFFu, nd[1]) & 0x01010101u;
                    need |= ((b1 | (b1 >> 7) | (b1 >> 14) | (b1 >> 21)) & 0xFu) << 4;
                }
            }
#ifdef PCCL_A2_PROFILE
            pc[7] += clock64() - q1;
#endif
            if (need) {
                if ((++spins & 63u) == 0u) {
                    if (ldcg32(a.abort_flag) != 0u) return;
                    if (spins > (1u << 24)) { if (lane == 0) atomicOr(a.abort_flag, 64u); return; }
                }
            }
        }
        // ---- arrivals at the sources at time t become candidates (a3, a5).  First the pending table (arrivals consumed at
        //      earlier events), then the entries consumed just now: their table words are the last loads issued, and their
        //      round trip (about 800 cycles when an entry and its header became visible in the same poll) runs beside the
        //      table scan.  An entry that arrives later waits in the pending table ----
        ++st_actions;
        A2_TICK(1)
        unsigned long long nt_o = min(lane_lb[0], lane_lb[1]);     // this lane's share of the next event time
#pragma unroll
        for (int sl = 0; sl < 2; ++sl) {
            if (sl < nslots) {
                const uint32_t h = sl * 32 + lane;
                const unsigned long long te = f.pend_te[h];
                if (te <= t) {
                    const uint32_t e = f.pend_e[h];
                    f.pend_te[h] = T_INF;
                    if (e != NONE32 && ((live[e >> 5] >> (e & 31)) & 1u)) {
                        uint32_t m = f.s_mask[h >> 3];
                        while (m) {
                            const uint32_t j = __ffs(m) - 1;
                            m &= m - 1;
                            atomicOr(&cb[j * Wd + (e >> 5)], 1u << (e & 31));
                            atomicAdd(&grp[j * G + (e >> 10)], 1u);
                            atomicAdd(&f.n[j], 1u);
                        }
                    }
                } else {
                    nt_o = min(nt_o, te);
                }
            }
        }
        __syncwarp();                                               // (a slot is scanned before a new entry may take it)
#pragma unroll
        for (int sl = 0; sl < 2; ++sl) {
            if (xh[sl] != NONE32) {
                if (xte[sl] <= t) {
                    const uint32_t e = xv[sl];
                    if (e != NONE32 && ((live[e >> 5] >> (e & 31)) & 1u)) {
                        uint32_t m = f.s_mask[xh[sl] >> 3];
                        while (m) {
                            const uint32_t j = __ffs(m) - 1;
                            m &= m - 1;
                            atomicOr(&cb[j * Wd + (e >> 5)], 1u << (e & 31));
                            atomicAdd(&grp[j * G + (e >> 10)], 1u);
                            atomicAdd(&f.n[j], 1u);
                        }
                    }
                } else {
                    f.pend_e[xh[sl]] = xv[sl];
                    f.pend_te[xh[sl]] = xte[sl];
                    nt_o = min(nt_o, xte[sl]);
                }
            }
        }
        __syncwarp();
        A2_TICK(2)
        // ---- match (a4..a8): every free in-link with candidates picks; in-links in ascending link id, each seeing the
        //      earlier claims.  All picks are first made against the same state (one quad of lanes per in-link); the
        //      longest prefix that no earlier pick invalidates stands, the rest re-pick one by one.
        const uint32_t j4 = lane >> 2, q4 = lane & 3;
        uint32_t claims = 0;
        unsigned long long nt;
        {
            const bool inl = j4 < nin;
            const uint32_t nj = inl ? f.n[j4] : 0u;
            const unsigned long long frj = inl ? f.free_te[j4] : 0ull;
            const bool on = inl && nj != 0u && frj <= t;
            if (inl && q4 == 0 && frj > t) nt_o = min(nt_o, frj);                       // a busy in-link frees
            const uint32_t rj = __shfl_sync(0xFFFFFFFFu, r_mine, j4);
            const uint32_t e_spec = a2_pick<PRIO>(cb + (inl ? j4 : 0u) * Wd, grp + (inl ? j4 : 0u) * G, Wd, G, nj, rj, on, q4, lane, pb, W);
            const uint32_t onmask = __ballot_sync(0xFFFFFFFFu, on && q4 == 0);          // bit 4j
            // is an earlier pick i < j a candidate of in-link j?
            bool bad = false;
#pragma unroll
            for (int x = 0; x < 2; ++x) {
                const uint32_t i = q4 + 4 * x;
                const uint32_t ei = __shfl_sync(0xFFFFFFFFu, e_spec, (i * 4) & 31);
                if (on && i < j4 && ((onmask >> (4 * i)) & 1u) && ((cb[j4 * Wd + (ei >> 5)] >> (ei & 31)) & 1u)) bad = true;
            }
            const uint32_t badl = __ballot_sync(0xFFFFFFFFu, bad);
            const uint32_t first_bad = badl ? (uint32_t)(__ffs(badl) - 1) >> 2 : nin;
            A2_TICK(3)
            const bool stand = on && j4 < first_bad;
            const uint32_t smask = __ballot_sync(0xFFFFFFFFu, stand && q4 == 0);        // bit 4j
            if (stand && e_spec == NONE32) { atomicOr(a.abort_flag, 4u); return; }      // cannot happen
            U128* slot = mylog + (size_t)(cnt + __popc(smask & ((1u << (4 * j4)) - 1u))) * A2_LOG_STRIDE;
            claims = (uint32_t)__popc(smask);
            if (first_bad >= nin) {
                // the common case: every pick stands.  Publish first -- the claims, then the header with the next event
                // time -- and do the bookkeeping while the neighbours already read them
                if (stand && q4 == 0) {
                    st128(slot, t, (unsigned long long)e_spec | ((unsigned long long)j4 << 32));
                    nt_o = min(nt_o, t + f.w[j4]);
                }
                {   // 64-bit min over the warp: high words first, then the low words of the lanes that hold the smallest one
                    const uint32_t hi = (uint32_t)(nt_o >> 32), mh = __reduce_min_sync(0xFFFFFFFFu, hi);
                    const uint32_t ml = __reduce_min_sync(0xFFFFFFFFu, hi == mh ? (uint32_t)nt_o : 0xFFFFFFFFu);
                    nt = ((unsigned long long)mh << 32) | ml;
                }
                if (lane == 0) st128(A2_HDR(a, v), remaining == claims ? T_INF : nt, (unsigned long long)(cnt + claims));
                a2_commit(f, live, cb, grp, nin, Wd, G, stand, e_spec, j4, q4, t, nullptr);
                __syncwarp();
            } else {
                a2_commit(f, live, cb, grp, nin, Wd, G, stand, e_spec, j4, q4, t, slot);
                __syncwarp();
                for (uint32_t j = first_bad; j < nin; ++j) {
                    // exact re-pick against the state net of the claims so far
                    const uint32_t n2 = f.n[j];
                    if (n2 == 0u || f.free_te[j] > t) continue;
                    const uint32_t r2 = __shfl_sync(0xFFFFFFFFu, r_mine, j);
                    const uint32_t e2 = a2_pick<PRIO>(cb + j * Wd, grp + j * G, Wd, G, n2, r2, j4 == j, q4, lane, pb, W);
                    const uint32_t e = __shfl_sync(0xFFFFFFFFu, e2, 4 * j);
                    if (e == NONE32) { if (lane == 0) atomicOr(a.abort_flag, 4u); return; }   // cannot happen
                    a2_commit(f, live, cb, grp, nin, Wd, G, j4 == j, e, j4, q4, t, mylog + (size_t)(cnt + claims) * A2_LOG_STRIDE);
                    ++claims;
                    ++st_slow;
                    __syncwarp();
                }
                if (inl && q4 == 0) { const unsigned long long fr = f.free_te[j4]; if (fr > t) nt_o = min(nt_o, fr); }
                {
                    const uint32_t hi = (uint32_t)(nt_o >> 32), mh = __reduce_min_sync(0xFFFFFFFFu, hi);
                    const uint32_t ml = __reduce_min_sync(0xFFFFFFFFu, hi == mh ? (uint32_t)nt_o : 0xFFFFFFFFu);
                    nt = ((unsigned long long)mh << 32) | ml;
                }
                if (lane == 0) st128(A2_HDR(a, v), remaining == claims ? T_INF : nt, (unsigned long long)(cnt + claims));
            }
        }
        A2_TICK(4)
        st_picks += claims;
        cnt += claims;
        remaining -= claims;
        if (remaining == 0) break;
        if (nt == T_INF || nt <= t) { if (lane == 0) atomicOr(a.abort_flag, 128u); return; }   // cannot happen
        t = nt;
        A2_TICK(5)
    }
    if (lane == 0) {
        atomicAdd(&a.ctrl->actions, st_actions);
        atomicAdd(&a.ctrl->polls, st_polls);
        atomicAdd(&a.ctrl->picks, st_picks);
        atomicAdd(&a.ctrl->slow, st_slow);
        atomicAdd(&a.ctrl->bytes, st_bytes + 20ull * st_picks);   // + a log entry stored and a table word loaded per claim
#ifdef PCCL_A2_PROFILE
        for (int i = 0; i < 8; ++i) atomicAdd(&a.ctrl->prof[i], (unsigned long long)pc[i]);
#endif
    }
}

// ---------------------------------------------------------------------------------------------------------------
// emit: rank the logged claims into canonical (t_start, link) order (a8/a9) -- in WINDOWS of start times.
//
// A window takes every claim that starts before a bound `gvt` and has not been emitted yet.  With gvt = the smallest
// header time over all nodes (the simulation's global virtual time) those claims are final -- every node has logged
// all its claims that start before its own header time -- and all of them start at or after the previous window's
// bound, so their ranks simply continue where the previous window stopped: the windows can run on a second stream
// WHILE k_loop2 is still going (they only read headers and logs, k_loop2 never waits for them), and the host copies
// the finished prefix of the records out meanwhile.  A last window with gvt = inf after the loop takes the rest; a run
// that does not stream uses that window alone.  Per window: start times are hashed into a small table, the new
// distinct ones ranked, and a per-event link bitmap gives the position  base(event) + rank(link).
// A node's log is in time order, so a window's claims are the log entries [wcur, wnext) of each node.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t a2_time_slot(const A2Args& a, unsigned long long t) {
    const uint32_t mask = a.tcap - 1;
    uint32_t h = (uint32_t)((t * 0x9E3779B97F4A7C15ull) >> 32) & mask;
    for (uint32_t probes = 0; probes < a.tcap; ++probes) {
        unsigned long long k = ldcg64((const uint64_t*)a.tkey + h);
        if (k == t) return h;
        if (k == T_INF) {
            k = atomicCAS(a.tkey + h, T_INF, t);
            if (k == T_INF || k == t) return h;
        }
        h = (h + 1) & mask;
    }
    atomicOr(&a.ctrl->err, 1u);
    return 0;
}

// one block: the window's bound and the first of its distinct start times
__global__ void __launch_bounds__(1024) k_win_begin(A2Args a, int final) {
    __shared__ unsigned long long sm[32];
    unsigned long long g = T_INF;
    if (!final)
        for (uint32_t v = threadIdx.x; v < a.N; v += 1024) g = min(g, ld128(A2_HDR(a, v)).lo);
    for (int o = 16; o; o >>= 1) g = min(g, __shfl_xor_sync(0xFFFFFFFFu, g, o));
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = g;
    __syncthreads();
    if (threadIdx.x < 32) {
        g = sm[threadIdx.x];
        for (int o = 16; o; o >>= 1) g = min(g, __shfl_xor_sync(0xFFFFFFFFu, g, o));
        if (threadIdx.x == 0) { a.win->gvt = g; a.win->used0 = min(a.ctrl->n_start, a.ecap); }
    }
}

// block per node: hash the start and end time of every claim of the window; count the records per start time
__global__ void __launch_bounds__(256) k_win_times(A2Args a) {
    __shared__ uint32_t s_n;
    const unsigned long long gvt = a.win->gvt;
    unsigned long long tmax = 0;
  for (uint32_t v = blockIdx.x; v < a.N; v += gridDim.x) {   // (a block per node, or fewer blocks striding over the nodes)
    const uint32_t cnt = (uint32_t)ld128(A2_HDR(a, v)).hi, c0 = a.wcur[v];
    const unsigned long long base = a.nbase[v];
    const uint32_t e0 = a.in_off[v];
    __syncthreads();
    if (threadIdx.x == 0) s_n = 0;
    __syncthreads();
    uint32_t mine = 0;
    // A warp takes 32 consecutive log entries: claims of one event share their start time (and, on equal links, their
    // end time), so the lanes with the same time are served by ONE table lookup and one atomic per counter (config 5:
    // 7.76 M records on 2,744 start times -- every counter took thousands of atomics).
    for (uint32_t ib = c0 + (threadIdx.x & ~31u); ib < cnt; ib += blockDim.x) {   // (warp-uniform bounds)
        const uint32_t i = ib + (threadIdx.x & 31u);
        bool on = i < cnt;
        U128 en = {T_INF, T_INF};
        if (on) {
            en = ld128(A2_LOG(a, base + i));
            for (uint32_t spins = 0; en.hi == T_INF; ++spins) {   // counted by the header, the store is on its way
                if (spins > (1u << 22)) { atomicOr(a.abort_flag, 256u); break; }
                en = ld128(A2_LOG(a, base + i));
            }
            if (en.lo >= gvt) on = false;                         // (log in time order: so are the later ones)
        }
        if (!__any_sync(0xFFFFFFFFu, on)) break;
        uint32_t l = 0;
        unsigned long long te = T_INF;
        if (on) {
            ++mine;
            l = a.in_link[e0 + ((uint32_t)(en.hi >> 32) & 7u)];
            te = en.lo + a.w[l];
            tmax = max(tmax, te);
        }
        const unsigned long long ks = on ? en.lo : T_INF;
        const uint32_t g1 = __match_any_sync(0xFFFFFFFFu, ks), lead1 = (uint32_t)__ffs(g1) - 1u;
        uint32_t s = 0;
        if (on && lead1 == (threadIdx.x & 31u)) {
            s = a2_time_slot(a, en.lo);
            atomicAdd(&a.tcnt[s], (uint32_t)__popc(g1));
            if (!(atomicOr(&a.tflag[s], 2u) & 2u)) {
                const uint32_t k = atomicAdd(&a.ctrl->n_start, 1u);
                if (k < a.ecap) a.used[k] = s; else atomicOr(&a.ctrl->err, 1u);
            }
        }
        s = __shfl_sync(0xFFFFFFFFu, s, lead1);
        if (on) a.eslot[base + i] = s;
        const uint32_t g2 = __match_any_sync(0xFFFFFFFFu, te);
        if (on && (uint32_t)__ffs(g2) - 1u == (threadIdx.x & 31u)) {
            const uint32_t s2 = a2_time_slot(a, te);
            if (!(atomicOr(&a.tflag[s2], 1u) & 1u)) atomicAdd(&a.ctrl->n_end, 1u);
        }
    }
    if (mine) atomicAdd(&s_n, mine);
    __syncthreads();
    if (threadIdx.x == 0) {
        a.wnext[v] = c0 + s_n;
        if (s_n) atomicAdd(&a.ctrl->total, (unsigned long long)s_n);
    }
  }
    for (int o = 16; o; o >>= 1) tmax = max(tmax, __shfl_xor_sync(0xFFFFFFFFu, tmax, o));
    if ((threadIdx.x & 31) == 0) {
        if (tmax) atomicMax(&a.ctrl->tmax, tmax);
        if (2u * (a.ctrl->n_start + a.ctrl->n_end) > a.tcap) atomicOr(&a.ctrl->err, 1u);   // keep the table half empty
    }
}

// rank of every distinct start time of the window (a thread per time, all times compared through shared-memory tiles)
__global__ void __launch_bounds__(256) k_win_rank(A2Args a) {
    __shared__ unsigned long long tile[256];
    const uint32_t u0 = a.win->used0, n = min(a.ctrl->n_start, a.ecap) - u0;
    const uint32_t i = blockIdx.x * 256 + threadIdx.x;
    if (blockIdx.x * 256 >= n) return;
    const uint32_t slot = i < n ? a.used[u0 + i] : 0u;
    const unsigned long long mine = i < n ? a.tkey[slot] : T_INF;
    uint32_t rank = 0;
    for (uint32_t b = 0; b < n; b += 256) {
        __syncthreads();
        tile[threadIdx.x] = b + threadIdx.x < n ? a.tkey[a.used[u0 + b + threadIdx.x]] : T_INF;
        __syncthreads();
        const uint32_t m = min(256u, n - b);
        for (uint32_t k = 0; k < m; ++k) rank += tile[k] < mine;
    }
    if (i < n) { a.trank[slot] = u0 + rank; a.cnt_sorted[u0 + rank] = a.tcnt[slot]; }
}

// first record of every start time of the window (one block)
__global__ void __launch_bounds__(1024) k_win_base(A2Args a) {
    __shared__ unsigned long long sm[33];
    const uint32_t u0 = a.win->used0, n = min(a.ctrl->n_start, a.ecap) - u0;
    unsigned long long carry = a.win->emitted, tot;
    for (uint32_t b = 0; b < n; b += 1024) {
        const uint32_t i = b + threadIdx.x;
        const unsigned long long x = i < n ? a.cnt_sorted[u0 + i] : 0ull;
        const unsigned long long ex = block_excl_scan_1024(x, &tot, sm);
        if (i < n) a.ebase[u0 + i] = carry + ex;
        carry += tot;
    }
    if (threadIdx.x == 0) a.win->emitted_next = carry;
}

// the links matched at every start time of the window
__global__ void __launch_bounds__(256) k_win_bits(A2Args a) {
    if (a.ctrl->err & 1u) return;   // the table or the bitmaps overflowed: ranks are not valid, the host sorts instead
    for (uint32_t v = blockIdx.x; v < a.N; v += gridDim.x) {
        const uint32_t c0 = a.wcur[v], c1 = a.wnext[v];
        const unsigned long long base = a.nbase[v];
        const uint32_t e0 = a.in_off[v];
        for (uint32_t i = c0 + threadIdx.x; i < c1; i += blockDim.x) {
            const U128 en = ld128(A2_LOG(a, base + i));
            const uint32_t l = a.in_link[e0 + ((uint32_t)(en.hi >> 32) & 7u)];
            const uint32_t r = a.trank[a.eslot[base + i]];
            atomicOr(a.bm + (size_t)r * a.nLw + (l >> 6), 1ull << (l & 63));
        }
    }
}

// matched links before each 64-link word of every start time's row (a warp per row of the window)
__global__ void __launch_bounds__(256) k_win_wbase(A2Args a) {
    const uint32_t u0 = a.win->used0, u1 = min(a.ctrl->n_start, a.ecap);
    const uint32_t lane = threadIdx.x & 31;
    for (uint32_t r = u0 + blockIdx.x * 8 + (threadIdx.x >> 5); r < u1; r += gridDim.x * 8) {
        uint32_t run = 0;
        for (uint32_t wb = 0; wb < a.nLw; wb += 32) {
            const uint32_t wi = wb + lane;
            const uint32_t pc = wi < a.nLw ? __popcll(a.bm[(size_t)r * a.nLw + wi]) : 0u;
            const uint32_t incl = warp_incl_scan(pc, lane);
            if (wi < a.nLw) a.wbase[(size_t)r * a.nLw + wi] = run + incl - pc;
            run += __shfl_sync(0xFFFFFFFFu, incl, 31);
        }
    }
}

__global__ void __launch_bounds__(256) k_win_write(A2Args a) {
  const bool bad = (a.ctrl->err & 1u) != 0u;
  for (uint32_t v = blockIdx.x; v < a.N; v += gridDim.x) {
    const uint32_t c0 = a.wcur[v], c1 = a.wnext[v];
    __syncthreads();
    if (threadIdx.x == 0) a.wcur[v] = c1;                        // the next window starts here
    if (bad) continue;
    const unsigned long long base = a.nbase[v];
    const uint32_t e0 = a.in_off[v];
    const uint32_t* ids = a.ids + base;
    for (uint32_t i = c0 + threadIdx.x; i < c1; i += blockDim.x) {
        const U128 en = ld128(A2_LOG(a, base + i));
        const uint32_t l = a.in_link[e0 + ((uint32_t)(en.hi >> 32) & 7u)];
        const uint32_t r = a.trank[a.eslot[base + i]];
        const unsigned long long word = a.bm[(size_t)r * a.nLw + (l >> 6)];
        const unsigned long long pos = a.ebase[r] + a.wbase[(size_t)r * a.nLw + (l >> 6)] + __popcll(word & ((1ull << (l & 63)) - 1ull));
        if (pos >= a.out_cap) { atomicOr(&a.ctrl->err, 2u); continue; }
        const unsigned long long ts = en.lo + a.t_offset, te = en.lo + a.w[l] + a.t_offset;
        uint4* o = reinterpret_cast<uint4*>(a.out + pos);
        const uint32_t ch = ids[(uint32_t)en.hi];
        o[0] = make_uint4(a.orig != nullptr ? a.orig[ch] : ch, a.psrc[l], a.pdst[l], l);
        o[1] = make_uint4((uint32_t)ts, (uint32_t)(ts >> 32), (uint32_t)te, (uint32_t)(te >> 32));
    }
  }
}

// the window is written: records [0, emitted) are final (and told to the host when it is streaming them out)
__global__ void k_win_end(A2Args a) {
    const unsigned long long e = a.win->emitted_next;
    a.win->emitted = e;
    if (a.progress != nullptr && !(a.ctrl->err & 3u)) {
        __threadfence_system();
        *(volatile unsigned long long*)a.progress = e;
    }
}

// the claims as records in log order (no ranking): input of the reduce emitter's sort, and the fall-back when
// the time table or the per-event bitmaps are too small
__global__ void __launch_bounds__(256) k_emit_raw(A2Args a) {
    const uint32_t v = blockIdx.x;
    const uint32_t cnt = (uint32_t)ld128(A2_HDR(a, v)).hi;
    const unsigned long long base = a.nbase[v];
    const uint32_t e0 = a.in_off[v];
    const uint32_t* ids = a.ids + base;
    for (uint32_t i = threadIdx.x; i < cnt; i += blockDim.x) {
        const U128 en = *A2_LOG(a, base + i);
        const uint32_t l = a.in_link[e0 + ((uint32_t)(en.hi >> 32) & 7u)];
        if (base + i >= a.out_cap) { atomicOr(&a.ctrl->err, 2u); continue; }
        const unsigned long long ts = en.lo + a.t_offset, te = en.lo + a.w[l] + a.t_offset;
        uint4* o = reinterpret_cast<uint4*>(a.out + base + i);
        const uint32_t ch = ids[(uint32_t)en.hi];
        o[0] = make_uint4(a.orig != nullptr ? a.orig[ch] : ch, a.psrc[l], a.pdst[l], l);
        o[1] = make_uint4((uint32_t)ts, (uint32_t)(ts >> 32), (uint32_t)te, (uint32_t)(te >> 32));
    }
}

}  // namespace pccl
