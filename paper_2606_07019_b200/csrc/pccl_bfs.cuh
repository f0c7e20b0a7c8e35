// =====================================================================================
//  pccl_bfs.cuh -- the paper's own synthesizer on the GPU: Algorithms 1-3 with the timing
//  rules of section 4.6, condition by condition
//  (readings Q19-Q22).  PCCL_FLAG_BFS selects it.
//
//  What is computed (the same result as routing the conditions strictly one after another):
//    order      Alg. 3 lines 1-7: conditions by descending c.dist; ties by a Philox draw keyed
//               on the chunk (tag 2), then chunk id.
//    search     Alg. 2 + 4.6: earliest arrival of the chunk at every device, where link l may
//               start at the first s >= arrival(src(l)) with [s, s + w(l)) free on l; of
//               several links reaching a device at its earliest time the lowest link id is
//               recorded.
//    filter     PAPER.md:298: only the recorded paths src -> dests are kept.
//    remove     Alg. 3 line 13 / Fig. 10: their intervals become busy for later conditions.
//
//  How: conditions depend on each other only through busy intervals, so a WINDOW of B
//  consecutive conditions (one per CTA) is searched at once against the same snapshot of the
//  busy intervals, optimistically.  A result stays exact as long as none of its kept transfers
//  overlaps an interval taken by a condition earlier in the order (arrivals can only grow when
//  intervals are added, and a path whose own intervals are untouched still reaches its nodes
//  at the snapshot's earliest times, through the same lowest-id links).  Each round:
//    S  search (only CTAs whose result was invalidated or whose slot moved on) and post every
//       kept transfer on its link's round list
//    C  every condition looks for an overlap with a lower-positioned one on those lists;
//       first_bad = the lowest position that has one
//    M  conditions below first_bad commit: records are emitted, their intervals are merged into
//       the links' busy runs (one thread per link, no locks); later results that overlap a
//       committed interval are invalidated; the window slides to first_bad
//  with a grid barrier after each.  The position at the window base never has a conflict, so
//  every round commits at least one condition.
//
//  Busy runs of a link: sorted, disjoint [start, end) pairs in a row of R 16-byte entries
//  (entry 0 holds the count).  Every transfer on link l lasts w(l), so a gap shorter than w(l)
//  can never be used: such gaps are closed when runs are merged, which keeps rows short.
// =====================================================================================
#pragma once

namespace pccl {

struct BfsCtrl {
    unsigned long long first_bad[2];   // per round parity: lowest conflicting position
    unsigned long long nrec;           // records emitted (counted past the capacity too)
    unsigned long long tmax;           // max t_end (without the phase offset)
    unsigned long long searches, relax, rounds;
    unsigned long long ns_search, ns_check, ns_commit, iters;   // phase times seen by CTA 0 (barrier waits included)
    unsigned long long ns_sweeps, ns_filter;                    // summed over all searches: the sweeps, the path filter
    uint32_t nact;                     // conditions with at least one dest
    uint32_t err;                      // 1 unreachable, 2 time bits, 4 run row full, 8 record buffer full, 16 internal
};

struct BfsArgs {
    uint32_t os_in_smem, os_smem_off8;   // oslot copied to shared memory at this offset (in 8-byte words)
    uint32_t N, L, R, B, link_bits, nact, deg_shift;   // deg_shift: log2 of the lanes per frontier device
    const uint32_t* out_off;              // [N + 1] out-links per device in the direction being synthesized
    const uint4* oslot;                   // [L] per out-link entry: {link, far end, w lo, w hi}
    const uint32_t *esrc, *edst, *psrc, *pdst;
    const uint64_t* w;
    const uint32_t* cond_src;
    const uint64_t* dest_off;
    const uint32_t* dests;
    const uint32_t* order;             // [nact] chunk ids in routing order
    ulonglong2* runs;                  // [L][R]
    uint32_t* rl_n;                    // [L]    round list length
    uint64_t* rl_start;                // [L][B]
    uint32_t* rl_pos;                  // [L][B]
    uint32_t* tr_link;                 // [B][N] kept transfers of each slot
    uint64_t* tr_start;                // [B][N]
    Rec* out;
    uint64_t out_cap, t_offset;
    BfsCtrl* ctrl;
    const unsigned long long* t_ready;   // [C] time from which each chunk is at its source (pipelined All-Reduce, Q26), or null
    // switch model of section 4.7 (Q23-Q25); swidx == nullptr: none.  With a switch model the
    // window is one condition wide (B == 1): conditions are routed strictly one after another
    const uint32_t* swidx;            // [N] row of a node with a buffer limit in the stay tables, NONE32 otherwise
    const uint32_t* buf_limit;        // [N] chunks the node buffers at once (NONE32: no limit)
    const unsigned char* no_mcast;    // [N] non-zero: the node forwards one transfer at a time
    uint32_t n_lim, sb_cap;           // limited nodes; stays a row holds
    unsigned long long* sb_arr;       // [n_lim][sb_cap] arrival times of the stays committed so far, ascending
    unsigned long long* sb_rel;       // [n_lim][sb_cap] their release times, ascending
    uint32_t* sb_n;                   // [n_lim]
    unsigned long long* st_arr;       // [B][n_lim] stay of the slot's current result at each limited node ...
    unsigned long long* st_rel;       // [B][n_lim] ... release 0: the node does not forward the chunk
};

constexpr uint32_t BFS_THREADS = 1024;
constexpr unsigned long long BFS_INF = ~0ull;

__device__ __forceinline__ unsigned long long globaltimer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// ---- Alg. 3 lines 1-7: c.dist and the two sort keys ----------------------------------------
__global__ void k_bfs_keys(const uint32_t* __restrict__ cond_src, const uint64_t* __restrict__ dest_off,
                           const uint32_t* __restrict__ dests, uint32_t C, const uint32_t* __restrict__ sidx,
                           const uint64_t* __restrict__ D, uint32_t N, uint32_t k0, uint32_t k1,
                           uint64_t* __restrict__ cdist, uint64_t* __restrict__ key, uint32_t* __restrict__ val,
                           BfsCtrl* ctrl) {
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    const uint64_t d0 = dest_off[c], d1 = dest_off[c + 1];
    uint64_t dmax = 0;
    if (d1 > d0) {
        const uint64_t* row = D + (size_t)sidx[cond_src[c]] * N;
        for (uint64_t i = d0; i < d1; ++i) dmax = max(dmax, (uint64_t)row[dests[i]]);
        if (dmax == T_INF) atomicOr(&ctrl->err, 1u);
        atomicAdd(&ctrl->nact, 1u);
    }
    cdist[c] = dmax;                                   // 0 = nothing to route: sorts last
    key[c] = ((uint64_t)philox_draw(c, 0, 0, 2, k0, k1) << 32) | c;
    val[c] = c;
}

// second (stable) pass: descending c.dist
__global__ void k_bfs_keys2(const uint64_t* __restrict__ cdist, const uint32_t* __restrict__ val_in, uint32_t C,
                            uint64_t* __restrict__ key, uint32_t* __restrict__ val) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= C) return;
    const uint32_t c = val_in[i];
    key[i] = ~cdist[c];
    val[i] = c;
}

__global__ void k_bfs_pack(const uint32_t* __restrict__ out_link, const uint32_t* __restrict__ edst,
                           const uint64_t* __restrict__ w, uint32_t L, uint4* __restrict__ oslot) {
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= L) return;
    const uint32_t l = out_link[e];
    const uint64_t wl = w[l];
    oslot[e] = make_uint4(l, edst[l], (uint32_t)wl, (uint32_t)(wl >> 32));
}

__global__ void k_bfs_init(BfsArgs a) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < a.L) {
        a.runs[(size_t)i * a.R] = make_ulonglong2(0ull, 0ull);
        a.rl_n[i] = 0;
    }
    if (a.swidx != nullptr && i < a.n_lim) a.sb_n[i] = 0;
    if (i == 0) {
        a.ctrl->first_bad[0] = BFS_INF; a.ctrl->first_bad[1] = BFS_INF;
        a.ctrl->nrec = 0; a.ctrl->tmax = 0; a.ctrl->searches = 0; a.ctrl->relax = 0; a.ctrl->rounds = 0;
        a.ctrl->ns_search = 0; a.ctrl->ns_check = 0; a.ctrl->ns_commit = 0; a.ctrl->iters = 0; a.ctrl->ns_sweeps = 0; a.ctrl->ns_filter = 0;
    }
}

// ---- NextAvailableTime for one link (Alg. 1 + Fig. 10): first s >= a with [s, s + w) free ---
// bfs_occupy keeps every gap between consecutive runs >= w, so the first fit is either `a` itself (it fits
// in front of the first run that ends after a) or the end of that run.  Entry 0 of the row holds the run count
// and the end of the last run.  Measured on config 4: 67 % of the lookups come after the last run and are
// decided by entry 0 alone, 21 % by the first three runs, the rest have 4.5 runs on average.  A lookup is a
// scattered 16-byte load per lane and round, so it is written to need as few rounds as possible: entry 0 (the
// caller passes it, from shared memory when the headers fit there), then runs 1-7 together (the rest of the
// row's first 128-byte line), then a binary search.
__device__ __forceinline__ uint64_t bfs_depart(const ulonglong2* __restrict__ row, ulonglong2 h, uint64_t a, uint64_t w) {
    if (a >= h.y) return a;                            // h = entry 0: x = count, y = end of the last run (0: empty row)
    const uint32_t n = (uint32_t)h.x;
    ulonglong2 e[8];
#pragma unroll
    for (int k = 1; k <= 7; ++k) e[k] = __ldcg(row + k);   // the rest of the row's first 128-byte line, one round
    ulonglong2 r = make_ulonglong2(0ull, 0ull);
    bool found = false;
#pragma unroll
    for (int k = 7; k >= 1; --k)
        if ((uint32_t)k <= n && e[k].y > a) { r = e[k]; found = true; }
    if (!found) {                                      // a < end of the last run, so some run in [8, n] ends after a
        uint32_t lo = 8, hi = n;
        while (lo < hi) {
            const uint32_t mid = (lo + hi) >> 1;
            if (__ldcg(row + mid).y <= a) lo = mid + 1; else hi = mid;
        }
        r = __ldcg(row + lo);
    }
    return (a + w <= r.x) ? a : r.y;
}

// ---- section 4.7: chunks buffered at a limited node at time t = stays with arrival <= t < release -----------------
__device__ __forceinline__ uint32_t sb_upper(const unsigned long long* a, uint32_t n, unsigned long long t) {
    uint32_t lo = 0, hi = n;                            // first index with a[i] > t
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if (__ldcg(a + mid) <= t) lo = mid + 1; else hi = mid;
    }
    return lo;
}
// earliest start s >= a of link `row` (cost w) whose arrival s + w finds fewer than `limit` chunks buffered at the far
// node (stay tables arr / rel of n entries): first fit on the link, then wait for a release, and again
__device__ __forceinline__ uint64_t bfs_depart_buffered(const ulonglong2* __restrict__ row, uint64_t a, uint64_t w,
                                                        const unsigned long long* arr, const unsigned long long* rel, uint32_t n,
                                                        uint32_t limit) {
    for (;;) {
        const uint64_t s = bfs_depart(row, __ldcg(row), a, w);
        unsigned long long t = s + w;
        if (sb_upper(arr, n, t) - sb_upper(rel, n, t) < limit) return s;
        for (;;) {                                      // next time with a free buffer: walk the releases after t
            const uint32_t r = sb_upper(rel, n, t);
            t = __ldcg(rel + r);                        // (occupancy > 0: a release after t exists)
            if (sb_upper(arr, n, t) - sb_upper(rel, n, t) < limit) break;
        }
        a = t - w;
    }
}

// ---- Alg. 3 line 13: take [s, s + w) on a link (single writer per link) ----------------------
__device__ __forceinline__ bool bfs_occupy(ulonglong2* row, uint32_t R, uint64_t s, uint64_t w) {
    uint32_t n = (uint32_t)row[0].x;
    const uint64_t e = s + w;
    uint32_t i = 1;                                    // first run starting after s
    while (i <= n && row[i].x <= s) ++i;
    const bool mp = i > 1 && s - row[i - 1].y < w;     // gap to the run in front is unusable (or none)
    const bool mn = i <= n && row[i].x - e < w;
    if (mp && mn) {
        row[i - 1].y = row[i].y;
        for (uint32_t j = i; j < n; ++j) row[j] = row[j + 1];
        --n;
    } else if (mp) {
        row[i - 1].y = e;
    } else if (mn) {
        row[i].x = s;
    } else {
        if (n + 2 > R) return false;
        for (uint32_t j = n + 1; j > i; --j) row[j] = row[j - 1];
        row[i] = make_ulonglong2(s, e);
        ++n;
    }
    row[0] = make_ulonglong2((unsigned long long)n, row[n].y);
    return true;
}

// ---- pipelined All-Reduce (Q26): the reduce phase's records pre-occupy the links of the copy phase ----------
// ready[c] = end of the last transfer of chunk c into its root (the copy phase's source)
__global__ void k_bfs_ready(const Rec* __restrict__ pre, uint64_t n, const uint32_t* __restrict__ root,
                            unsigned long long* __restrict__ ready, uint32_t tbits, uint64_t* __restrict__ keys,
                            uint32_t* __restrict__ idx) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const Rec r = pre[i];
    if (r.dst == root[r.chunk]) atomicMax(&ready[r.chunk], (unsigned long long)r.t_end);
    keys[i] = ((uint64_t)r.link << tbits) | r.t_start;            // for the sort by (link, t_start)
    idx[i] = (uint32_t)i;
}
// one thread per link: its reduce-phase intervals, in time order, become busy runs
__global__ void k_bfs_preoccupy(BfsArgs a, const Rec* __restrict__ pre, uint64_t n, const uint64_t* __restrict__ keys,
                                const uint32_t* __restrict__ idx, uint32_t tbits) {
    const uint32_t l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= a.L) return;
    uint64_t lo = 0, hi = n;
    const uint64_t first = (uint64_t)l << tbits;
    while (lo < hi) {
        const uint64_t mid = (lo + hi) >> 1;
        if (keys[mid] < first) lo = mid + 1; else hi = mid;
    }
    ulonglong2* row = a.runs + (size_t)l * a.R;
    for (uint64_t i = lo; i < n && (keys[i] >> tbits) == l; ++i) {
        const Rec r = pre[idx[i]];
        if (!bfs_occupy(row, a.R, r.t_start, r.t_end - r.t_start)) { atomicOr(&a.ctrl->err, 4u); return; }
    }
}

// ---- Alg. 2 + 4.6 for one condition, by one CTA ---------------------------------------------
// key[v] = (arrival(v) << link_bits) | recorded link, so that one 64-bit min keeps the earliest
// arrival and, among equal arrivals, the lowest link id (reading Q20).  Label-correcting sweeps:
// the devices whose arrival improved in one sweep are the frontier of the next, one thread per
// (frontier device, out-link).  A device that arrives after every dest has been reached
// (`bound`) is not expanded: it can not lie on a kept path.  One block barrier per sweep.
struct BfsShared {
    unsigned long long bound;
    uint32_t nf[3];                 // frontier sizes, ring: sweep `it` reads [it % 3], fills [(it + 1) % 3]
    uint32_t cnt, minconf, fb_lo, fb_hi, base_idx_lo, base_idx_hi;
    unsigned long long tmax;
};

template <bool SW>   // SW: the switch model of section 4.7 is compiled in
__device__ void bfs_search(const BfsArgs& a, uint32_t chunk, unsigned long long* key, uint32_t* stamp, uint32_t* fr0, uint32_t* fr1,
                           const uint32_t* s_off, const uint4* s_os, ulonglong2* s_hdr,
                           BfsShared& sh, uint32_t slot, uint32_t& ntr, uint64_t& relax) {
    const uint32_t tid = threadIdx.x, lb = a.link_bits;
    const uint64_t lmask = (1ull << lb) - 1;
    const uint32_t src = a.cond_src[chunk];
    const uint64_t d0 = a.dest_off[chunk];
    const uint32_t nd = (uint32_t)(a.dest_off[chunk + 1] - d0);
    const uint32_t mds = a.deg_shift;
#ifdef PCCL_BFS_PROFILE
    unsigned long long dbg0 = 0, dbg1 = 0;
    if (tid == 0) dbg0 = globaltimer_ns();
#endif
    for (uint32_t v = tid; v < a.N; v += BFS_THREADS) { key[v] = BFS_INF; stamp[v] = NONE32; }
    if (s_hdr) for (uint32_t l = tid; l < a.L; l += BFS_THREADS) s_hdr[l] = __ldcg(a.runs + (size_t)l * a.R);
    if (tid == 0) { sh.nf[0] = 1; sh.nf[1] = 0; sh.nf[2] = 0; fr0[0] = src; }
    __syncthreads();
    if (tid == 0) {
        const unsigned long long t0 = a.t_ready != nullptr ? a.t_ready[chunk] : 0ull;
        if (t0 >> (64 - lb)) atomicOr(&a.ctrl->err, 2u);
        key[src] = t0 << lb;
    }
    __syncthreads();
    // 32 warps run every sweep, most of them without a frontier device: what they execute between two block
    // barriers is kept to a handful of instructions (the sweep is issue-bound otherwise)
    const uint32_t d_first = a.dests[d0];
    uint32_t r0 = 0, r1 = 1, r2 = 2;                    // ring positions of this, the next and the sweep after
    for (uint32_t it = 0;; ++it) {
        const uint32_t nf = sh.nf[r0];
        if (nf == 0 || it > a.N + 1) {
#ifdef PCCL_BFS_PROFILE
            if (tid == 0) atomicAdd(&a.ctrl->iters, (unsigned long long)it);
#endif
            if (tid == 0 && nf) atomicOr(&a.ctrl->err, 16u);
            break;
        }
        if (nd > 8) {                                   // many dests: max of their arrivals, by the whole CTA
            if (tid == 0) sh.bound = 0;
            __syncthreads();
            unsigned long long bl = 0;
            for (uint32_t k = tid; k < nd; k += BFS_THREADS) bl = max(bl, key[a.dests[d0 + k]] >> lb);
            if (bl) atomicMax(&sh.bound, bl);
            __syncthreads();
        }
        if (tid == 0) sh.nf[r2] = 0;
        const uint32_t* cur = (it & 1) ? fr1 : fr0;
        uint32_t* nxt = (it & 1) ? fr0 : fr1;
        uint32_t* nfn = &sh.nf[r1];
        { const uint32_t t = r0; r0 = r1; r1 = r2; r2 = t; }
        if (((tid & ~31u) >> mds) >= nf) { __syncthreads(); continue; }   // no frontier device for this whole warp
        unsigned long long bound;
        if (nd > 8) bound = sh.bound;
        else {
            bound = ((volatile unsigned long long*)key)[d_first] >> lb;
            for (uint32_t k = 1; k < nd; ++k) bound = max(bound, ((volatile unsigned long long*)key)[a.dests[d0 + k]] >> lb);
        }
        for (uint32_t j = tid >> mds; j < nf; j += BFS_THREADS >> mds) {     // 2^mds lanes per frontier device
            const uint32_t u = cur[j];
            const uint32_t o0 = s_off[u], deg = s_off[u + 1] - o0;
            const unsigned long long au = ((volatile unsigned long long*)key)[u] >> lb;
            if (au > bound) continue;
            // a node without multicast forwards over its out-links one after the other, in ascending link id (4.7): one
            // lane walks them, each transfer starting no earlier than the end of the one before
            const bool serial = SW && a.no_mcast[u] != 0;
            const uint32_t kstep = serial ? 1u : (1u << mds);
            uint64_t from = au;
            if (serial && (tid & ((1u << mds) - 1)) != 0) continue;
            for (uint32_t k = serial ? 0u : (tid & ((1u << mds) - 1)); k < deg; k += kstep) {
                const uint4 os = s_os ? s_os[o0 + k] : a.oslot[o0 + k];
                const uint32_t l = os.x, v = os.y;
                if (v == src && !serial) continue;
                const uint64_t wl = ((uint64_t)os.w << 32) | os.z;
                // a transfer over l ends no earlier than au + w(l): past the arrival at the last dest it can neither lie on
                // a kept path nor tie with one (only the paths to the dests are kept), so it is not looked up
                // and its far end is not expanded -- the search ends with the sweep that reaches the last dest
                if (!SW && au + wl > bound) continue;
                const ulonglong2* row = a.runs + (size_t)l * a.R;
                uint64_t cand;
                const uint32_t sr = SW ? a.swidx[v] : NONE32;
                if (sr != NONE32) {
                    const uint32_t lim = a.buf_limit[v];
                    if (lim == 0) continue;                        // a node that buffers nothing is never visited
                    cand = bfs_depart_buffered(row, from, wl, a.sb_arr + (size_t)sr * a.sb_cap, a.sb_rel + (size_t)sr * a.sb_cap,
                                               ldcg32(a.sb_n + sr), lim) + wl;
                } else {
                    cand = bfs_depart(row, s_hdr ? s_hdr[l] : __ldcg(row), from, wl) + wl;
                }
                if (serial) from = cand;
                ++relax;
                if (v == src) continue;
                if (cand >> (64 - lb)) { atomicOr(&a.ctrl->err, 2u); continue; }
                const unsigned long long kc = (cand << lb) | l;
                if (kc >= ((volatile unsigned long long*)key)[v]) continue;
                const unsigned long long old = atomicMin(&key[v], kc);
                if (kc < old && cand < (old >> lb)) {   // arrival improved: v is in the next frontier (once)
                    if (atomicExch(&stamp[v], it) != it) {
                        cg::coalesced_group g = cg::coalesced_threads();         // one counter update per warp
                        uint32_t b0 = 0;
                        if (g.thread_rank() == 0) b0 = atomicAdd(nfn, g.size());
                        nxt[g.shfl(b0, 0) + g.thread_rank()] = v;
                    }
                }
            }
        }
        __syncthreads();
    }
#ifdef PCCL_BFS_PROFILE
    if (tid == 0) dbg1 = globaltimer_ns();
#endif
    uint32_t* keep = fr0;                               // the frontier lists are dead now
    for (uint32_t v = tid; v < a.N; v += BFS_THREADS) keep[v] = 0;
    __syncthreads();
    // walk back from every dest; stop at a node that is already kept
    for (uint32_t k = tid; k < nd; k += BFS_THREADS) {
        uint32_t v = a.dests[d0 + k];
        if (key[v] == BFS_INF) { atomicOr(&a.ctrl->err, 1u); continue; }
        uint32_t guard = 0;
        while (v != src && atomicExch(&keep[v], 1u) == 0u) {
            v = a.esrc[(uint32_t)(key[v] & lmask)];
            if (++guard > a.N) { atomicOr(&a.ctrl->err, 16u); break; }
        }
    }
    if (tid == 0) sh.cnt = 0;
    __syncthreads();
    uint32_t* tl = a.tr_link + (size_t)slot * a.N;
    uint64_t* ts = a.tr_start + (size_t)slot * a.N;
    if (SW)                                             // (section 4.7) the stays of this result, per limited node
        for (uint32_t r = tid; r < a.n_lim; r += BFS_THREADS) a.st_rel[(size_t)slot * a.n_lim + r] = 0ull;
    __syncthreads();
    for (uint32_t v = tid; v < a.N; v += BFS_THREADS) {
        if (!keep[v]) continue;
        const uint32_t i = atomicAdd(&sh.cnt, 1u);
        const uint32_t l = (uint32_t)(key[v] & lmask);
        tl[i] = l;
        ts[i] = (key[v] >> lb) - a.w[l];
        if (SW) {                                       // the chunk stays buffered at the sender until this transfer ends
            const uint32_t u = a.esrc[l];
            const uint32_t sr = u != src ? a.swidx[u] : NONE32;
            if (sr != NONE32) {
                a.st_arr[(size_t)slot * a.n_lim + sr] = key[u] >> lb;
                atomicMax(&a.st_rel[(size_t)slot * a.n_lim + sr], key[v] >> lb);
            }
        }
    }
    __syncthreads();
    ntr = sh.cnt;
#ifdef PCCL_BFS_PROFILE
    if (tid == 0) { const unsigned long long dbg2 = globaltimer_ns(); atomicAdd(&a.ctrl->ns_sweeps, dbg1 - dbg0); atomicAdd(&a.ctrl->ns_filter, dbg2 - dbg1); }
#endif
}

template <bool SW>
__global__ void __launch_bounds__(BFS_THREADS) k_bfs(BfsArgs a) {
    cg::grid_group grid = cg::this_grid();
    extern __shared__ unsigned long long bfs_smem[];
    unsigned long long* key = bfs_smem;                         // [N]
    uint32_t* stamp = (uint32_t*)(key + a.N);                   // [N]
    uint32_t* fr0 = stamp + a.N;                                // [N] frontier lists; fr0 doubles as the keep marks
    uint32_t* fr1 = fr0 + a.N;                                  // [N]
    uint32_t* s_off = fr1 + a.N;                                // [N + 1] copy of out_off
    uint4* s_os = a.os_in_smem ? (uint4*)(bfs_smem + a.os_smem_off8) : nullptr;   // [L] copy of oslot when it fits
    ulonglong2* s_hdr = a.os_in_smem ? (ulonglong2*)(s_os + a.L) : nullptr;        // [L] entry 0 of every row, reloaded per search
    __shared__ BfsShared sh;
    const uint32_t tid = threadIdx.x, slot = blockIdx.x, B = a.B;
    const uint32_t gtid = blockIdx.x * BFS_THREADS + tid, gthreads = gridDim.x * BFS_THREADS;
    uint32_t* tl = a.tr_link + (size_t)slot * a.N;
    uint64_t* ts = a.tr_start + (size_t)slot * a.N;
    uint64_t base = 0, relax = 0, searches = 0;
    uint32_t pos = NONE32, ntr = 0;   // the result this CTA holds (CTA-uniform)
    for (uint32_t v = tid; v <= a.N; v += BFS_THREADS) s_off[v] = a.out_off[v];
    if (s_os) for (uint32_t e = tid; e < a.L; e += BFS_THREADS) s_os[e] = a.oslot[e];
    __syncthreads();
    bool valid = false;
    for (uint32_t round = 0; base < a.nact; ++round) {
        // ---- S: search + post ---------------------------------------------------------------
#ifdef PCCL_BFS_PROFILE
        unsigned long long tq0 = 0;
        if (gtid == 0) tq0 = globaltimer_ns();
#endif
        const uint64_t p64 = base + ((slot + B - (uint32_t)(base % B)) % B);
        const bool active = p64 < a.nact;
        const uint32_t p = (uint32_t)p64;
        if (active) {
            if (!(valid && pos == p)) {
                bfs_search<SW>(a, a.order[p], key, stamp, fr0, fr1, s_off, s_os, s_hdr, sh, slot, ntr, relax);
                pos = p; valid = true; ++searches;
            }
            for (uint32_t i = tid; i < ntr; i += BFS_THREADS) {
                const uint32_t l = tl[i];
                const uint32_t j = atomicAdd(&a.rl_n[l], 1u);
                if (j < B) { a.rl_start[(size_t)l * B + j] = ts[i]; a.rl_pos[(size_t)l * B + j] = p; }
                else atomicOr(&a.ctrl->err, 16u);
            }
        }
        grid.sync();
#ifdef PCCL_BFS_PROFILE
        unsigned long long tq1 = 0;
        if (gtid == 0) tq1 = globaltimer_ns();
#endif
        // ---- C: lowest earlier position whose transfer overlaps one of mine --------------------
        // (err is only written before the barrier above or after the next one: every CTA reads the same value)
        if (tid == 0) { sh.minconf = NONE32; sh.tmax = 0; sh.cnt = ldcg32(&a.ctrl->err) & (2u | 4u | 16u); }
        __syncthreads();
        if (sh.cnt) break;   // a run row overflowed or an invariant broke: the host retries or reports
        if (active) {
            uint32_t mc = NONE32;
            for (uint32_t i = tid; i < ntr; i += BFS_THREADS) {
                const uint32_t l = tl[i];
                const uint64_t s = ts[i], wl = a.w[l];
                const uint32_t n = min(ldcg32(a.rl_n + l), B);
                for (uint32_t j = 0; j < n; ++j) {
                    const uint32_t q = ldcg32(a.rl_pos + (size_t)l * B + j);
                    if (q >= p) continue;
                    const uint64_t sq = ldcg64(a.rl_start + (size_t)l * B + j);
                    if (s < sq + wl && sq < s + wl) mc = min(mc, q);
                }
            }
            if (mc != NONE32) atomicMin(&sh.minconf, mc);
        }
        __syncthreads();
        if (active && tid == 0 && sh.minconf != NONE32) atomicMin(&a.ctrl->first_bad[round & 1], (unsigned long long)p);
        grid.sync();
#ifdef PCCL_BFS_PROFILE
        unsigned long long tq2 = 0;
        if (gtid == 0) tq2 = globaltimer_ns();
#endif
        // ---- M: commit below first_bad ----------------------------------------------------------
        if (tid == 0) {
            const unsigned long long fbv = ldcg64((const uint64_t*)&a.ctrl->first_bad[round & 1]);
            const uint64_t lim = min((uint64_t)a.nact, base + B);
            const uint64_t fb = fbv < lim ? fbv : lim;
            sh.fb_lo = (uint32_t)fb; sh.fb_hi = (uint32_t)(fb >> 32);
            if (active && p < fb) {
                const unsigned long long bi = atomicAdd(&a.ctrl->nrec, (unsigned long long)ntr);
                sh.base_idx_lo = (uint32_t)bi; sh.base_idx_hi = (uint32_t)(bi >> 32);
            }
        }
        __syncthreads();
        const uint64_t fb = ((uint64_t)sh.fb_hi << 32) | sh.fb_lo;
        if (active && p < fb) {
            const uint64_t bi = ((uint64_t)sh.base_idx_hi << 32) | sh.base_idx_lo;
            const uint32_t chunk = a.order[p];
            unsigned long long tm = 0;
            for (uint32_t i = tid; i < ntr; i += BFS_THREADS) {
                const uint32_t l = tl[i];
                const uint64_t s = ts[i], e = s + a.w[l];
                tm = max(tm, (unsigned long long)e);
                if (bi + i < a.out_cap) a.out[bi + i] = Rec{chunk, a.psrc[l], a.pdst[l], l, s + a.t_offset, e + a.t_offset};
                else atomicOr(&a.ctrl->err, 8u);
            }
            if (tm) atomicMax(&sh.tmax, tm);
            __syncthreads();
            if (tid == 0 && sh.tmax) atomicMax(&a.ctrl->tmax, sh.tmax);
            if (SW) {
                // (section 4.7; one condition commits per round) its stays join the limited nodes' sorted tables
                __threadfence();
                for (uint32_t r = tid; r < a.n_lim; r += BFS_THREADS) {
                    const unsigned long long rel = __ldcg(a.st_rel + (size_t)slot * a.n_lim + r);
                    if (rel == 0ull) continue;
                    const unsigned long long arv = __ldcg(a.st_arr + (size_t)slot * a.n_lim + r);
                    const uint32_t n = a.sb_n[r];
                    if (n >= a.sb_cap) { atomicOr(&a.ctrl->err, 16u); continue; }
                    unsigned long long* A = a.sb_arr + (size_t)r * a.sb_cap;
                    unsigned long long* R = a.sb_rel + (size_t)r * a.sb_cap;
                    uint32_t i = n;
                    while (i > 0 && A[i - 1] > arv) { A[i] = A[i - 1]; --i; }
                    A[i] = arv;
                    i = n;
                    while (i > 0 && R[i - 1] > rel) { R[i] = R[i - 1]; --i; }
                    R[i] = rel;
                    a.sb_n[r] = n + 1;
                }
            }
            valid = false;
        } else if (active) {
            valid = sh.minconf == NONE32 || sh.minconf >= fb;
        }
        for (uint32_t l = gtid; l < a.L; l += gthreads) {
            const uint32_t n = min(ldcg32(a.rl_n + l), B);
            if (!n) continue;
            ulonglong2* row = a.runs + (size_t)l * a.R;
            const uint64_t wl = a.w[l];
            for (uint32_t j = 0; j < n; ++j) {
                if (ldcg32(a.rl_pos + (size_t)l * B + j) >= fb) continue;
                if (!bfs_occupy(row, a.R, ldcg64(a.rl_start + (size_t)l * B + j), wl)) atomicOr(&a.ctrl->err, 4u);
            }
            a.rl_n[l] = 0;
        }
        if (gtid == 0) { a.ctrl->first_bad[(round + 1) & 1] = BFS_INF; a.ctrl->rounds = round + 1; }
        base = fb;
        grid.sync();
#ifdef PCCL_BFS_PROFILE
        if (gtid == 0) {
            const unsigned long long tq3 = globaltimer_ns();
            a.ctrl->ns_search += tq1 - tq0; a.ctrl->ns_check += tq2 - tq1; a.ctrl->ns_commit += tq3 - tq2;
        }
#endif
    }
    // statistics
    for (int o = 16; o; o >>= 1) relax += __shfl_down_sync(0xFFFFFFFFu, relax, o);
    if ((tid & 31) == 0 && relax) atomicAdd(&a.ctrl->relax, (unsigned long long)relax);
    if (tid == 0 && searches) atomicAdd(&a.ctrl->searches, (unsigned long long)searches);
}

}  // namespace pccl
