// =========================================================================================
// pccl_device.cuh -- device code of the link-chunk matching synthesizer (sm_100a).
//
// Rows of DESIGN.md's hot-path table implemented here:
//   a0 k_link_cost      alpha-beta link cost
//   a1 k_distances      per-source shortest alpha-beta distances    (Alg. 3)
//   a2 k_have/k_wants   holdings + thin-relay-tree wants bitmaps
//   a3 loop phase P1    arrivals
//   a4 loop phase P2    active in-link compaction per destination   (Alg. 1)
//   a5 loop phase P2    candidate bitmap  have[src] & wants[dst]
//   a6 loop phase P2    Philox-keyed k-th-candidate pick
//   a7 loop phase P2    serial conflict resolve among in-links of one destination
//   a8 loop phase P2/P1 free-time advance, next-event min, ordered emit
//   a9 k_reverse + radix sort   reversal for reductions
//
// Nothing here is shared with oracle/ (the oracle is set-based C++ with its own Philox).
// =========================================================================================
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace cg = cooperative_groups;

namespace pccl {

constexpr uint64_t T_INF = 0xFFFFFFFFFFFFFFFFull;
constexpr uint32_t NONE32 = 0xFFFFFFFFu;
constexpr int NB = 8;              // most in-links of one destination served in one sweep (one warp each);
                                   // k_loop<NBT> runs NBT * 32 threads per CTA, NBT = 8 or 4
constexpr int LIST_CAP = 2048;     // candidate-sector work list entries per sweep (8 KB of shared memory)
constexpr int SEG_U4 = 32;         // uint4 per segment (one warp-wide load) = 64 words = 4096 chunks

struct Rec {  // == pccl_transfer_t
    uint32_t chunk, src, dst, link;
    uint64_t t_start, t_end;
};
static_assert(sizeof(Rec) == 32, "layout");

// ---- cache-bypassing accessors: all mutable state is read from / written to L2 ------------
// (the loop kernel is persistent, so L1 lines could otherwise outlive a grid barrier)
__device__ __forceinline__ uint64_t ldcg64(const uint64_t* p) { return __ldcg((const unsigned long long*)p); }
__device__ __forceinline__ uint32_t ldcg32(const uint32_t* p) { return __ldcg(p); }
__device__ __forceinline__ uint4 ldcg128(const uint4* p) { return __ldcg(p); }
__device__ __forceinline__ void stcg64(uint64_t* p, uint64_t v) { __stcg((unsigned long long*)p, (unsigned long long)v); }
__device__ __forceinline__ void stcg32(uint32_t* p, uint32_t v) { __stcg(p, v); }

__device__ __forceinline__ int popc128(uint4 a) { return __popc(a.x) + __popc(a.y) + __popc(a.z) + __popc(a.w); }
__device__ __forceinline__ uint4 and128(uint4 a, uint4 b) { return make_uint4(a.x & b.x, a.y & b.y, a.z & b.z, a.w & b.w); }

// ---- a6: Philox4x32-10 (Salmon et al., SC'11), first output word only ----------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__device__ __forceinline__ uint32_t philox_draw(uint32_t a, uint32_t b, uint32_t c, uint32_t tag,
                                                uint32_t k0, uint32_t k1) {
    uint32_t o[4];
    philox4x32_10(a, b, c, tag, k0, k1, o);
    return o[0];
}

__global__ void k_philox(const uint32_t* ctr, uint64_t n, uint32_t k0, uint32_t k1, uint32_t* out) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t o[4];
    philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], k0, k1, o);
    out[4 * i] = o[0]; out[4 * i + 1] = o[1]; out[4 * i + 2] = o[2]; out[4 * i + 3] = o[3];
}

// ---- a0: link cost ---------------------------------------------------------------------------
__global__ void k_link_cost(const uint64_t* __restrict__ alpha, const uint64_t* __restrict__ bpp,
                            uint32_t L, uint64_t chunk_bytes, uint64_t* __restrict__ w) {
    const uint32_t l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= L) return;
    const uint64_t b = bpp[l];
    w[l] = alpha[l] + chunk_bytes / b + (chunk_bytes % b != 0);
}

// ---- a1: shortest alpha-beta distances, one CTA per distinct source (Bellman-Ford in smem) ---
// esrc/edst: link endpoints in the direction being synthesized (swapped for the transposed run).
__global__ void k_distances(const uint32_t* __restrict__ esrc, const uint32_t* __restrict__ edst,
                            const uint64_t* __restrict__ w, uint32_t N, uint32_t L,
                            const uint32_t* __restrict__ sources, uint64_t* __restrict__ D) {
    extern __shared__ unsigned long long sdist[];
    __shared__ int s_changed;
    const uint32_t s = sources[blockIdx.x];
    for (uint32_t v = threadIdx.x; v < N; v += blockDim.x) sdist[v] = (v == s) ? 0ull : T_INF;
    __syncthreads();
    for (;;) {
        if (threadIdx.x == 0) s_changed = 0;
        __syncthreads();
        int changed = 0;
        for (uint32_t l = threadIdx.x; l < L; l += blockDim.x) {
            const unsigned long long du = ((volatile unsigned long long*)sdist)[esrc[l]];
            if (du == T_INF) continue;
            const unsigned long long nd = du + w[l];
            const uint32_t v = edst[l];
            if (nd < ((volatile unsigned long long*)sdist)[v]) {
                atomicMin(&sdist[v], nd);
                changed = 1;
            }
        }
        if (changed) s_changed = 1;
        __syncthreads();
        const int any = s_changed;
        __syncthreads();
        if (!any) break;
    }
    uint64_t* row = D + (size_t)blockIdx.x * N;
    for (uint32_t v = threadIdx.x; v < N; v += blockDim.x) row[v] = sdist[v];
}

// ---- a2: holdings ------------------------------------------------------------------------------
// hsum / wsum: one bit per 32-byte sector (4 words, 256 chunks) of a have / wants row, set while the
// sector may hold a set bit.  They are a filter only: a sector whose bit is 0 in either row cannot hold a
// candidate, so the count sweep never requests it.
__global__ void k_have(const uint32_t* __restrict__ cond_src, uint32_t C, uint32_t Wp, uint32_t SWp,
                       uint64_t* __restrict__ have, uint64_t* __restrict__ hsum) {
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    const uint32_t s = cond_src[c];
    atomicOr((unsigned long long*)&have[(size_t)s * Wp + (c >> 6)], 1ull << (c & 63));
    atomicOr((unsigned long long*)&hsum[(size_t)s * SWp + (c >> 14)], 1ull << ((c >> 8) & 63));
}

// ---- a2: wants = thin relay tree, one thread per (chunk, dest) pair ----------------------------
// Walk from the dest towards the source; at node `cur` the predecessor is the j-th tight
// in-link (ascending link id), j = (Philox(c, cur, 0, 1)[0] * |tight|) >> 32.  The choice is
// keyed on (c, cur) only, so walks of one chunk merge into a tree whatever order they run in;
// a walk stops at the first node already marked for its chunk.
__global__ void __launch_bounds__(128, 12) k_wants(const uint32_t* __restrict__ cond_src, const uint32_t* __restrict__ dests,
                        const uint32_t* __restrict__ dchunk, uint64_t n_pairs,
                        const uint32_t* __restrict__ esrc, const uint32_t* __restrict__ in_off,
                        const uint32_t* __restrict__ in_link, const uint64_t* __restrict__ w,
                        const uint32_t* __restrict__ sidx, const uint64_t* __restrict__ D, uint32_t N,
                        uint32_t Wp, uint32_t k0, uint32_t k1, uint64_t* __restrict__ wants, uint32_t* __restrict__ err,
                        const uint32_t* __restrict__ orig, uint32_t stage) {   // orig: the caller's id of a relabelled chunk (keys the draw)
    // stage != 0 (N * 8 bytes of dynamic shared memory): the distance row of the block's FIRST pair's source is copied to
    // shared memory.  Collectives list their chunks source by source, so nearly every pair of the block walks on that
    // row (config 4: 511 consecutive pairs per source) and its ~40 distance loads hit shared memory instead of L2;
    // a pair of another source reads its row from global memory as before.
    extern __shared__ uint64_t s_row[];
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t staged = NONE32;
    if (stage) {
        staged = sidx[cond_src[dchunk[(uint64_t)blockIdx.x * blockDim.x]]];
        const uint64_t* row = D + (size_t)staged * N;
        for (uint32_t i = threadIdx.x; i < N; i += blockDim.x) s_row[i] = row[i];
        __syncthreads();
    }
    if (p >= n_pairs) return;
    const uint32_t c = dchunk[p];
    const uint32_t ck = orig != nullptr ? orig[c] : c;
    const uint32_t s = cond_src[c];
    const uint32_t si = sidx[s];
    const uint64_t* Ds = si == staged ? s_row : D + (size_t)si * N;
    uint32_t cur = dests[p];
    if (Ds[cur] == T_INF) { atomicOr(err, 1u); return; }
    const unsigned long long bit = 1ull << (c & 63);
    while (cur != s) {
        // the mark's round trip (a third of the kernel's stall samples when it was waited for first) runs beside the
        // choice of the predecessor: `old` is only looked at once the next node is known
        const uint64_t dcur = Ds[cur];
        const uint32_t e0 = in_off[cur], e1 = in_off[cur + 1];
        const unsigned long long old = atomicOr((unsigned long long*)&wants[(size_t)cur * Wp + (c >> 6)], bit);
        uint32_t nxt = cur;
        if (e1 - e0 <= 32) {
            // one pass: tight in-links as a bit mask (ascending link id = ascending bit), then the j-th set bit
            uint32_t mask = 0;
            for (uint32_t e = e0; e < e1; ++e) {
                const uint32_t l = in_link[e];
                const uint64_t du = Ds[esrc[l]];
                if (du != T_INF && du + w[l] == dcur) mask |= 1u << (e - e0);
            }
            if (mask == 0) { atomicOr(err, 2u); return; }
            const uint32_t j = __umulhi(philox_draw(ck, cur, 0u, 1u, k0, k1), (uint32_t)__popc(mask));
            nxt = esrc[in_link[e0 + __fns(mask, 0, (int)j + 1)]];
        } else {
            uint32_t ntight = 0;
            for (uint32_t e = e0; e < e1; ++e) {
                const uint32_t l = in_link[e];
                const uint64_t du = Ds[esrc[l]];
                ntight += (du != T_INF && du + w[l] == dcur);
            }
            if (ntight == 0) { atomicOr(err, 2u); return; }
            uint32_t j = __umulhi(philox_draw(ck, cur, 0u, 1u, k0, k1), ntight);
            for (uint32_t e = e0; e < e1; ++e) {
                const uint32_t l = in_link[e];
                const uint32_t u = esrc[l];
                const uint64_t du = Ds[u];
                if (du != T_INF && du + w[l] == dcur) {
                    if (j == 0) { nxt = u; break; }
                    --j;
                }
            }
        }
        if (old & bit) break;                    // another walk of this chunk marked the node: it also goes on from here
        cur = nxt;
    }
}

// wants_cnt[v] = popcount of the wants row, wsum[v] = its sector summary: one streaming pass over the rows after the
// walks.  (Counted by the walks themselves these were 2 atomics per mark on N and N * C / 16384 hot addresses --
// same-address atomics are served one after the other: k_wants 180 -> ... us at config 4.)  One block per node.
__global__ void __launch_bounds__(256) k_wants_finish(const uint64_t* __restrict__ wants, uint32_t Wp, uint32_t SWp,
                                                      uint64_t* __restrict__ wsum, uint32_t* __restrict__ wants_cnt) {
    const uint32_t v = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint64_t* row = wants + (size_t)v * Wp;
    __shared__ uint32_t s_cnt[8];
    uint32_t cnt = 0;
    for (uint32_t sw = warp; sw < SWp; sw += 8) {          // a warp per summary word: 64 sectors of 4 words
        bool any[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t w0 = (sw * 64 + h * 32 + lane) * 4;
            uint64_t x[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) x[k] = w0 + k < Wp ? row[w0 + k] : 0ull;
            any[h] = (x[0] | x[1] | x[2] | x[3]) != 0ull;
            cnt += __popcll(x[0]) + __popcll(x[1]) + __popcll(x[2]) + __popcll(x[3]);
        }
        const uint32_t lo = __ballot_sync(0xFFFFFFFFu, any[0]), hi = __ballot_sync(0xFFFFFFFFu, any[1]);
        if (lane == 0) wsum[(size_t)v * SWp + sw] = ((uint64_t)hi << 32) | lo;
    }
    cnt = __reduce_add_sync(0xFFFFFFFFu, cnt);
    if (lane == 0) s_cnt[warp] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int k = 0; k < 8; ++k) t += s_cnt[k];
        wants_cnt[v] = t;
    }
}

// ---- a2 (dynamic relay, Q18): best[p] for every (chunk, dest) pair p starts at dist(source -> dest);
// Dto[row(d)][v] = alpha-beta shortest cost v -> d (k_distances on the reversed links)
__global__ void k_best_init(const uint32_t* __restrict__ cond_src, const uint32_t* __restrict__ dests,
                            const uint32_t* __restrict__ dchunk, uint64_t n_pairs,
                            const uint32_t* __restrict__ didx, const uint64_t* __restrict__ Dto, uint32_t N,
                            uint64_t* __restrict__ best, uint32_t* __restrict__ drow, uint32_t* __restrict__ err) {
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    const uint32_t row = didx[dests[p]];
    drow[p] = row;
    const uint64_t d0 = Dto[(size_t)row * N + cond_src[dchunk[p]]];
    if (d0 == T_INF) atomicOr(err, 1u);
    best[p] = d0;
}

// wants[u][c] = 1 iff some dest d of c has dist(u -> d) < best[c, d]; one warp per (node, 64-chunk word)
__global__ void k_wants_dyn_init(const uint64_t* __restrict__ dest_off, const uint32_t* __restrict__ dests,
                                 const uint32_t* __restrict__ didx, const uint64_t* __restrict__ Dto,
                                 const uint64_t* __restrict__ best, uint32_t N, uint32_t C, uint32_t Wp,
                                 uint32_t SWp, uint64_t* __restrict__ wants, uint64_t* __restrict__ wsum,
                                 uint32_t* __restrict__ wants_cnt) {
    // a warp per (node, 64-chunk word): lane b evaluates chunks b and 32 + b of the word, so the per-chunk tables
    // (dest_off, dests, best) are read coalesced; the two ballots are the word
    const uint32_t words = (C + 63) >> 6;
    const uint64_t wid = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t lane = threadIdx.x & 31;
    if (wid >= (uint64_t)N * words) return;   // warp-uniform
    const uint32_t u = (uint32_t)(wid / words), wi = (uint32_t)(wid % words);
    unsigned long long word = 0;
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        const uint32_t c = wi * 64 + half * 32 + lane;
        bool w = false;
        if (c < C) {
            const uint64_t p1 = dest_off[c + 1];
            for (uint64_t p = dest_off[c]; p < p1 && !w; ++p) w = Dto[(size_t)didx[dests[p]] * N + u] < best[p];
        }
        word |= (unsigned long long)__ballot_sync(0xFFFFFFFFu, w) << (32 * half);
    }
    if (lane == 0 && word) {
        wants[(size_t)u * Wp + wi] = word;
        atomicOr((unsigned long long*)&wsum[(size_t)u * SWp + (wi >> 8)], 1ull << ((wi >> 2) & 63));
        atomicAdd(&wants_cnt[u], (uint32_t)__popcll(word));
    }
}

// Alg. 3 lines 1-6: c.dist = max over dests of ShortestPath(c.src, dest); key = ~c.dist so that an
// ascending stable sort lists the farthest conditions first, equal ones in ascending chunk id
__global__ void k_cdist(const uint32_t* __restrict__ cond_src, const uint64_t* __restrict__ dest_off,
                        const uint32_t* __restrict__ dests, uint32_t C, const uint32_t* __restrict__ sidx,
                        const uint64_t* __restrict__ D, uint32_t N, uint64_t* __restrict__ cdist, uint64_t* __restrict__ key,
                        uint32_t* __restrict__ val) {
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    const uint64_t d0 = dest_off[c], d1 = dest_off[c + 1];
    uint64_t dmax = 0;
    if (d1 > d0) {
        const uint64_t* row = D + (size_t)sidx[cond_src[c]] * N;
        for (uint64_t i = d0; i < d1; ++i) dmax = max(dmax, (uint64_t)row[dests[i]]);
    }
    cdist[c] = dmax;
    key[c] = ~dmax;
    val[c] = c;
}

// sum of wants_cnt -> ctrl (one block)
__global__ void k_sum_u32(const uint32_t* __restrict__ x, uint32_t n, unsigned long long* out) {
    __shared__ unsigned long long s[32];
    unsigned long long acc = 0;
    for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) acc += x[i];
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        acc = (threadIdx.x < (blockDim.x >> 5)) ? s[threadIdx.x] : 0;
        for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
        if (threadIdx.x == 0) *out = acc;
    }
}

// wants bitmap -> (node, chunk) pairs in (node, chunk) order (parity-test accessor for row a2)
__global__ void k_wants_pairs(const uint64_t* __restrict__ wants, uint32_t N, uint32_t Wp,
                              const uint64_t* __restrict__ node_base, uint32_t* __restrict__ out_pairs,
                              uint64_t cap) {
    // one warp per node, sequential over the row
    const uint32_t v = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (v >= N) return;
    const uint32_t lane = threadIdx.x & 31;
    uint64_t pos = node_base[v];
    for (uint32_t wb = 0; wb < Wp; wb += 32) {
        const uint32_t wi = wb + lane;
        const uint64_t word = (wi < Wp) ? wants[(size_t)v * Wp + wi] : 0ull;
        const uint32_t pc = __popcll(word);
        uint32_t incl = pc;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if ((int)lane >= o) incl += y;
        }
        uint64_t my = pos + incl - pc;
        uint64_t x = word;
        while (x) {
            const int b = __ffsll((long long)x) - 1;
            x &= x - 1;
            if (my < cap) { out_pairs[2 * my] = v; out_pairs[2 * my + 1] = wi * 64 + b; }
            ++my;
        }
        pos += __shfl_sync(0xFFFFFFFFu, incl, 31);
    }
}

// ==================================================================================================
//  The event loop: one persistent cooperative kernel, two grid barriers per event time.
// ==================================================================================================
struct LoopCtrl {                 // device-resident control block (zeroed / initialised by k_loop_init)
    unsigned long long tnext[3];  // ring: next event time candidates
    unsigned long long total;     // transfers emitted so far
    unsigned long long tmax;      // max t_end
    unsigned long long events;    // event times processed
    unsigned long long rows_scanned;
    unsigned long long links_scanned;
    unsigned long long slow_picks;
    unsigned long long bytes_requested;
    unsigned long long wants_total;
    uint32_t err;
    uint32_t pad;
};

struct LoopArgs {
    uint32_t N, L, Wp, S;   // nodes, links, words per padded row, segments per row
    uint32_t nLw;           // words of the per-event matched-link bitmap
    uint32_t SWp;           // words per row of the sector summaries
    uint32_t flags;
    uint32_t k0, k1;        // Philox key
    const uint32_t* esrc;   // link endpoints in the synthesized direction
    const uint32_t* edst;
    const uint32_t* psrc;   // physical endpoints (what a record reports)
    const uint32_t* pdst;
    const uint32_t* in_off; // per-destination in-link table, ascending link id
    const uint32_t* in_link;
    const uint64_t* w;
    uint64_t* have;
    uint64_t* wants;
    uint64_t* hsum;         // [N][SWp] sector summaries of have / wants
    uint64_t* wsum;
    uint32_t* gcnt;         // [L][S] candidates of every link per 64-word segment, kept current (null: rescan mode)
    uint32_t* gtot;         // [L] their sum
    const uint32_t* out_link;  // per-node out-link table in the synthesized direction (entries)
    const uint32_t* out_far;   // far end of each entry: edst[out_link[e]]
    const uint32_t* lo_off;    // per link l: first entry / number of entries of the out-links of edst[l]
    const uint32_t* lo_deg;
    uint32_t* wants_cnt;
    uint64_t* free_t;
    uint32_t* inflight;
    uint32_t* have_epoch;
    uint32_t* empty_epoch;
    uint64_t* matchbits;    // [2][nLw]
    LoopCtrl* ctrl;
    Rec* out;
    uint64_t t_offset;      // added to the emitted times (phase 2 of all-reduce)
    // dynamic relay rule (null best: static thin relay tree)
    uint64_t* best;             // [pairs] smallest dist to the pair's dest over the source and all claimants
    const uint64_t* Dto;        // [distinct dests][N]
    const uint32_t* didx;       // [N] node -> row of Dto
    const uint64_t* dest_off;   // [C+1] pairs of each chunk
    const uint32_t* dests;      // [pairs]
    uint64_t out_cap;           // records the output buffer holds
    uint64_t* st_free;          // [2][L] link state double-buffered by event parity (k_loop1 only)
    uint32_t* st_inf;
    uint64_t* trace;        // optional [events][TRACE_SLOTS] globaltimer stamps of CTA 0 (diagnostic), or null
    uint32_t trace_cap;     // events the trace buffer holds
    // dynamic rule with kept counts: the holders of each chunk (nodes whose have bit is stored), so that a tightened
    // best only revisits the out-neighbours of holders (null: every node is revisited)
    const uint32_t* drow;       // [pairs] didx[dests[p]]: the pair's row of Dto
    const uint32_t* in_far;     // per in-link table entry: the link's source (esrc[in_link[e]])
    const uint32_t* csrc;       // [C] source of each chunk
    const uint32_t* out_off;    // [N+1] per-node offsets into out_link / out_far
    uint32_t* hold_cnt;         // [C] arrivals of the chunk so far
    uint32_t* hold;             // [C][HOLD_ROW] slots 1..HOLD_CAP: the first HOLD_CAP arrival nodes
    unsigned long long* progress;   // optional word in mapped pinned HOST memory: records [0, *progress) of `out` are
                                    // final (k_loop1 only; the host streams them out while the loop runs), or null
};

constexpr uint32_t HOLD_ROW = 32, HOLD_CAP = 31;
constexpr int TRACE_SLOTS = 12;  // 0 loop top, 1 links phase, 2 barrier 1, 3 in-link list, 4 count, 5 pick, 6 commit,
                                 // 7 barrier 2, 8 summary scan, 9 work list, 10 conflict resolve, 11 dynamic rule: the
                                 // wants-shrink of the event before (stamped between 0 and 1)
__device__ __forceinline__ void trace_stamp(const LoopArgs& a, uint32_t step, int slot) {
    if (a.trace != nullptr && blockIdx.x == 0 && threadIdx.x == 0 && step < a.trace_cap) {
        unsigned long long ns;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns));
        a.trace[(size_t)step * TRACE_SLOTS + slot] = ns;
    }
}

// a5 (initial): cnt[l][s] = | have[src_l] & wants[dst_l] | restricted to segment s, for every link; one CTA per
// link streams both rows once (128-bit coalesced loads).  The event loop then keeps the counts current.
__global__ void __launch_bounds__(256) k_count_init(LoopArgs a) {
    const uint32_t l = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t Q = a.Wp >> 1;
    const uint4* hrow = reinterpret_cast<const uint4*>(a.have) + (size_t)a.esrc[l] * Q;
    const uint4* wrow = reinterpret_cast<const uint4*>(a.wants) + (size_t)a.edst[l] * Q;
    __shared__ uint32_t wsumc[8];
    uint32_t mine = 0;
    for (uint32_t qb = warp * 32; qb < Q; qb += blockDim.x) {
        const uint32_t q = qb + lane;
        uint32_t pc = 0;
        if (q < Q) pc = popc128(and128(__ldg(hrow + q), __ldg(wrow + q)));
        const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, pc);
        if (lane == 0) { a.gcnt[(size_t)l * a.S + (qb >> 5)] = tot; mine += tot; }
    }
    if (lane == 0) wsumc[warp] = mine;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < 8; ++w) t += wsumc[w];
        a.gtot[l] = t;
    }
}

__global__ void k_loop_init(LoopArgs a) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < a.L) {
        a.free_t[i] = 0;
        a.inflight[i] = NONE32;
        a.empty_epoch[i] = 0;
    }
    if (i < a.N) a.have_epoch[i] = 0;
    if (i < a.L && a.st_free != nullptr) {
        a.st_free[i] = 0; a.st_free[a.L + i] = 0;
        a.st_inf[i] = NONE32; a.st_inf[a.L + i] = NONE32;
    }
    if (i < 3 * a.nLw) a.matchbits[i] = 0;
    if (i == 0) {
        a.ctrl->tnext[0] = 0;
        a.ctrl->tnext[1] = T_INF;
        a.ctrl->tnext[2] = T_INF;
        a.ctrl->total = 0;
        a.ctrl->tmax = 0;
        a.ctrl->events = 0;
        a.ctrl->rows_scanned = 0;
        a.ctrl->links_scanned = 0;
        a.ctrl->slow_picks = 0;
        a.ctrl->bytes_requested = 0;
    }
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t x, uint32_t lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
        if ((int)lane >= o) x += y;
    }
    return x;
}

// position of the k-th (0-based) set bit of a 128-bit value in ascending bit order
__device__ __forceinline__ uint32_t kth_bit128(uint4 m, uint32_t k) {
    uint32_t part[4] = {m.x, m.y, m.z, m.w};
    uint32_t base = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t pc = __popc(part[i]);
        if (k < pc) return base + __fns(part[i], 0, (int)k + 1);
        k -= pc;
        base += 32;
    }
    return 0xFFFFFFFFu;
}

// dynamic rule (Q18): node u still wants chunk c iff it is strictly closer to some dest of c than the
// best holder so far
__device__ __forceinline__ bool dyn_still_wants(const LoopArgs& a, uint32_t u, uint32_t c) {
    const uint64_t p1 = a.dest_off[c + 1];
    for (uint64_t p = a.dest_off[c]; p < p1; ++p)
        if (a.Dto[(size_t)a.drow[p] * a.N + u] < ldcg64(a.best + p)) return true;
    return false;
}

__device__ __forceinline__ void dyn_drop(const LoopArgs& a, uint32_t u, uint32_t c, uint64_t t);

// ---- P1: ordered emit of the previous event's matches (a8) + arrivals at time t (a3) ---------------
template <bool DYN>
__device__ __forceinline__ void loop_phase_links(const LoopArgs& a, uint32_t step, uint64_t t,
                                                 uint64_t emit_base) {
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t nW = (gridDim.x * blockDim.x) >> 5;
    const uint64_t* mbprev = a.matchbits + (size_t)((step + 1) & 1) * a.nLw;
    for (uint32_t lb = gw * 32; lb < a.L; lb += nW * 32) {
        const uint32_t l = lb + lane;
        const bool ok = l < a.L;
        uint32_t c = NONE32;
        uint64_t f = 0;
        if (ok) {
            c = ldcg32(a.inflight + l);
            f = ldcg64(a.free_t + l);
        }
        if (step > 0) {
            const uint32_t wq = lb >> 6;
            const uint64_t word = ldcg64(mbprev + wq);
            const uint32_t mine = (uint32_t)(word >> (lb & 32));   // this warp's 32 links
            if (mine != 0) {                                        // warp-uniform
                uint32_t pre = 0;
                for (uint32_t i = lane; i < wq; i += 32) pre += __popcll(ldcg64(mbprev + i));
                pre = __reduce_add_sync(0xFFFFFFFFu, pre);
                if (lb & 32) pre += __popc((uint32_t)word);
                if ((mine >> lane) & 1u) {
                    const uint64_t rank = pre + __popc(mine & ((1u << lane) - 1u));
                    const uint64_t wl = a.w[l];
                    if (emit_base + rank >= a.out_cap) {
                        atomicOr(&a.ctrl->err, 32u);   // the record is dropped, the run goes on: its total sizes the rerun
                    } else {
                        uint4* o = reinterpret_cast<uint4*>(a.out + emit_base + rank);
                        const uint64_t ts = f - wl + a.t_offset, te = f + a.t_offset;
                        o[0] = make_uint4(c, a.psrc[l], a.pdst[l], l);
                        o[1] = make_uint4((uint32_t)ts, (uint32_t)(ts >> 32), (uint32_t)te, (uint32_t)(te >> 32));
                    }
                }
            }
        }
        if (ok && c != NONE32 && f == t) {   // arrival: forwardable from t on
            const uint32_t d = a.edst[l];
            atomicOr((unsigned long long*)&a.have[(size_t)d * a.Wp + (c >> 6)], 1ull << (c & 63));
            atomicOr((unsigned long long*)&a.hsum[(size_t)d * a.SWp + (c >> 14)], 1ull << ((c >> 8) & 63));
            stcg32(a.have_epoch + d, step + 1);   // (inflight keeps the chunk: free_t == t holds at this event only)
            if (DYN && a.hold != nullptr) {
                const uint32_t k = atomicAdd(a.hold_cnt + c, 1u) + 1u;
                if (k <= HOLD_CAP) stcg32(a.hold + (size_t)c * HOLD_ROW + k, d);
            }
        }
    }
    // a5 (kept counts): the receiving node d now holds c, so c is a new candidate of every out-link of d whose
    // far end wants it.  One thread per (arriving link, k-th out-link of d), taken from the END of the grid so
    // that they run beside the warps above; three dependent round trips (link state, table entry, wants word).
    if (a.gcnt != nullptr) {
        constexpr uint32_t K = 8;
        const uint32_t nthreads = gridDim.x * blockDim.x;
        const uint32_t rid = nthreads - 1u - (blockIdx.x * blockDim.x + threadIdx.x);
        for (uint64_t it = rid; it < (uint64_t)a.L * K; it += nthreads) {
            const uint32_t l = (uint32_t)(it / K), k0 = (uint32_t)(it % K);
            const uint32_t c = ldcg32(a.inflight + l);
            const uint64_t f = ldcg64(a.free_t + l);
            const uint32_t off = a.lo_off[l], deg = a.lo_deg[l];
            if (c == NONE32 || f != t) continue;
            for (uint32_t k = k0; k < deg; k += K) {
                const uint32_t o = a.out_link[off + k], v2 = a.out_far[off + k];
                if ((ldcg64(a.wants + (size_t)v2 * a.Wp + (c >> 6)) >> (c & 63)) & 1ull) {
                    if (DYN && a.hold != nullptr && !dyn_still_wants(a, v2, c)) {
                        // lazy dynamic rule: v2 stopped wanting c -- either long ago, while no neighbour held it (then no
                        // count includes it), or at the event before this one (the shrink of that event runs beside
                        // these arrivals: whoever clears the bit takes the candidate away from the earlier holders)
                        dyn_drop(a, v2, c, t);
                    } else {
                        atomicAdd(&a.gcnt[(size_t)o * a.S + (c >> 12)], 1u);
                        atomicAdd(&a.gtot[o], 1u);
                    }
                }
            }
        }
    }
    // clear the bitmap the coming match phase writes; re-arm the ring slot after next
    uint64_t* mbcur = a.matchbits + (size_t)(step & 1) * a.nLw;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < a.nLw; i += gridDim.x * blockDim.x) stcg64(mbcur + i, 0);
    if (blockIdx.x == 0 && threadIdx.x == 0) stcg64((uint64_t*)&a.ctrl->tnext[(step + 2) % 3], T_INF);
}

// ---- dynamic relay rule, end of an event (Q18).  Every claim (c, v) of the event has tightened
// best[p] = min(best[p], dist(v -> d_p)) for the pairs p of c at commit; after the event's second barrier, for every
// claimed chunk, each node that is no longer strictly closer to some dest than the best holder stops wanting it
// (and, with kept counts, its in-links lose the candidate).  No barrier of its own: the phase runs BESIDE the
// arrivals of the next event time t (loop_phase_links), which read wants and set have bits -- both sides evaluate
// the same rule on the same best[] (nothing commits between the two barriers), the one that clears a bit does the
// whole upkeep, and "the source held c" below means "before the arrivals of time t".
// v stops wanting c (dynamic rule): clear the bit once, and with kept counts take the candidate away from every
// in-link of u whose source held c before time t.  A source that receives c at t itself (an in-link of it has
// inflight == c and free_t == t; its have bit may or may not be stored yet) never counted the candidate: its own
// arrival thread sees the bit cleared, or sees the rule fail.
__device__ __forceinline__ void dyn_drop(const LoopArgs& a, uint32_t u, uint32_t c, uint64_t t) {
    const unsigned long long bit = 1ull << (c & 63);
#ifdef PCCL_DEBUG_COUNTS
    if (u >= a.N || c >= a.Wp * 64u) { printf("[dbg] drop u %u c %u\n", u, c); return; }
#endif
    if (!(atomicAnd((unsigned long long*)&a.wants[(size_t)u * a.Wp + (c >> 6)], ~bit) & bit)) return;   // once per (u, c)
    atomicSub(&a.wants_cnt[u], 1u);
    if (a.gcnt == nullptr) return;
    const uint32_t e1 = a.in_off[u + 1];
    for (uint32_t eb = a.in_off[u]; eb < e1; eb += 4) {   // four in-links per round: table, source, have word
        uint32_t l2[4], u2[4];
        unsigned long long hw[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const bool in = eb + k < e1;
            l2[k] = in ? a.in_link[eb + k] : NONE32;
            u2[k] = in ? a.in_far[eb + k] : 0u;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) hw[k] = (l2[k] != NONE32) ? ldcg64(a.have + (size_t)u2[k] * a.Wp + (c >> 6)) : 0ull;
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if ((hw[k] >> (c & 63)) & 1ull) {
                bool now = false;                          // is c arriving at the source right now?
                const uint32_t f1 = a.in_off[u2[k] + 1];
                for (uint32_t f0 = a.in_off[u2[k]]; f0 < f1; f0 += 8) {   // eight in-links of the source per round trip
                    uint32_t li[8], ci[8];
#pragma unroll
                    for (int q = 0; q < 8; ++q) li[q] = f0 + q < f1 ? a.in_link[f0 + q] : NONE32;
#pragma unroll
                    for (int q = 0; q < 8; ++q) ci[q] = li[q] != NONE32 ? ldcg32(a.inflight + li[q]) : NONE32;
#pragma unroll
                    for (int q = 0; q < 8; ++q)
                        if (li[q] != NONE32 && ci[q] == c && ldcg64(a.free_t + li[q]) == t) now = true;
                }
                if (now) continue;
                atomicSub(&a.gcnt[(size_t)l2[k] * a.S + (c >> 12)], 1u);
                atomicSub(&a.gtot[l2[k]], 1u);
            }
    }
}

// every node that no longer wants claimed chunk c loses the bit (whole warp; scans all nodes)
__device__ __forceinline__ void dyn_shrink_chunk(const LoopArgs& a, uint32_t c, uint32_t lane, uint64_t t) {
    const uint64_t p0 = a.dest_off[c], p1 = a.dest_off[c + 1];
    const unsigned long long bit = 1ull << (c & 63);
    if (p1 - p0 <= 32) {
        // lane q holds pair q (row of its dest in Dto, current best); four nodes per lane and round, their
        // wants words loaded together, then one coalesced Dto load per pair and node
        const uint32_t np = (uint32_t)(p1 - p0);
        uint32_t row = 0;
        unsigned long long bst = 0;
        if (lane < np) { row = a.drow[p0 + lane]; bst = ldcg64(a.best + p0 + lane); }
        for (uint32_t ub = 0; ub < a.N; ub += 128) {
            bool need[4], keep[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t u = ub + 32 * k + lane;
                need[k] = u < a.N && (ldcg64(a.wants + (size_t)u * a.Wp + (c >> 6)) & bit) != 0ull;
                keep[k] = false;
            }
            for (uint32_t q = 0; q < np; ++q) {
                const uint32_t r = __shfl_sync(0xFFFFFFFFu, row, q);
                const unsigned long long b = __shfl_sync(0xFFFFFFFFu, bst, q);
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (need[k] && !keep[k]) keep[k] = a.Dto[(size_t)r * a.N + ub + 32 * k + lane] < b;
            }
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (need[k] && !keep[k]) dyn_drop(a, ub + 32 * k + lane, c, t);
        }
    } else {
        for (uint32_t u = lane; u < a.N; u += 32) {
            if (!(ldcg64(a.wants + (size_t)u * a.Wp + (c >> 6)) & bit)) continue;
            if (!dyn_still_wants(a, u, c)) dyn_drop(a, u, c, t);
        }
    }
}

// With holder lists (kept counts) only the out-neighbours of the chunk's holders are revisited: a wants bit can
// only be read through an in-link whose source holds the chunk (candidates are have[src] & wants[dst]), so the
// bits of all other nodes may stay stale until a neighbour receives the chunk -- the arrival then applies the rule
// (loop_phase_links).  A chunk with more than HOLD_CAP arrivals falls back to the scan over all nodes, which is
// exact whatever was skipped before.
// `step` is the event whose claims are applied, t the time of the event after it (whose arrivals run beside this).
__device__ __forceinline__ void dyn_shrink_wants(const LoopArgs& a, uint32_t step, uint64_t t) {
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nW = (gridDim.x * blockDim.x) >> 5;
    const uint64_t* mb = a.matchbits + (size_t)(step & 1) * a.nLw;
    for (uint32_t l = gw; l < a.L; l += nW) {   // a warp per link matched at this event
        if (!((ldcg64(mb + (l >> 6)) >> (l & 63)) & 1ull)) continue;
        const uint32_t c = ldcg32(a.inflight + l);
#ifdef PCCL_DEBUG_COUNTS
        if (c >= a.Wp * 64u) { if (lane == 0) printf("[dbg] shrink step %u link %u: inflight %u\n", step, l, c); continue; }
#endif
        if (a.hold == nullptr) { dyn_shrink_chunk(a, c, lane, t); continue; }
        // everything keyed on c in one round trip: the arrival count, the pairs, the holder slots (slots past the
        // count hold garbage and are masked below).  Lane 0: the source, lanes 1..nh: the arrival nodes
        // (the count moves while this runs -- the arrivals of time t append their nodes: ONE read for the whole warp)
        const uint32_t nh = __shfl_sync(0xFFFFFFFFu, ldcg32(a.hold_cnt + c), 0);
        const uint64_t p0 = a.dest_off[c], p1 = a.dest_off[c + 1];
        uint32_t u = (lane == 0) ? a.csrc[c] : ldcg32(a.hold + (size_t)c * HOLD_ROW + lane);
        if (nh > HOLD_CAP || p1 - p0 > 32) { dyn_shrink_chunk(a, c, lane, t); continue; }
        // (a slot of an arrival that is being appended right now may not be stored yet: whatever it holds, a node id is
        // revisited harmlessly -- the rule decides -- and anything else is skipped; the arrival's own thread applies the
        // rule to that node's out-neighbours)
        if (lane > nh || u >= a.N) u = NONE32;
        const uint32_t np = (uint32_t)(p1 - p0);
        uint32_t row = 0;               // lane q: pair q of c (row of its dest in Dto, current best)
        unsigned long long bst = 0;
        if (lane < np) { row = a.drow[p0 + lane]; bst = ldcg64(a.best + p0 + lane); }
        uint32_t off = 0, deg = 0;      // the holders' out-links, flattened over the warp
        if (u != NONE32) { off = a.out_off[u]; deg = a.out_off[u + 1] - off; }
        const uint32_t incl = warp_incl_scan(deg, lane);
        const uint32_t T = __shfl_sync(0xFFFFFFFFu, incl, 31);
        const unsigned long long bit = 1ull << (c & 63);
        for (uint32_t x0 = 0; x0 < T; x0 += 32) {
            const uint32_t x = x0 + lane;
            uint32_t j = 0;   // holder of item x: the number of holders whose items all come before x
            for (uint32_t jj = 0; jj <= nh; ++jj) j += (__shfl_sync(0xFFFFFFFFu, incl, jj) <= x) ? 1u : 0u;
            const uint32_t js = min(j, 31u);
            const uint32_t first = __shfl_sync(0xFFFFFFFFu, incl - deg, js), offj = __shfl_sync(0xFFFFFFFFu, off, js);
            uint32_t v2 = 0;
            bool need = false, keep = false;
            if (x < T) {
                v2 = a.out_far[offj + (x - first)];
                need = (ldcg64(a.wants + (size_t)v2 * a.Wp + (c >> 6)) & bit) != 0ull;
            }
            for (uint32_t q = 0; q < np; ++q) {
                const uint32_t r = __shfl_sync(0xFFFFFFFFu, row, q);
                const unsigned long long b = __shfl_sync(0xFFFFFFFFu, bst, q);
                if (need && !keep) keep = a.Dto[(size_t)r * a.N + v2] < b;
            }
            if (need && !keep) dyn_drop(a, v2, c, t);
        }
    }
}

// ---- P2: match one destination (a4..a8) -----------------------------------------------------------------
struct CtaScratch {
    uint32_t act[32];     // active in-links of the current window, ascending link id
    uint32_t src[32];     // their sources
    uint64_t actw[32];    // their costs
    uint32_t sempty[NB];  // speculative pick j empties its wants sector
    uint32_t acte[32];    // position of each active in-link in the destination's in-link list
    uint32_t pbits[NB];   // per speculative pick: mask over the in-links whose source holds the picked chunk
    uint32_t nact;
    uint32_t wc;          // chunks this destination still wants
    uint32_t wtot[NB];   // block scan scratch (one per warp)
    uint32_t spec[NB];    // speculative pick of each in-link of the sweep (NONE32: no candidate)
    uint32_t claimed[NB]; // chunks claimed so far in this sweep (warp 0 only)
};

struct LoopStats {
    unsigned long long rows, links, slow, bytes;
};

// (`extra[0..nextra)`: chunks to treat as held by the source although their have bit is not stored yet.)
// The k-th candidate (0-based, ascending chunk id) of link-row `hrow` AND wants-row `wrow`, given the
// per-segment candidate counts cj[0..S).  `excl[0..nex)` are chunks to treat as no longer wanted (claims
// made earlier in the same sweep); cj must already be net of them.  Whole warp; returns the chunk id.
__device__ __forceinline__ uint32_t kth_candidate(const uint32_t* cj, uint32_t S, uint32_t Q, const uint4* hrow,
                                                  const uint4* wrow, uint32_t rem, const uint32_t* excl,
                                                  uint32_t nex, uint32_t lane, bool& sector_empty,
                                                  const uint32_t* extra = nullptr, uint32_t nextra = 0) {
    uint32_t seg = 0;
    for (uint32_t sb = 0; sb < S; sb += 32) {
        const uint32_t x = (sb + lane < S) ? cj[sb + lane] : 0u;
        const uint32_t incl = warp_incl_scan(x, lane);
        const uint32_t tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
        if (rem < tot) {
            const uint32_t m = __ballot_sync(0xFFFFFFFFu, incl > rem);
            const int fl = __ffs(m) - 1;
            seg = sb + fl;
            rem -= __shfl_sync(0xFFFFFFFFu, incl - x, fl);
            break;
        }
        rem -= tot;
    }
    const uint32_t q = seg * SEG_U4 + lane;
    uint4 m4 = make_uint4(0, 0, 0, 0), wv = m4;
    if (q < Q) {
        wv = ldcg128(wrow + q);
        uint4 hv = ldcg128(hrow + q);
        for (uint32_t i = 0; i < nextra; ++i) {   // chunks the source holds as of now but whose bit is not stored yet
            const uint32_t c = extra[i];
            if (c != NONE32 && (c >> 7) == q) {
                const uint32_t b = c & 127u, bitm = 1u << (b & 31);
                if (b < 32) hv.x |= bitm; else if (b < 64) hv.y |= bitm; else if (b < 96) hv.z |= bitm; else hv.w |= bitm;
            }
        }
        m4 = and128(hv, wv);
    }
    for (uint32_t i = 0; i < nex; ++i) {
        const uint32_t c = excl[i];
        if ((c >> 7) == q) {
            const uint32_t b = c & 127u;
            const uint32_t msk = ~(1u << (b & 31));
            if (b < 32) { m4.x &= msk; wv.x &= msk; } else if (b < 64) { m4.y &= msk; wv.y &= msk; }
            else if (b < 96) { m4.z &= msk; wv.z &= msk; } else { m4.w &= msk; wv.w &= msk; }
        }
    }
    const uint32_t pc = popc128(m4);
    const uint32_t incl = warp_incl_scan(pc, lane);
    const uint32_t mm = __ballot_sync(0xFFFFFFFFu, incl > rem);
    const int fl = (__ffs(mm) - 1) & 31;
    const uint32_t rem2 = rem - __shfl_sync(0xFFFFFFFFu, incl - pc, fl);
    uint32_t c = NONE32;
    if ((int)lane == fl && mm != 0) {
        const uint32_t b = kth_bit128(m4, rem2);
        c = q * 128u + b;
        const uint32_t msk = ~(1u << (b & 31));
        if (b < 32) wv.x &= msk; else if (b < 64) wv.y &= msk; else if (b < 96) wv.z &= msk; else wv.w &= msk;
    }
    // the sector (this lane's 16 bytes and its pair lane's) holds no other wanted chunk
    const uint32_t z = (wv.x | wv.y | wv.z | wv.w) == 0u;
    sector_empty = (__shfl_sync(0xFFFFFFFFu, z, fl) & __shfl_sync(0xFFFFFFFFu, z, fl ^ 1)) != 0u;
    return __shfl_sync(0xFFFFFFFFu, c, fl);
}

__device__ __forceinline__ uint32_t warp_sum_counts(const uint32_t* cj, uint32_t S, uint32_t lane) {
    uint32_t n = 0;
    for (uint32_t s = lane; s < S; s += 32) n += cj[s];
    return __reduce_add_sync(0xFFFFFFFFu, n);
}

// a8: link l carries chunk c over [t, t + w_l); destination v no longer wants c
// dynamic relay rule: v becomes a holder of c, best[p] of c's pairs tightens (read only after the event's barrier)
template <bool DYN>
__device__ __forceinline__ void commit_best(const LoopArgs& a, uint32_t v, uint32_t c) {
    if (!DYN || a.best == nullptr) return;
    const uint64_t p1 = a.dest_off[c + 1];
    for (uint64_t p = a.dest_off[c]; p < p1; ++p)
        atomicMin((unsigned long long*)&a.best[p], (unsigned long long)a.Dto[(size_t)a.drow[p] * a.N + v]);
}

template <bool DYN>
__device__ __forceinline__ uint64_t commit_claim(const LoopArgs& a, uint32_t v, uint32_t l, uint64_t wl, uint32_t c,
                                                 bool sector_empty, uint32_t step, uint64_t t, bool tighten = true) {
    const uint64_t te = t + wl;
    atomicAnd((unsigned long long*)&a.wants[(size_t)v * a.Wp + (c >> 6)], ~(1ull << (c & 63)));
    // the pick saw no other wanted chunk in c's 32-byte sector: drop it from the wants summary.  (Two claims
    // of one sweep in one sector each see the other's bit and leave the summary bit set: a wasted load later,
    // never a wrong result -- the summaries are a filter only.)
    if (sector_empty) atomicAnd((unsigned long long*)&a.wsum[(size_t)v * a.SWp + (c >> 14)], ~(1ull << ((c >> 8) & 63)));
    stcg32(a.inflight + l, c);
    stcg64(a.free_t + l, te);
    atomicOr((unsigned long long*)&a.matchbits[(size_t)(step & 1) * a.nLw + (l >> 6)], 1ull << (l & 63));
    if (tighten) commit_best<DYN>(a, v, c);
    return te;
}

// static per-destination tables kept in shared memory for the destinations a CTA serves first
constexpr int DEST_CACHE = 2;
struct DestCache {
    uint32_t n_in;        // NONE32: not cached (more than 32 in-links)
    uint32_t link[32];
    uint32_t src[32];
    uint64_t w[32];
};

template <int NBT, bool DYN>
__device__ __forceinline__ void match_destination(const LoopArgs& a, uint32_t v, uint32_t step, uint64_t t,
                                                  uint32_t* cnt, uint32_t* list, CtaScratch& sh, LoopStats& st,
                                                  const DestCache* dc) {
    constexpr int THREADS = NBT * 32;   // one warp per in-link of a sweep
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t Q = a.Wp >> 1;  // uint4 per row
    const uint32_t SWp = a.SWp;
    const uint32_t S = a.S;
    const uint4* have4 = reinterpret_cast<const uint4*>(a.have);
    const uint4* wrow = reinterpret_cast<const uint4*>(a.wants) + (size_t)v * Q;
    uint32_t e0 = 0, e1 = 0;
    if (dc != nullptr) e1 = dc->n_in; else { e0 = a.in_off[v]; e1 = a.in_off[v + 1]; }
    uint32_t wc_start = 0;               // warp 0 only
    if (warp == 0) {
        wc_start = ldcg32(a.wants_cnt + v);
        if (lane == 0) sh.wc = wc_start;   // the other warps read it after the barrier below
    }
    uint64_t mymin = T_INF, mymax = 0;   // meaningful in warp 0 only
    const bool idle_skip = !(a.flags & 2u);

    for (uint32_t eb = e0; eb < e1; eb += 32) {
        // a4: active in-links of this window, ascending link id
        if (warp == 0) {
            const uint32_t e = eb + lane;
            const uint32_t wc = (eb == e0) ? wc_start : sh.wc;
            bool active = false;
            uint32_t l = 0, u = 0;
            if (e < e1) {
                if (dc != nullptr) { l = dc->link[e]; u = dc->src[e]; } else { l = a.in_link[e]; u = a.esrc[l]; }
                // one round trip: the three loads are independent
                const uint64_t f = ldcg64(a.free_t + l);
                const uint32_t ee = ldcg32(a.empty_epoch + l);
                const uint32_t he = ldcg32(a.have_epoch + u);
                const uint32_t nc = (a.gtot != nullptr) ? ldcg32(a.gtot + l) : 1u;
                if (f > t) {
                    mymin = min(mymin, f);
                } else if (wc > 0) {
                    // idle filter: nothing arrived at the source since this link last found no candidate
                    active = !(idle_skip && ee != 0 && ee >= he) && nc != 0u;
                }
            }
            const uint32_t m = __ballot_sync(0xFFFFFFFFu, active);
            if (active) {
                const uint32_t k = __popc(m & ((1u << lane) - 1u));
                sh.act[k] = l;
                sh.src[k] = u;
                sh.actw[k] = (dc != nullptr) ? dc->w[e] : a.w[l];
                sh.acte[k] = e - e0;
            }
            if (lane == 0) sh.nact = __popc(m);
        }
        __syncthreads();
        trace_stamp(a, step, 3);
        const uint32_t nact = sh.nact;
        for (uint32_t b0 = 0; b0 < nact; b0 += NBT) {
            if (sh.wc == 0) break;   // CTA-uniform: sh.wc only changes between the barriers below
            const uint32_t nb = min((uint32_t)NBT, nact - b0);
            // a5: candidate counts per 64-word segment.  Only sectors whose summary bit is set in BOTH the
            // wants row and the source row can hold a candidate.  (1) AND the summary rows; (2) expand the set
            // bits into a work list of (in-link, sector) items in shared memory (block-wide scan); (3) all
            // threads stride the list: two 128-bit loads of the source sector, two of the wants sector, AND,
            // popcount, shared-memory atomicAdd into the segment's counter.  Rows too dense for the list
            // (more than LIST_CAP candidate sectors) take the plain dense sweep instead.
            if (a.gcnt != nullptr) {
                // counts are kept current by arrivals (+) and claims (-): warp j copies the row of in-link j
                if (warp < nb) {
                    const uint32_t* g = a.gcnt + (size_t)sh.act[b0 + warp] * S;
                    for (uint32_t x = lane; x < S; x += 32) cnt[warp * S + x] = ldcg32(g + x);
                    if (lane == 0) st.bytes += (unsigned long long)S * 4u;
                }
            } else {
                const uint64_t* ws = a.wsum + (size_t)v * SWp;
                const uint32_t nitems = nb * SWp;
                const bool force_dense = (a.flags & 16u) != 0u;
                uint32_t total = force_dense ? (uint32_t)LIST_CAP + 1u : 0u;
                for (uint32_t base = 0; base < nitems && !force_dense; base += THREADS) {
                    const uint32_t it = base + tid;
                    unsigned long long m = 0;
                    uint32_t j = 0, i = 0;
                    if (it < nitems) {
                        j = it / SWp;
                        i = it - j * SWp;
                        m = ldcg64(ws + i) & ldcg64(a.hsum + (size_t)sh.src[b0 + j] * SWp + i);
                    }
                    const uint32_t pc = __popcll(m);
                    const uint32_t incl = warp_incl_scan(pc, lane);
                    if (lane == 31) sh.wtot[warp] = incl;
                    __syncthreads();
                    uint32_t pre = 0, blk = 0;
#pragma unroll
                    for (int w2 = 0; w2 < THREADS / 32; ++w2) {
                        const uint32_t x = sh.wtot[w2];
                        pre += (w2 < (int)warp) ? x : 0u;
                        blk += x;
                    }
                    uint32_t off = total + pre + incl - pc;
                    while (m) {
                        const uint32_t b = __ffsll((long long)m) - 1;
                        m &= m - 1;
                        if (off < LIST_CAP) list[off] = (j << 28) | (i * 64u + b);
                        ++off;
                    }
                    total += blk;
                    trace_stamp(a, step, 8);
                    __syncthreads();
                }
                for (uint32_t x = tid; x < nb * S; x += THREADS) cnt[x] = 0;
                __syncthreads();
                trace_stamp(a, step, 9);
                if (total <= LIST_CAP && total * 2u <= (nb + 1) * (Q >> 1)) {   // fewer sectors than the dense sweep
                    // a lane pair per item: even lane the first 16 bytes of the sector, odd lane the second, so
                    // that one warp-wide load touches 16 whole sectors; four items in flight per lane
                    const uint32_t half = tid & 1u;
                    constexpr uint32_t PAIRS = THREADS / 2, UNR = 4;
                    for (uint32_t idx = tid >> 1; idx < total; idx += UNR * PAIRS) {
                        uint32_t jj[UNR], ss[UNR];
                        uint4 hv[UNR], wv[UNR];
#pragma unroll
                        for (uint32_t k = 0; k < UNR; ++k) {
                            const uint32_t ix = idx + k * PAIRS;
                            hv[k] = make_uint4(0, 0, 0, 0);
                            wv[k] = hv[k];
                            jj[k] = 0; ss[k] = 0;
                            if (ix < total) {
                                const uint32_t e = list[ix];
                                jj[k] = e >> 28;
                                ss[k] = e & 0x0FFFFFFFu;
                                hv[k] = ldcg128(have4 + (size_t)sh.src[b0 + jj[k]] * Q + 2u * ss[k] + half);
                                wv[k] = ldcg128(wrow + 2u * ss[k] + half);
                            }
                        }
#pragma unroll
                        for (uint32_t k = 0; k < UNR; ++k) {
                            const uint32_t pcs = popc128(and128(hv[k], wv[k]));
                            if (pcs) atomicAdd(&cnt[jj[k] * S + (ss[k] >> 4)], pcs);
                        }
                    }
                    if (tid == 0) st.bytes += (unsigned long long)total * 64u + (unsigned long long)nitems * 16u;
                } else {
                    // dense sweep: every lane one uint4 of the wants row and of each source row
                    size_t hoff[NBT];
#pragma unroll
                    for (int j = 0; j < NBT; ++j) hoff[j] = (size_t)sh.src[b0 + (j < (int)nb ? j : 0)] * Q;
                    for (uint32_t qb = warp * 32; qb < Q; qb += blockDim.x) {
                        const uint32_t q = qb + lane;
                        const bool ok = q < Q;
                        uint4 wv = make_uint4(0, 0, 0, 0);
                        uint4 h[NBT];
                        if (ok) wv = ldcg128(wrow + q);
#pragma unroll
                        for (int j = 0; j < NBT; ++j) {   // all loads of the slice in flight before the first use
                            h[j] = make_uint4(0, 0, 0, 0);
                            if (j < (int)nb && ok) h[j] = ldcg128(have4 + hoff[j] + q);
                        }
#pragma unroll
                        for (int j = 0; j < NBT; ++j) {
                            if (j < (int)nb) {
                                const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, (uint32_t)popc128(and128(h[j], wv)));
                                if (lane == 0) cnt[j * S + (qb >> 5)] = tot;
                            }
                        }
                    }
                    if (tid == 0) st.bytes += (unsigned long long)(nb + 1) * a.Wp * 8u + (force_dense ? 0ull : (unsigned long long)nitems * 16u);
                }
            }
            __syncthreads();
            trace_stamp(a, step, 4);
            // a6: every in-link of the sweep picks from the wants row as it stood at the start of the
            // sweep -- exact unless an earlier in-link's claim is also held by a later in-link's source
            if (warp < nb) {
                const uint32_t l = sh.act[b0 + warp];
                const uint32_t* cj = cnt + warp * S;
                const uint32_t n = warp_sum_counts(cj, S, lane);
                uint32_t c = NONE32;
                bool sem = false;
                if (n != 0) {
                    const uint32_t r = philox_draw((uint32_t)t, (uint32_t)(t >> 32), l, 0u, a.k0, a.k1);
                    c = kth_candidate(cj, S, Q, have4 + (size_t)sh.src[b0 + warp] * Q, wrow, __umulhi(r, n), nullptr, 0, lane, sem);
                    if (c == NONE32 && lane == 0) atomicOr(&a.ctrl->err, 4u);   // cannot happen
                }
                if (lane == 0) {
                    sh.spec[warp] = c;
                    sh.sempty[warp] = sem;
                    if (n != 0) st.bytes += 2u * SEG_U4 * 16u;   // one segment of the source row and of the wants row
                }
            }
            __syncthreads();
            trace_stamp(a, step, 5);
            // a7: conflict resolve.  In-links are served in ascending link id, each seeing the earlier
            // claims.  Link j's speculative pick stands iff no earlier claim is a candidate of j.
            if (warp == 0 && dc != nullptr && a.gcnt != nullptr) {
                // <= 32 in-links, tables in shared memory, kept counts.  The picks are settled prefix by prefix: the
                // longest run of picks that no earlier final pick invalidates is committed at once; the first
                // invalidated link re-picks exactly (it is the first unsettled one), its new pick replaces its
                // speculative one in the test, and the links after it keep their speculative picks unless THAT
                // invalidates them.  Same result as serving the links one by one.
                st.rows += nb + 1;
                st.links += nb;
                // H[i] (sh.pbits[i]): mask over the in-links of v whose source holds pick i -- one load per (pick,
                // in-link); serves the test and the count upkeep
                if (lane < NBT) sh.pbits[lane] = 0;
                __syncwarp();
                const uint32_t npairs = nb * e1;
                for (uint32_t p0 = 0; p0 < npairs; p0 += 64) {   // two pairs per lane and round, loads first
                    const uint32_t pa = p0 + lane, pb = p0 + 32 + lane;
                    uint32_t ia = 0, ea = 0, ib = 0, eb2 = 0, ca = NONE32, cb = NONE32;
                    unsigned long long wa = 0, wb = 0;
                    if (pa < npairs) { ia = pa / e1; ea = pa - ia * e1; ca = sh.spec[ia]; }
                    if (pb < npairs) { ib = pb / e1; eb2 = pb - ib * e1; cb = sh.spec[ib]; }
                    if (ca != NONE32) wa = ldcg64(a.have + (size_t)dc->src[ea] * a.Wp + (ca >> 6));
                    if (cb != NONE32) wb = ldcg64(a.have + (size_t)dc->src[eb2] * a.Wp + (cb >> 6));
                    if (ca != NONE32 && ((wa >> (ca & 63)) & 1ull)) atomicOr(&sh.pbits[ia], 1u << ea);
                    if (cb != NONE32 && ((wb >> (cb & 63)) & 1ull)) atomicOr(&sh.pbits[ib], 1u << eb2);
                }
                __syncwarp();
                if (lane == 0) st.bytes += (unsigned long long)nb * e1 * 32u;
                trace_stamp(a, step, 8);
                const uint32_t ej = (lane < nb) ? sh.acte[b0 + lane] : 0u;
                uint32_t wc = sh.wc, ncl = 0, done = 0, repicked = 0;
                while (done < nb) {
                    // the first unsettled link whose source holds an earlier pick (sh.spec holds the final pick of every
                    // settled link and the speculative one of the others)
                    bool isbad = false;
                    if (lane >= done && lane < nb)
                        for (uint32_t i = 0; i < lane; ++i)
                            if (sh.spec[i] != NONE32 && ((sh.pbits[i] >> ej) & 1u)) isbad = true;
                    const uint32_t bm = __ballot_sync(0xFFFFFFFFu, isbad);
                    const uint32_t fb = bm ? (uint32_t)(__ffs(bm) - 1) : nb;
                    // commit [done, fb): one lane per link
                    {
                        const bool mine = lane >= done && lane < fb;
                        uint32_t c = NONE32, l = 0;
                        if (mine) { c = sh.spec[lane]; l = sh.act[b0 + lane]; }
                        const uint32_t cm = __ballot_sync(0xFFFFFFFFu, c != NONE32);
                        if (mine) {
                            if (c != NONE32) {
                                const uint64_t te = commit_claim<DYN>(a, v, l, sh.actw[b0 + lane], c, sh.sempty[lane] != 0u, step, t);
                                mymin = min(mymin, te);
                                mymax = max(mymax, te);
                                sh.claimed[ncl + __popc(cm & ((1u << lane) - 1u))] = c;
                            } else {
                                stcg32(a.empty_epoch + l, step + 1);
                            }
                        }
                        ncl += __popc(cm);
                        wc -= __popc(cm);
                        __syncwarp();
                        if (lane < e1) {   // count upkeep for these picks: lane e owns in-link e of v
                            const uint32_t l2 = dc->link[lane];
                            uint32_t dec = 0;
                            for (uint32_t i = done; i < fb; ++i) {
                                const uint32_t ci = sh.spec[i];
                                if (ci != NONE32 && ((sh.pbits[i] >> lane) & 1u)) {
                                    atomicSub(&a.gcnt[(size_t)l2 * S + (ci >> 12)], 1u);
                                    ++dec;
                                }
                            }
                            if (dec) atomicSub(&a.gtot[l2], dec);
                        }
                    }
                    if (fb >= nb) break;
                    if (wc == 0) break;   // v wants nothing more: no later link can have a candidate
                    // link fb re-picks against the wants row net of the claims so far
                    if (lane == 0) ++st.slow;
                    const uint32_t j = fb;
                    const uint32_t l = sh.act[b0 + j], u = sh.src[b0 + j], ejj = sh.acte[b0 + j];
                    uint32_t* cj = cnt + j * S;
                    if (lane < j) {   // earlier final picks held by u leave its counts (H says which: no load)
                        const uint32_t ci = sh.spec[lane];
                        if (ci != NONE32 && ((sh.pbits[lane] >> ejj) & 1u)) atomicSub(&cj[ci >> 12], 1u);
                    }
                    __syncwarp();
                    const uint32_t n = warp_sum_counts(cj, S, lane);
                    uint32_t cnew = NONE32;
                    if (n == 0) {
                        if (lane == 0) stcg32(a.empty_epoch + l, step + 1);
                    } else {
                        const uint32_t r = philox_draw((uint32_t)t, (uint32_t)(t >> 32), l, 0u, a.k0, a.k1);
                        bool sem = false;
                        cnew = kth_candidate(cj, S, Q, have4 + (size_t)u * Q, wrow, __umulhi(r, n), sh.claimed, ncl, lane, sem);
                        if (cnew == NONE32) {   // cannot happen; fail loudly instead of corrupting
                            if (lane == 0) atomicOr(&a.ctrl->err, 4u);
                        } else {
                            if (lane == 0) {
                                sh.claimed[ncl] = cnew;
                                const uint64_t te = commit_claim<DYN>(a, v, l, sh.actw[b0 + j], cnew, sem, step, t, false);
                                mymin = min(mymin, te);
                                mymax = max(mymax, te);
                            }
                            repicked |= 1u << ncl;
                            ++ncl;
                            --wc;
                        }
                    }
                    // the new pick's holders among the in-links of v: the next test and its count upkeep
                    bool holds = false;
                    if (cnew != NONE32 && lane < e1)
                        holds = ((ldcg64(a.have + (size_t)dc->src[lane] * a.Wp + (cnew >> 6)) >> (cnew & 63)) & 1ull) != 0ull;
                    const uint32_t hm = __ballot_sync(0xFFFFFFFFu, holds);
                    if (holds) {
                        atomicSub(&a.gcnt[(size_t)dc->link[lane] * S + (cnew >> 12)], 1u);
                        atomicSub(&a.gtot[dc->link[lane]], 1u);
                    }
                    if (lane == 0) {
                        sh.spec[j] = cnew;
                        sh.pbits[j] = hm;
                        if (cnew != NONE32) st.bytes += (unsigned long long)e1 * 32u;
                    }
                    __syncwarp();
                    done = j + 1;
                }
                // the best[] updates of re-picked claims are off the serial chain: one lane per claim
                if (lane < ncl && ((repicked >> lane) & 1u)) commit_best<DYN>(a, v, sh.claimed[lane]);
                trace_stamp(a, step, 10);
                if (lane == 0) sh.wc = wc;
                // another sweep of this destination follows: its loads must see the wants bits just cleared
                if (b0 + NBT < nact || eb + 32 < e1) __threadfence();
            } else if (warp == 0) {
                st.rows += nb + 1;
                st.links += nb;
                uint32_t bad = 0;
                const bool fastpairs = dc != nullptr;   // <= 32 in-links, tables in shared memory
                if (fastpairs) {
                    // one load per (speculative pick i, in-link e of v): does e's source hold pick i?  The answers
                    // serve the conflict test (active later in-links) and the count upkeep (all in-links).
                    if (lane < NBT) sh.pbits[lane] = 0;
                    __syncwarp();
                    const uint32_t npairs = nb * e1;
                    for (uint32_t p0 = 0; p0 < npairs; p0 += 64) {   // two pairs per lane and round, loads first
                        const uint32_t pa = p0 + lane, pb = p0 + 32 + lane;
                        uint32_t ia = 0, ea = 0, ib = 0, eb2 = 0, ca = NONE32, cb = NONE32;
                        unsigned long long wa = 0, wb = 0;
                        if (pa < npairs) { ia = pa / e1; ea = pa - ia * e1; ca = sh.spec[ia]; }
                        if (pb < npairs) { ib = pb / e1; eb2 = pb - ib * e1; cb = sh.spec[ib]; }
                        if (ca != NONE32) wa = ldcg64(a.have + (size_t)dc->src[ea] * a.Wp + (ca >> 6));
                        if (cb != NONE32) wb = ldcg64(a.have + (size_t)dc->src[eb2] * a.Wp + (cb >> 6));
                        if (ca != NONE32 && ((wa >> (ca & 63)) & 1ull)) atomicOr(&sh.pbits[ia], 1u << ea);
                        if (cb != NONE32 && ((wb >> (cb & 63)) & 1ull)) atomicOr(&sh.pbits[ib], 1u << eb2);
                    }
                    __syncwarp();
                    if (lane < nb) {   // lane j: is an earlier pick held by my in-link's source?
                        const uint32_t ej = sh.acte[b0 + lane];
                        for (uint32_t i = 0; i < lane; ++i)
                            if ((sh.pbits[i] >> ej) & 1u) bad |= 1u << lane;
                    }
                    if (lane == 0) st.bytes += (unsigned long long)nb * e1 * 32u;
                } else {
                    for (uint32_t p = lane; p < nb * nb; p += 32) {
                        const uint32_t i = p / nb, j = p % nb;
                        if (i < j) {
                            const uint32_t ci = sh.spec[i];
                            if (ci != NONE32 && cnt[j * S + (ci >> 12)] != 0) {
                                const uint32_t u = sh.src[b0 + j];
                                if ((ldcg64(a.have + (size_t)u * a.Wp + (ci >> 6)) >> (ci & 63)) & 1ull) bad |= 1u << j;
                            }
                        }
                    }
                }
                bad = __reduce_or_sync(0xFFFFFFFFu, bad);
                trace_stamp(a, step, 8);
                const uint32_t first_bad = bad ? (uint32_t)(__ffs(bad) - 1) : nb;
                // commit the picks that stand (one lane per link)
                uint32_t wc = sh.wc;
                {
                    uint32_t c = NONE32, l = 0;
                    if (lane < first_bad) { c = sh.spec[lane]; l = sh.act[b0 + lane]; }
                    const uint32_t cm = __ballot_sync(0xFFFFFFFFu, c != NONE32);
                    if (lane < first_bad) {
                        if (c != NONE32) {
                            const uint64_t te = commit_claim<DYN>(a, v, l, sh.actw[b0 + lane], c, sh.sempty[lane] != 0u, step, t);
                            mymin = min(mymin, te);
                            mymax = max(mymax, te);
                            sh.claimed[__popc(cm & ((1u << lane) - 1u))] = c;
                        } else {
                            stcg32(a.empty_epoch + l, step + 1);
                        }
                    }
                    wc -= __popc(cm);
                }
                uint32_t ncl = __popc(__ballot_sync(0xFFFFFFFFu, lane < first_bad && sh.spec[lane] != NONE32));
                __syncwarp();
                const uint32_t ncl_spec = ncl;
                trace_stamp(a, step, 9);
                if (fastpairs && a.gcnt != nullptr && lane < e1) {
                    // count upkeep for the committed picks: lane e owns in-link e of v
                    const uint32_t l2 = dc->link[lane];
                    uint32_t dec = 0;
                    for (uint32_t i = 0; i < first_bad; ++i) {
                        const uint32_t ci = sh.spec[i];
                        if (ci != NONE32 && ((sh.pbits[i] >> lane) & 1u)) {
                            atomicSub(&a.gcnt[(size_t)l2 * S + (ci >> 12)], 1u);
                            ++dec;
                        }
                    }
                    if (dec) atomicSub(&a.gtot[l2], dec);
                }
                // the rest, one by one, against the wants row net of the claims so far
                for (uint32_t j = first_bad; j < nb && wc > 0; ++j) {
                    if (lane == 0) ++st.slow;
                    const uint32_t l = sh.act[b0 + j];
                    const uint32_t u = sh.src[b0 + j];
                    uint32_t* cj = cnt + j * S;
                    if (lane < ncl) {   // (at most NBT claims: one lane each, one round trip)
                        const uint32_t c = sh.claimed[lane];
                        if ((ldcg64(a.have + (size_t)u * a.Wp + (c >> 6)) >> (c & 63)) & 1ull) atomicSub(&cj[c >> 12], 1u);
                    }
                    __syncwarp();
                    const uint32_t n = warp_sum_counts(cj, S, lane);
                    if (n == 0) {
                        if (lane == 0) stcg32(a.empty_epoch + l, step + 1);
                        continue;
                    }
                    const uint32_t r = philox_draw((uint32_t)t, (uint32_t)(t >> 32), l, 0u, a.k0, a.k1);
                    bool sem = false;
                    const uint32_t c = kth_candidate(cj, S, Q, have4 + (size_t)u * Q, wrow, __umulhi(r, n), sh.claimed, ncl, lane, sem);
                    if (c == NONE32) {   // cannot happen; fail loudly instead of corrupting
                        if (lane == 0) atomicOr(&a.ctrl->err, 4u);
                        continue;
                    }
                    if (lane == 0) {
                        sh.claimed[ncl] = c;
                        const uint64_t te = commit_claim<DYN>(a, v, l, sh.actw[b0 + j], c, sem, step, t, false);
                        mymin = min(mymin, te);
                        mymax = max(mymax, te);
                    }
                    ++ncl;
                    --wc;
                    __syncwarp();
                }
                // (their best[] updates are off the serial chain: one lane per re-picked claim)
                if (lane >= ncl_spec && lane < ncl) commit_best<DYN>(a, v, sh.claimed[lane]);
                trace_stamp(a, step, 10);
                const uint32_t dec0 = fastpairs ? ncl_spec : 0u;   // claims before dec0 were handled above
                if (a.gcnt != nullptr && ncl > dec0) {
                    // v no longer wants the claimed chunks: every in-link of v (free or busy) whose source
                    // holds one loses that candidate
                    __syncwarp();
                    const uint32_t n_in = e1 - e0;
                    for (uint32_t p2 = lane; p2 < (ncl - dec0) * n_in; p2 += 32) {
                        const uint32_t i = dec0 + p2 / n_in, e = e0 + (p2 % n_in);
                        uint32_t l2, u2;
                        if (dc != nullptr) { l2 = dc->link[e]; u2 = dc->src[e]; } else { l2 = a.in_link[e]; u2 = a.esrc[l2]; }
                        const uint32_t c = sh.claimed[i];
                        if ((ldcg64(a.have + (size_t)u2 * a.Wp + (c >> 6)) >> (c & 63)) & 1ull) {
                            atomicSub(&a.gcnt[(size_t)l2 * S + (c >> 12)], 1u);
                            atomicSub(&a.gtot[l2], 1u);
                        }
                    }
                    if (lane == 0) st.bytes += (unsigned long long)(ncl - dec0) * n_in * 32u;
                }
                if (lane == 0) sh.wc = wc;
                // another sweep of this destination follows: its loads must see the wants bits just cleared
                if (b0 + NBT < nact || eb + 32 < e1) __threadfence();
            }
            __syncthreads();
        }
        __syncthreads();
    }
    if (warp == 0) {
        for (int o = 16; o; o >>= 1) {
            mymin = min(mymin, __shfl_xor_sync(0xFFFFFFFFu, mymin, o));
            mymax = max(mymax, __shfl_xor_sync(0xFFFFFFFFu, mymax, o));
        }
        if (lane == 0) {
            if (mymin != T_INF) atomicMin(&a.ctrl->tnext[(step + 1) % 3], (unsigned long long)mymin);
            const uint32_t wc = sh.wc;
            if (wc != wc_start) {
                stcg32(a.wants_cnt + v, wc);
                atomicAdd(&a.ctrl->total, (unsigned long long)(wc_start - wc));
                atomicMax(&a.ctrl->tmax, (unsigned long long)mymax);
            }
        }
    }
    __syncthreads();
}

// DYN: the dynamic relay rule's code (best[], holder lists, the wants-shrink phase) is compiled in; the thin-tree
// instantiation stays lean
template <int NBT, bool DYN>
__global__ void __launch_bounds__(NBT * 32, 1024 / (NBT * 32)) k_loop(const LoopArgs a) {
    constexpr int THREADS = NBT * 32;
    extern __shared__ __align__(16) uint32_t cnt[];   // [NBT][S] candidate counts per segment, then the work list
    uint32_t* list = cnt + ((NBT * a.S + 3u) & ~3u);   // [LIST_CAP] (in-link << 28 | sector)
    __shared__ CtaScratch sh;
    __shared__ DestCache dcache[DEST_CACHE];
    cg::grid_group grid = cg::this_grid();
    for (uint32_t k = threadIdx.x >> 5; k < DEST_CACHE; k += THREADS / 32) {   // warp k fills slot k
        const uint32_t v = blockIdx.x + k * gridDim.x, lane = threadIdx.x & 31;
        if (v < a.N) {
            const uint32_t e0 = a.in_off[v], n = a.in_off[v + 1] - e0;
            if (lane == 0) dcache[k].n_in = (n <= 32) ? n : NONE32;
            if (n <= 32 && lane < n) {
                const uint32_t l = a.in_link[e0 + lane];
                dcache[k].link[lane] = l;
                dcache[k].src[lane] = a.esrc[l];
                dcache[k].w[lane] = a.w[l];
            }
        }
    }
    __syncthreads();
    LoopStats st = {0, 0, 0, 0};
    uint32_t step = 0;
    uint64_t t = 0;
    uint64_t emit_base = 0;
    uint64_t total_now = 0;                 // transfers through event step-1
    __shared__ unsigned long long s_next[2];   // one thread per CTA reads the two hot words after a barrier
    for (;;) {
        trace_stamp(a, step, 0);
        // dynamic rule: the wants-shrink of the event before runs beside this event's arrivals (no barrier between
        // them, see dyn_drop); best[] is final since that event's second barrier
        if (DYN && a.best != nullptr && step > 0) {
            dyn_shrink_wants(a, step - 1, t);
            trace_stamp(a, step, 11);
        }
        loop_phase_links<DYN>(a, step, t, emit_base);
        emit_base = total_now;
        trace_stamp(a, step, 1);
        grid.sync();
        trace_stamp(a, step, 2);
#ifdef PCCL_DEBUG_COUNTS   /* debugging build: the kept counts against a recount of have[src] & wants[dst] */
        if (a.gtot != nullptr) {
            const uint32_t lane = threadIdx.x & 31;
            const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nW = (gridDim.x * blockDim.x) >> 5;
            for (uint32_t l = gw; l < a.L; l += nW) {
                uint32_t n = 0;
                for (uint32_t wi = lane; wi < a.Wp; wi += 32)
                    n += __popcll(ldcg64(a.have + (size_t)a.esrc[l] * a.Wp + wi) & ldcg64(a.wants + (size_t)a.edst[l] * a.Wp + wi));
                n = __reduce_add_sync(0xFFFFFFFFu, n);
                const uint32_t g = ldcg32(a.gtot + l);
                if (lane == 0 && g != n) {
                    printf("[counts] step %u t %llu link %u (%u -> %u): kept %u actual %u\n", step, (unsigned long long)t, l, a.esrc[l], a.edst[l], g, n);
                    for (uint32_t wi = 0; wi < a.Wp; ++wi) {
                        const unsigned long long x = ldcg64(a.have + (size_t)a.esrc[l] * a.Wp + wi) & ldcg64(a.wants + (size_t)a.edst[l] * a.Wp + wi);
                        if (x) printf("[counts]   link %u word %u: %llx\n", l, wi, x);
                    }
                }
            }
            grid.sync();
        }
#endif
        {
            uint32_t k = 0;
            for (uint32_t v = blockIdx.x; v < a.N; v += gridDim.x, ++k)
                match_destination<NBT, DYN>(a, v, step, t, cnt, list, sh, st,
                                  (k < DEST_CACHE && dcache[k].n_in != NONE32) ? &dcache[k] : nullptr);
        }
        trace_stamp(a, step, 6);
        grid.sync();
        trace_stamp(a, step, 7);
        if (threadIdx.x == 0) {
            s_next[0] = ldcg64((const uint64_t*)&a.ctrl->tnext[(step + 1) % 3]);
            s_next[1] = ldcg64((const uint64_t*)&a.ctrl->total);
        }
        __syncthreads();
        t = s_next[0];
        total_now = s_next[1];
        __syncthreads();
        ++step;
        if (t == T_INF) break;
    }
    {   // bytes requested: every lane counted its own sectors
        unsigned long long b = st.bytes;
        for (int o = 16; o; o >>= 1) b += __shfl_xor_sync(0xFFFFFFFFu, b, o);
        if ((threadIdx.x & 31) == 0 && b) atomicAdd(&a.ctrl->bytes_requested, b);
    }
    if (threadIdx.x == 0) {   // warp 0 lane 0 holds this CTA's counters
        if (st.rows) atomicAdd(&a.ctrl->rows_scanned, st.rows);
        if (st.links) atomicAdd(&a.ctrl->links_scanned, st.links);
        if (st.slow) atomicAdd(&a.ctrl->slow_picks, st.slow);
        if (blockIdx.x == 0) a.ctrl->events = step;
    }
}

// ==================================================================================================
//  a9: emitter for reductions -- reverse in direction and time, then sort by (t_start, link).
// ==================================================================================================
// raw record of the transposed broadcast (c, psrc, pdst, l, ts, te)  ->  (c, psrc, pdst, l, T-te, T-ts);
// the loop already reported the PHYSICAL endpoints, which are the reversed transfer's src -> dst.
__global__ void k_reverse_keys(Rec* __restrict__ raw, uint64_t n, uint64_t T, uint32_t link_bits,
                               uint64_t* __restrict__ keys, uint32_t* __restrict__ idx, bool reverse = true) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Rec r = raw[i];
    uint64_t ts = r.t_start;
    if (reverse) {
        ts = T - r.t_end;
        r.t_end = T - r.t_start;
        r.t_start = ts;
        raw[i] = r;
    }
    keys[i] = (ts << link_bits) | r.link;
    idx[i] = (uint32_t)i;
}

__global__ void k_gather_shift(const Rec* __restrict__ raw, const uint32_t* __restrict__ idx, uint64_t n,
                               uint64_t shift, Rec* __restrict__ out) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Rec r = raw[idx[i]];
    r.t_start += shift;
    r.t_end += shift;
    out[i] = r;
}

// ---- stable LSD radix sort, 8 bits per pass, (u64 key, u32 payload) -------------------------------
constexpr int SORT_THREADS = 256;
constexpr int SORT_ITEMS = 8;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;   // 2048 keys per block

__global__ void __launch_bounds__(SORT_THREADS) k_sort_hist(const uint64_t* __restrict__ keys, uint64_t n,
                                                            uint32_t shift, uint32_t* __restrict__ ghist,
                                                            uint32_t nblocks) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint64_t base = (uint64_t)blockIdx.x * SORT_TILE;
    for (int i = 0; i < SORT_ITEMS; ++i) {
        const uint64_t p = base + (uint64_t)i * SORT_THREADS + threadIdx.x;
        if (p < n) atomicAdd(&h[(keys[p] >> shift) & 255u], 1u);
    }
    __syncthreads();
    ghist[(size_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

// exclusive scan of ghist (digit-major), single block
__global__ void __launch_bounds__(1024) k_sort_scan(uint32_t* __restrict__ ghist, uint64_t len) {
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (uint64_t b = 0; b < len; b += 1024) {
        const uint64_t i = b + threadIdx.x;
        const uint32_t x = (i < len) ? ghist[i] : 0u;
        uint32_t incl = warp_incl_scan(x, lane);
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const uint32_t y = wsum[lane];
            const uint32_t yi = warp_incl_scan(y, lane);
            wsum[lane] = yi - y;
        }
        __syncthreads();
        const uint32_t c = carry;
        const uint32_t excl = c + wsum[warp] + incl - x;
        if (i < len) ghist[i] = excl;
        __syncthreads();
        if (threadIdx.x == 1023) carry = excl + x;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(SORT_THREADS) k_sort_scatter(const uint64_t* __restrict__ kin,
                                                               const uint32_t* __restrict__ vin,
                                                               uint64_t* __restrict__ kout,
                                                               uint32_t* __restrict__ vout, uint64_t n,
                                                               uint32_t shift, const uint32_t* __restrict__ ghist,
                                                               uint32_t nblocks) {
    constexpr int NW = SORT_THREADS / 32;
    __shared__ uint32_t wcount[NW][256];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < NW * 256; i += SORT_THREADS) (&wcount[0][0])[i] = 0;
    __syncthreads();
    // warp w owns items [w*256, w*256+256) of the tile, visited in index order
    const uint64_t wbase = (uint64_t)blockIdx.x * SORT_TILE + (uint64_t)warp * (32 * SORT_ITEMS);
    uint64_t key[SORT_ITEMS];
    uint32_t val[SORT_ITEMS], rank[SORT_ITEMS];
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint64_t p = wbase + (uint64_t)r * 32 + lane;
        const bool valid = p < n;
        key[r] = valid ? kin[p] : 0;
        val[r] = valid ? vin[p] : 0;
        const uint32_t vm = __ballot_sync(0xFFFFFFFFu, valid);
        rank[r] = 0;
        if (valid) {
            const uint32_t d = (uint32_t)(key[r] >> shift) & 255u;
            const uint32_t peers = __match_any_sync(vm, d);
            rank[r] = wcount[warp][d] + __popc(peers & ((1u << lane) - 1u));
            __syncwarp(vm);
            if ((int)lane == __ffs(peers) - 1) wcount[warp][d] += __popc(peers);
            __syncwarp(vm);
        }
    }
    __syncthreads();
    {   // per digit: global base of this block, then exclusive prefix over the warps
        const uint32_t d = threadIdx.x;
        uint32_t run = ghist[(size_t)d * nblocks + blockIdx.x];
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const uint32_t c = wcount[w][d];
            wcount[w][d] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint64_t p = wbase + (uint64_t)r * 32 + lane;
        if (p < n) {
            const uint32_t d = (uint32_t)(key[r] >> shift) & 255u;
            const uint32_t pos = wcount[warp][d] + rank[r];
            kout[pos] = key[r];
            vout[pos] = val[r];
        }
    }
}

// ==================================================================================================
//  Translation (section 4.8): the schedule as one program per node.  Every transfer gives
//  two operations: its destination RECEIVES the chunk (completes at t_end) and its source SENDS it (starts
//  at t_start).  A node's program lists its operations by (time, kind: receive before send, link).
// ==================================================================================================
struct Op {   // == pccl_op_t
    uint32_t kind, peer, chunk, link;
    uint64_t time;
};
static_assert(sizeof(Op) == 24, "layout");

// operation i < M: the receive of record i; operation M + i: its send.  keyA orders within a node.
__global__ void k_ops_keys(const Rec* __restrict__ recs, uint64_t M, uint32_t link_bits, uint64_t* __restrict__ keyA,
                           uint32_t* __restrict__ idx) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * M) return;
    const bool send = i >= M;
    const Rec r = recs[send ? i - M : i];
    const uint64_t time = send ? r.t_start : r.t_end;
    keyA[i] = (time << (1 + link_bits)) | ((uint64_t)(send ? 1u : 0u) << link_bits) | r.link;
    idx[i] = (uint32_t)i;
}
// second (stable) pass: the node of every operation, in the order of the first pass
__global__ void k_ops_nodes(const Rec* __restrict__ recs, uint64_t M, const uint32_t* __restrict__ idx,
                            uint64_t* __restrict__ keyB) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * M) return;
    const uint32_t o = idx[i];
    const bool send = o >= M;
    const Rec r = recs[send ? o - M : o];
    keyB[i] = send ? r.src : r.dst;
}
__global__ void k_ops_gather(const Rec* __restrict__ recs, uint64_t M, const uint32_t* __restrict__ idx,
                             Op* __restrict__ ops) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * M) return;
    const uint32_t o = idx[i];
    const bool send = o >= M;
    const Rec r = recs[send ? o - M : o];
    Op op;
    op.kind = send ? 1u : 0u;
    op.peer = send ? r.dst : r.src;
    op.chunk = r.chunk;
    op.link = r.link;
    op.time = send ? r.t_start : r.t_end;
    ops[i] = op;
}
// offsets[v] = first operation of node v in the node-sorted key array (lower bound), offsets[n] = 2M
__global__ void k_ops_offsets(const uint64_t* __restrict__ keyB, uint64_t n_ops, uint32_t n_nodes,
                              uint64_t* __restrict__ offsets) {
    const uint32_t v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v > n_nodes) return;
    uint64_t lo = 0, hi = n_ops;
    while (lo < hi) {
        const uint64_t mid = (lo + hi) >> 1;
        if (keyB[mid] < v) lo = mid + 1; else hi = mid;
    }
    offsets[v] = lo;
}

}  // namespace pccl
