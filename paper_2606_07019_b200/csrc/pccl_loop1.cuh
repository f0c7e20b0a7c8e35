// =========================================================================================
// pccl_loop1.cuh -- the event loop with ONE grid barrier per event (kept counts only).
//
// k_loop (pccl_device.cuh) separates "apply arrivals" from "match" with a barrier.  Here the
// arrivals leave the critical path: a destination CTA does not wait for its in-neighbours'
// arrivals to be stored, it derives them.  Link state is double-buffered by event parity
// (an event reads the buffer the previous event wrote), so at event time t the chunks that
// arrive at a source u right now are exactly  { inflight_i : i in-link of u, free_i == t }
// in the read buffer -- "pending" chunks.  The CTA of destination v
//   * reads the state of its own in-links AND of the in-links of its sources (a two-hop
//     table cached in shared memory),
//   * treats pending chunks as held by the source: they patch the have segment a pick loads,
//     the conflict test and the count upkeep,
//   * is the ONLY writer of the candidate counts of its in-links: +1 when a pending chunk is
//     wanted by v (exactly once, at the event it arrives), -1 when v claims a chunk the
//     source holds,
//   * stores its own arrivals into have[v] for later events (this event's readers patch).
// The emit of event k's records runs at the end of event k+1, after the matching, where it
// hides in the barrier skew.  Same results as k_loop, bit for bit (tests/test_parity_gpu.py).
// Used when every node has at most 8 in-links (<= 64 two-hop links) and rows have at most
// 128 segments; otherwise, and for the recount / dynamic-rule modes, k_loop runs.
// =========================================================================================
#pragma once
#include "pccl_device.cuh"

namespace pccl {

constexpr int HOP_CAP = 64;

struct FastCache {          // static tables of one destination
    uint32_t n_in;          // <= NBT
    uint32_t nhop;          // <= HOP_CAP
    uint32_t link[NB];
    uint32_t src[NB];
    uint64_t w[NB];
    uint32_t hop_off[NB + 1];     // two-hop links of in-link j: hop_link[hop_off[j] .. hop_off[j+1])
    uint32_t hop_link[HOP_CAP];   // the in-links of src[j]
};

struct FastScratch {
    uint64_t free_[NB];        // own in-links, read buffer
    uint32_t inf_[NB];         // their in-flight chunk after this event's arrivals (NONE32 if none)
    uint32_t pend_c[HOP_CAP];  // chunk arriving now over two-hop link h (NONE32 if none)
    uint32_t pend_w[HOP_CAP];  // ... and this destination wants it
    uint32_t spec[NB];         // pick of in-link j (NONE32: inactive or no candidate)
    uint32_t sempty[NB];
    uint32_t pbits[NB];        // pick i: mask over in-links whose source holds it
    uint32_t claimed[NB];
    uint32_t newc[NB];         // committed claim per in-link (NONE32 if none)
    uint64_t newte[NB];
    uint32_t wc;
};

// does source of in-link e hold chunk c at this event (stored bit or pending arrival)?
__device__ __forceinline__ bool holds_now(const LoopArgs& a, const FastCache& fc, const FastScratch& sh, uint32_t e,
                                          uint32_t c) {
    for (uint32_t h = fc.hop_off[e]; h < fc.hop_off[e + 1]; ++h)
        if (sh.pend_c[h] == c) return true;
    return ((ldcg64(a.have + (size_t)fc.src[e] * a.Wp + (c >> 6)) >> (c & 63)) & 1ull) != 0ull;
}

// emit the records of event `ev` (claims are in the state buffer written at that event) in canonical order.
// 32-link tasks; the calling warp is worker `wk` of `nwk` in its CTA.
__device__ __forceinline__ void emit_event(const LoopArgs& a, uint32_t ev, uint64_t emit_base, uint32_t wk, uint32_t nwk) {
    const uint32_t lane = threadIdx.x & 31;
    const uint64_t* mb = a.matchbits + (size_t)(ev % 3) * a.nLw;
    const uint32_t wr = ((ev & 1u) ^ 1u) * a.L;
    for (uint32_t lb = (wk * gridDim.x + blockIdx.x) * 32; lb < a.L; lb += nwk * gridDim.x * 32) {
        const uint32_t l = lb + lane, wq = lb >> 6;
        const uint64_t word = ldcg64(mb + wq);
        const uint32_t mine = (uint32_t)(word >> (lb & 32));
        if (mine == 0) continue;   // warp-uniform
        uint32_t pre = 0;
        for (uint32_t i = lane; i < wq; i += 32) pre += __popcll(ldcg64(mb + i));
        pre = __reduce_add_sync(0xFFFFFFFFu, pre);
        if (lb & 32) pre += __popc((uint32_t)word);
        if ((mine >> lane) & 1u) {
            const uint64_t rank = pre + __popc(mine & ((1u << lane) - 1u));
            if (emit_base + rank >= a.out_cap) { atomicOr(&a.ctrl->err, 32u); continue; }
            const uint32_t c = ldcg32(a.st_inf + wr + l);
            const uint64_t f = ldcg64(a.st_free + wr + l);
            const uint64_t ts = f - a.w[l] + a.t_offset, te = f + a.t_offset;
            uint4* o = reinterpret_cast<uint4*>(a.out + emit_base + rank);
            o[0] = make_uint4(c, a.psrc[l], a.pdst[l], l);
            o[1] = make_uint4((uint32_t)ts, (uint32_t)(ts >> 32), (uint32_t)te, (uint32_t)(te >> 32));
        }
    }
}

// barrier among the NBT warps of one team (named barrier team + 1; barrier 0 is __syncthreads)
template <int NBT, int TEAMS>
__device__ __forceinline__ void team_sync(uint32_t team) {
    static_assert(TEAMS <= 4, "one literal barrier id per team");
    if (TEAMS == 1) { __syncthreads(); return; }
    if (team == 0) asm volatile("bar.sync 1, %0;" ::"r"(NBT * 32) : "memory");
    else if (team == 1) asm volatile("bar.sync 2, %0;" ::"r"(NBT * 32) : "memory");
    else if (team == 2) asm volatile("bar.sync 3, %0;" ::"r"(NBT * 32) : "memory");
    else asm volatile("bar.sync 4, %0;" ::"r"(NBT * 32) : "memory");
}

template <int NBT, int TEAMS>
__device__ __forceinline__ void fast_match(const LoopArgs& a, uint32_t v, uint32_t step, uint64_t t, uint32_t* cnt,
                                           FastScratch& sh, const FastCache& fc, LoopStats& st, bool do_emit,
                                           uint64_t emit_base) {
    const uint32_t team = threadIdx.x / (NBT * 32);
    const uint32_t tid = threadIdx.x % (NBT * 32), lane = tid & 31, warp = tid >> 5;
    const uint32_t Q = a.Wp >> 1, S = a.S, L = a.L;
    const uint32_t rd = (step & 1u) * L, wr = ((step & 1u) ^ 1u) * L;
    const uint32_t n_in = fc.n_in, nhop = fc.nhop;
    const uint4* have4 = reinterpret_cast<const uint4*>(a.have);
    const uint4* wrow = reinterpret_cast<const uint4*>(a.wants) + (size_t)v * Q;

    // ---- all loads of the first round trip, issued before any is consumed --------------------------
    uint64_t f_own = 0, f_hop = 0;
    uint32_t c_own = NONE32, c_hop = NONE32;
    uint32_t rowv[4] = {0, 0, 0, 0};
    const bool is_own = tid < n_in, is_hop = tid >= 32 && tid < 32 + nhop;
    if (is_own) {
        f_own = ldcg64(a.st_free + rd + fc.link[tid]);
        c_own = ldcg32(a.st_inf + rd + fc.link[tid]);
    }
    if (is_hop) {
        const uint32_t hl = fc.hop_link[tid - 32];
        f_hop = ldcg64(a.st_free + rd + hl);
        c_hop = ldcg32(a.st_inf + rd + hl);
    }
    const uint32_t wc0 = ldcg32(a.wants_cnt + v);
    if (warp < n_in) {
        const uint32_t* g = a.gcnt + (size_t)fc.link[warp] * S;
#pragma unroll
        for (int x = 0; x < 4; ++x)
            if (lane + 32u * x < S) rowv[x] = ldcg32(g + lane + 32u * x);
    }
    // the pick's random draw depends only on (t, link): computed while the loads are in flight
    uint32_t r_pre = 0;
    if (warp < n_in) r_pre = philox_draw((uint32_t)t, (uint32_t)(t >> 32), fc.link[warp], 0u, a.k0, a.k1);
    // ---- consume -----------------------------------------------------------------------------------
    if (is_own) {
        const bool arrived = c_own != NONE32 && f_own == t;   // a3: the chunk is at v from now on
        if (arrived) {
            atomicOr((unsigned long long*)&a.have[(size_t)v * a.Wp + (c_own >> 6)], 1ull << (c_own & 63));
            atomicOr((unsigned long long*)&a.hsum[(size_t)v * a.SWp + (c_own >> 14)], 1ull << ((c_own >> 8) & 63));
        }
        sh.free_[tid] = f_own;
        sh.inf_[tid] = (c_own != NONE32 && f_own <= t) ? NONE32 : c_own;
    }
    if (is_hop) {
        const uint32_t h = tid - 32;
        const uint32_t p = (c_hop != NONE32 && f_hop == t) ? c_hop : NONE32;   // arrives at the source right now
        uint32_t wanted = 0;
        if (p != NONE32) wanted = (uint32_t)(ldcg64(a.wants + (size_t)v * a.Wp + (p >> 6)) >> (p & 63)) & 1u;
        sh.pend_c[h] = p;
        sh.pend_w[h] = wanted;
    }
    if (warp < n_in) {
#pragma unroll
        for (int x = 0; x < 4; ++x)
            if (lane + 32u * x < S) cnt[warp * S + lane + 32u * x] = rowv[x];
    }
    if (tid == 0) sh.wc = wc0;
    team_sync<NBT, TEAMS>(team);
    trace_stamp(a, step, 1);

    // ---- per in-link: count upkeep for the pending chunks, then the pick (a5, a6) ---------------------
    if (warp < n_in) {
        const uint32_t j = warp, l = fc.link[j];
        uint32_t* cj = cnt + j * S;
        const uint32_t h0 = fc.hop_off[j], h1 = fc.hop_off[j + 1];
        for (uint32_t h = h0 + lane; h < h1; h += 32) {
            if (sh.pend_w[h]) {   // new candidate of in-link j; this CTA is the only writer of its counts
                const uint32_t p = sh.pend_c[h];
                atomicAdd(&cj[p >> 12], 1u);
                atomicAdd(&a.gcnt[(size_t)l * S + (p >> 12)], 1u);
                atomicAdd(&a.gtot[l], 1u);
            }
        }
        __syncwarp();
        const uint32_t n = warp_sum_counts(cj, S, lane);
        uint32_t c = NONE32;
        bool sem = false;
        if (sh.free_[j] <= t && n != 0u && wc0 != 0u) {
            c = kth_candidate(cj, S, Q, have4 + (size_t)fc.src[j] * Q, wrow, __umulhi(r_pre, n), nullptr, 0, lane, sem,
                              sh.pend_c + h0, h1 - h0);
            if (c == NONE32 && lane == 0) atomicOr(&a.ctrl->err, 4u);   // cannot happen
            if (lane == 0) {
                st.bytes += (unsigned long long)S * 4u + 2u * SEG_U4 * 16u;
                st.links += 1;
                st.rows += 1;
            }
        }
        // which in-links' sources hold the pick (stored or arriving now)?  lane e answers for in-link e; the mask
        // serves the conflict test and the count upkeep
        uint32_t hit = 0;
        if (c != NONE32 && lane < n_in) hit = holds_now(a, fc, sh, lane, c);
        const uint32_t hm = __ballot_sync(0xFFFFFFFFu, hit != 0u);
        if (lane == 0) { sh.spec[j] = c; sh.sempty[j] = sem; sh.newc[j] = NONE32; sh.pbits[j] = hm; }
    }
    team_sync<NBT, TEAMS>(team);
    trace_stamp(a, step, 2);

    // ---- conflict resolve, commit, count upkeep, next state (a7, a8): warp 0 ---------------------------
    if (warp == 0) {
        uint64_t mymin = T_INF, mymax = 0;
        uint32_t anyspec = 0;
        trace_stamp(a, step, 6);
        uint32_t bad = 0;
        if (lane < n_in) {
            anyspec = sh.spec[lane] != NONE32;
            for (uint32_t i = 0; i < lane; ++i)
                if (sh.spec[i] != NONE32 && ((sh.pbits[i] >> lane) & 1u) && sh.spec[lane] != NONE32) bad |= 1u << lane;
        }
        if (__any_sync(0xFFFFFFFFu, anyspec != 0u) && lane == 0) st.rows += 1;   // the wants row of this sweep
        bad = __reduce_or_sync(0xFFFFFFFFu, bad);
        const uint32_t first_bad = bad ? (uint32_t)(__ffs(bad) - 1) : n_in;
        uint32_t wc = wc0;
        // commit the picks that stand
        {
            uint32_t c = NONE32;
            if (lane < first_bad) c = sh.spec[lane];
            const uint32_t cm = __ballot_sync(0xFFFFFFFFu, c != NONE32);
            if (c != NONE32) {
                const uint32_t l = fc.link[lane];
                const uint64_t te = t + fc.w[lane];
                atomicAnd((unsigned long long*)&a.wants[(size_t)v * a.Wp + (c >> 6)], ~(1ull << (c & 63)));
                if (sh.sempty[lane]) atomicAnd((unsigned long long*)&a.wsum[(size_t)v * a.SWp + (c >> 14)], ~(1ull << ((c >> 8) & 63)));
                atomicOr((unsigned long long*)&a.matchbits[(size_t)(step % 3) * a.nLw + (l >> 6)], 1ull << (l & 63));
                sh.newc[lane] = c;
                sh.newte[lane] = te;
                sh.claimed[__popc(cm & ((1u << lane) - 1u))] = c;
            }
            wc -= __popc(cm);
        }
        uint32_t ncl = __popc(__ballot_sync(0xFFFFFFFFu, lane < first_bad && sh.spec[lane] != NONE32));
        __syncwarp();
        trace_stamp(a, step, 7);
        if (lane < n_in) {   // count upkeep for the committed picks: lane e owns in-link e
            const uint32_t l2 = fc.link[lane];
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
        // the rest one by one, against counts and wants net of the claims so far
        for (uint32_t j = first_bad; j < n_in && wc > 0; ++j) {
            if (sh.spec[j] == NONE32) continue;   // inactive, or no candidate even before the earlier claims
            if (lane == 0) ++st.slow;
            const uint32_t l = fc.link[j];
            uint32_t* cj = cnt + j * S;
            if (lane == 0) {
                for (uint32_t i = 0; i < ncl; ++i) {
                    const uint32_t c = sh.claimed[i];
                    if (holds_now(a, fc, sh, j, c)) cj[c >> 12] -= 1;
                }
            }
            __syncwarp();
            const uint32_t n = warp_sum_counts(cj, S, lane);
            if (n == 0) continue;
            const uint32_t r = philox_draw((uint32_t)t, (uint32_t)(t >> 32), l, 0u, a.k0, a.k1);
            bool sem = false;
            const uint32_t c = kth_candidate(cj, S, Q, have4 + (size_t)fc.src[j] * Q, wrow, __umulhi(r, n), sh.claimed, ncl,
                                             lane, sem, sh.pend_c + fc.hop_off[j], fc.hop_off[j + 1] - fc.hop_off[j]);
            if (c == NONE32) {
                if (lane == 0) atomicOr(&a.ctrl->err, 4u);
                continue;
            }
            if (lane == 0) {
                atomicAnd((unsigned long long*)&a.wants[(size_t)v * a.Wp + (c >> 6)], ~(1ull << (c & 63)));
                if (sem) atomicAnd((unsigned long long*)&a.wsum[(size_t)v * a.SWp + (c >> 14)], ~(1ull << ((c >> 8) & 63)));
                atomicOr((unsigned long long*)&a.matchbits[(size_t)(step % 3) * a.nLw + (l >> 6)], 1ull << (l & 63));
                sh.newc[j] = c;
                sh.newte[j] = t + fc.w[j];
                sh.claimed[ncl] = c;
            }
            if (lane < n_in && holds_now(a, fc, sh, lane, c)) {   // v stops wanting c: its in-links lose the candidate
                atomicSub(&a.gcnt[(size_t)fc.link[lane] * S + (c >> 12)], 1u);
                atomicSub(&a.gtot[fc.link[lane]], 1u);
            }
            ++ncl;
            --wc;
            __syncwarp();
        }
        __syncwarp();
        trace_stamp(a, step, 8);
        // next state of every own in-link (the buffer the next event reads)
        if (lane < n_in) {
            const uint32_t l = fc.link[lane];
            uint64_t nf = sh.free_[lane];
            uint32_t ni = sh.inf_[lane];
            if (sh.newc[lane] != NONE32) { nf = sh.newte[lane]; ni = sh.newc[lane]; mymax = nf; }
            stcg64(a.st_free + wr + l, nf);
            stcg32(a.st_inf + wr + l, ni);
            if (nf > t) mymin = nf;
        }
        for (int o = 16; o; o >>= 1) {
            mymin = min(mymin, __shfl_xor_sync(0xFFFFFFFFu, mymin, o));
            mymax = max(mymax, __shfl_xor_sync(0xFFFFFFFFu, mymax, o));
        }
        if (lane == 0) {
            if (mymin != T_INF) atomicMin(&a.ctrl->tnext[(step + 1) % 3], (unsigned long long)mymin);
            if (wc != wc0) {
                stcg32(a.wants_cnt + v, wc);
                atomicAdd(&a.ctrl->total, (unsigned long long)(wc0 - wc));
                atomicMax(&a.ctrl->tmax, (unsigned long long)mymax);
            }
        }
        trace_stamp(a, step, 9);
    } else if (do_emit) {
        // the other warps are idle now: they emit the previous event's records (a8), which only needs that
        // event's finished bitmap and state buffer
        emit_event(a, step - 1, emit_base, team * (NBT - 1) + warp - 1, TEAMS * (NBT - 1));
    }
    team_sync<NBT, TEAMS>(team);
}

template <int NBT, int TEAMS>
__global__ void __launch_bounds__(NBT * 32 * TEAMS, 1024 / (NBT * 32 * TEAMS)) k_loop1(const LoopArgs a) {
    constexpr int THREADS = NBT * 32 * TEAMS;   // TEAMS teams of NBT warps, each serving its own destinations
    extern __shared__ __align__(16) uint32_t cnt_all[];   // [TEAMS][NBT][S]
    __shared__ FastScratch sh_all[TEAMS];
    __shared__ FastCache fc_all[TEAMS][DEST_CACHE];
    const uint32_t team = threadIdx.x / (NBT * 32), ttid = threadIdx.x % (NBT * 32);
    const uint32_t nslots = gridDim.x * TEAMS, slot = team * gridDim.x + blockIdx.x;   // team-major: CTAs stay balanced
    uint32_t* cnt = cnt_all + team * ((NBT * a.S + 3u) & ~3u);
    FastScratch& sh = sh_all[team];
    FastCache* fc = fc_all[team];
    __shared__ unsigned long long s_next[2];
    cg::grid_group grid = cg::this_grid();
    if (ttid < DEST_CACHE) {   // one thread builds the tables of one destination (once)
        const uint32_t k = ttid, v = slot + k * nslots;
        FastCache& c = fc[k];
        c.n_in = 0; c.nhop = 0; c.hop_off[0] = 0;
        if (v < a.N) {
            const uint32_t e0 = a.in_off[v], n = a.in_off[v + 1] - e0;
            c.n_in = n;
            uint32_t nh = 0;
            for (uint32_t j = 0; j < n; ++j) {
                const uint32_t l = a.in_link[e0 + j], u = a.esrc[l];
                c.link[j] = l; c.src[j] = u; c.w[j] = a.w[l];
                for (uint32_t e = a.in_off[u]; e < a.in_off[u + 1] && nh < HOP_CAP; ++e) c.hop_link[nh++] = a.in_link[e];
                c.hop_off[j + 1] = nh;
            }
            c.nhop = nh;
        }
    }
    __syncthreads();
    LoopStats st = {0, 0, 0, 0};
    uint32_t step = 0;
    uint64_t t = 0, tot_prev = 0, tot_cur = 0;
    for (;;) {
        trace_stamp(a, step, 0);
        {
            uint32_t k = 0;
            for (uint32_t v = slot; v < a.N && k < DEST_CACHE; v += nslots, ++k)
                fast_match<NBT, TEAMS>(a, v, step, t, cnt, sh, fc[k], st, k == 0 && step > 0, tot_prev);
            // (a team without a destination still takes its share of the emit)
            if (k == 0 && step > 0 && (ttid >> 5) != 0)
                emit_event(a, step - 1, tot_prev, team * (NBT - 1) + (ttid >> 5) - 1, TEAMS * (NBT - 1));
        }
        trace_stamp(a, step, 3);
        {   // clear the bitmap the next event writes; re-arm the ring slot after next
            uint64_t* mbn = a.matchbits + (size_t)((step + 1) % 3) * a.nLw;
            for (uint32_t i = blockIdx.x * THREADS + threadIdx.x; i < a.nLw; i += gridDim.x * THREADS) stcg64(mbn + i, 0);
            if (blockIdx.x == 0 && threadIdx.x == 0) stcg64((uint64_t*)&a.ctrl->tnext[(step + 2) % 3], T_INF);
        }
        trace_stamp(a, step, 4);
        grid.sync();
        trace_stamp(a, step, 5);
        if (threadIdx.x == 0) {
            s_next[0] = ldcg64((const uint64_t*)&a.ctrl->tnext[(step + 1) % 3]);
            s_next[1] = ldcg64((const uint64_t*)&a.ctrl->total);
        }
        __syncthreads();
        t = s_next[0];
        tot_prev = tot_cur;
        tot_cur = s_next[1];
        // the records of event step-1 were emitted before the barrier above: [0, tot_prev) is final, tell the host
        // (the host DMA-reads other CTAs' records on this signal: order them at system scope first)
        if (a.progress != nullptr && blockIdx.x == 0 && threadIdx.x == 0) {
            __threadfence_system();
            *(volatile unsigned long long*)a.progress = tot_prev;
        }
        __syncthreads();
        ++step;
        if (t == T_INF) break;
    }
    {
        unsigned long long b = st.bytes;
        for (int o = 16; o; o >>= 1) b += __shfl_xor_sync(0xFFFFFFFFu, b, o);
        if ((threadIdx.x & 31) == 0 && b) atomicAdd(&a.ctrl->bytes_requested, b);
        unsigned long long r = st.rows, ln = st.links, sl = st.slow;
        for (int o = 16; o; o >>= 1) {
            r += __shfl_xor_sync(0xFFFFFFFFu, r, o);
            ln += __shfl_xor_sync(0xFFFFFFFFu, ln, o);
            sl += __shfl_xor_sync(0xFFFFFFFFu, sl, o);
        }
        if ((threadIdx.x & 31) == 0) {
            if (r) atomicAdd(&a.ctrl->rows_scanned, r);
            if (ln) atomicAdd(&a.ctrl->links_scanned, ln);
            if (sl) atomicAdd(&a.ctrl->slow_picks, sl);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) a.ctrl->events = step;
}

}  // namespace pccl
