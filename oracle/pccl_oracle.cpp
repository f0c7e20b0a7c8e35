// =====================================================================================
//  oracle/pccl_oracle.cpp  --  TEST INFRASTRUCTURE ONLY.  NOT PART OF THE PRODUCT PATH.
//
//  A plain, slow, single-threaded CPU statement of the greedy link-chunk matching
//  synthesizer, written from /root/reference/PAPER.md and the readings listed in
//  DESIGN.md (section "Readings of the paper", Q1..Q17).  It shares no code with the CUDA
//  path under paper_2606_07019_b200/csrc (no headers, no helpers, no tables), and nothing
//  in the product imports, links or executes it.  Only tests/, __graft_entry__.smoke()
//  and bench.py's cpu_baseline / --impl reference legs may call it.
//
//  Representation: per-node holdings and wants are sorted std::vector<uint32_t> chunk-id
//  lists; the candidate set of a link is std::set_intersection of two such lists.  There
//  is no blocking, no bitmap, no fusion: each lettered step below is the step of the same
//  letter in DESIGN.md "The procedure (steps R, A..F)".
//
//  What the paper fixes (and where):
//    conditions (chunk: src -> dests) ............ PAPER.md:168-172  (section 4.1)
//    a TEN link carries one chunk ................ PAPER.md:308      (section 4.4)
//    alpha-beta link time  alpha + m*beta ........ PAPER.md:334      (section 4.6)
//    forward only after arrival .................. PAPER.md:338      (section 4.6)
//    a used link is busy for its whole interval .. PAPER.md:340      (section 4.6, Fig. 10)
//    non-group NPUs are intermediates only ....... PAPER.md:298-300, :320
//    Reduce = reversed Broadcast, RS = reversed AG, AR = RS then AG .. PAPER.md:324-330
//    c.dist = shortest path, used for ordering ... PAPER.md:276, :310 (Alg. 3)
//  What the paper does not fix (tie-break, conflict order, relay rule, rounding) follows
//  the readings in DESIGN.md; the pick rule (step E2) is "parity unpinned" by the paper:
//  it is pinned only by the Philox known-answer vectors, by brute-force enumeration of
//  the k-th candidate in tests, and by the closed forms / invariants that any valid pick
//  must satisfy.
//
//  synth_copy_bfs (relay mode 2) is the paper's OWN synthesizer (Alg. 1-3 + section 4.6), kept
//  beside the matching procedure: readings Q19-Q22; the paper prints no values for its worked
//  example (Fig. 6/7 are images), so it is "parity unpinned" by the paper and pinned by a
//  literal boolean-TEN brute force, a hand-worked example and closed forms in
//  tests/test_oracle_bfs.py.
// =====================================================================================
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <functional>
#include <limits>
#include <map>
#include <queue>
#include <set>
#include <utility>
#include <vector>

namespace {

constexpr uint64_t INF = std::numeric_limits<uint64_t>::max();
constexpr uint32_t NONE = 0xFFFFFFFFu;

enum {
    OR_OK = 0,
    OR_ERR_INVALID = -1,
    OR_ERR_UNSUPPORTED = -2,
    OR_ERR_UNREACHABLE = -3,
    OR_ERR_INTERNAL = -6
};

struct Link { uint32_t src, dst; uint64_t alpha_ps, bytes_per_ps; };
struct Pair { uint32_t npu, chunk; };
struct Rec  { uint32_t chunk, src, dst, link; uint64_t t_start_ps, t_end_ps; };
struct Cond { uint32_t src; std::vector<uint32_t> dests; bool present = false; };

// -------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2,
// 3", SC'11).  10 rounds; multipliers 0xD2511F53 (on ctr[0]) and 0xCD9E8D57 (on ctr[2]);
// Weyl key bumps 0x9E3779B9 / 0xBB67AE85.  Pinned by the published known-answer vectors
// in tests/golden/philox_kat.txt.
// -------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// first output word of Philox with key = (seed mod 2^32, seed >> 32)
uint32_t draw(uint64_t seed, uint32_t a, uint32_t b, uint32_t c, uint32_t tag) {
    const uint32_t ctr[4] = {a, b, c, tag};
    const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
    uint32_t out[4];
    philox4x32_10(ctr, key, out);
    return out[0];
}

// uniform index in [0, n) from a 32-bit draw:  (r * n) >> 32   (reading Q5)
uint32_t scale(uint32_t r, uint64_t n) { return (uint32_t)(((uint64_t)r * n) >> 32); }

// -------------------------------------------------------------------------------------
// Step A.  alpha-beta link cost: alpha + m*beta with beta = 1/bandwidth.
// Reading Q7: integer ceiling of m / bytes_per_ps, alpha added after.
// -------------------------------------------------------------------------------------
uint64_t link_cost(const Link& l, uint64_t chunk_bytes) {
    return l.alpha_ps + (chunk_bytes + l.bytes_per_ps - 1) / l.bytes_per_ps;
}

// -------------------------------------------------------------------------------------
// Step B.  ShortestPath(c.src, .) of Alg. 3, metric = alpha-beta cost
// (reading Q3).  Textbook Dijkstra; only the distance values are used.
// -------------------------------------------------------------------------------------
std::vector<uint64_t> dijkstra(uint32_t n, const std::vector<Link>& links,
                               const std::vector<uint64_t>& w, uint32_t s) {
    std::vector<std::vector<uint32_t>> out(n);
    for (uint32_t l = 0; l < links.size(); ++l) out[links[l].src].push_back(l);
    std::vector<uint64_t> D(n, INF);
    using QE = std::pair<uint64_t, uint32_t>;
    std::priority_queue<QE, std::vector<QE>, std::greater<QE>> pq;
    D[s] = 0;
    pq.push({0, s});
    while (!pq.empty()) {
        auto [d, u] = pq.top();
        pq.pop();
        if (d != D[u]) continue;
        for (uint32_t l : out[u]) {
            const uint32_t v = links[l].dst;
            if (d + w[l] < D[v]) { D[v] = d + w[l]; pq.push({D[v], v}); }
        }
    }
    return D;
}

struct CopyResult {
    std::vector<Rec> recs;   // canonical order: (t_start, link id)
    uint64_t T = 0;          // max t_end, 0 if empty
    uint64_t events = 0;     // number of event times processed (including t = 0)
    uint64_t wants_total = 0;// popcount(wants) after step C
};

// sorted-vector set helpers
bool contains(const std::vector<uint32_t>& v, uint32_t x) {
    return std::binary_search(v.begin(), v.end(), x);
}
void insert_sorted(std::vector<uint32_t>& v, uint32_t x) {
    auto it = std::lower_bound(v.begin(), v.end(), x);
    if (it == v.end() || *it != x) v.insert(it, x);
}
void erase_sorted(std::vector<uint32_t>& v, uint32_t x) {
    auto it = std::lower_bound(v.begin(), v.end(), x);
    if (it != v.end() && *it == x) v.erase(it);
}

// -------------------------------------------------------------------------------------
// synth_copy: steps A..F for non-reduction conditions (one source per chunk).
// conds[c] is the condition of chunk c; chunks with !present or no dests need nothing.
// -------------------------------------------------------------------------------------
// pick_dist (reading Q27): Alg. 3 routes the conditions with the largest c.dist first
// ("assigning paths to chunks that must traverse the network for the longest duration first").  As a
// pick policy of the matching loop: a link takes, among its candidates, one of those with the LARGEST c.dist =
// max over dests of ShortestPath(c.src, dest) (Alg. 3 lines 1-6, alpha-beta cost, reading Q3); ties by the same seeded
// draw as the default policy -- the k-th of the tied candidates in ascending chunk id, k = (Philox(t, link) * |tied|) >> 32.
int synth_copy(uint32_t n, const std::vector<Link>& links, const std::vector<Cond>& conds,
               uint64_t chunk_bytes, uint64_t seed, CopyResult& res,
               std::vector<std::vector<uint32_t>>* wants_out = nullptr, bool pick_dist = false) {
    const uint32_t L = (uint32_t)links.size();
    const uint32_t C = (uint32_t)conds.size();

    // A. cost
    std::vector<uint64_t> w(L);
    for (uint32_t l = 0; l < L; ++l) w[l] = link_cost(links[l], chunk_bytes);

    // in-links of every node in ascending link id
    std::vector<std::vector<uint32_t>> inl(n);
    for (uint32_t l = 0; l < L; ++l) inl[links[l].dst].push_back(l);

    // B. distances from every distinct source
    std::vector<std::vector<uint64_t>> D(n);
    for (uint32_t c = 0; c < C; ++c) {
        if (!conds[c].present || conds[c].dests.empty()) continue;
        const uint32_t s = conds[c].src;
        if (D[s].empty()) D[s] = dijkstra(n, links, w, s);
        for (uint32_t d : conds[c].dests)
            if (D[s][d] == INF) return OR_ERR_UNREACHABLE;
    }

    // C. wants = thin relay tree per chunk (reading Q4), have = the source
    std::vector<std::vector<uint32_t>> have(n), wants(n);
    for (uint32_t c = 0; c < C; ++c) {
        if (!conds[c].present) continue;
        const uint32_t s = conds[c].src;
        insert_sorted(have[s], c);
        if (conds[c].dests.empty()) continue;
        const std::vector<uint64_t>& Ds = D[s];
        std::set<uint32_t> marked;
        for (uint32_t d : conds[c].dests) {
            uint32_t cur = d;
            while (cur != s && !marked.count(cur)) {
                marked.insert(cur);
                std::vector<uint32_t> tight;
                for (uint32_t l : inl[cur]) {
                    const uint32_t u = links[l].src;
                    if (Ds[u] != INF && Ds[u] + w[l] == Ds[cur]) tight.push_back(l);
                }
                if (tight.empty()) return OR_ERR_INTERNAL;
                const uint32_t j = scale(draw(seed, c, cur, 0, 1), tight.size());
                cur = links[tight[j]].src;
            }
        }
        for (uint32_t v : marked) insert_sorted(wants[v], c);
    }
    res.wants_total = 0;
    for (uint32_t v = 0; v < n; ++v) res.wants_total += wants[v].size();
    if (wants_out) *wants_out = wants;
    std::vector<uint64_t> cdist(C, 0);                       // Alg. 3 lines 1-6
    if (pick_dist)
        for (uint32_t c = 0; c < C; ++c)
            if (conds[c].present)
                for (uint32_t d : conds[c].dests) cdist[c] = std::max(cdist[c], D[conds[c].src][d]);

    // D. init
    std::vector<uint64_t> free_t(L, 0);
    std::vector<uint32_t> inflight(L, NONE);
    uint64_t t = 0;
    res.recs.clear();
    res.events = 0;

    // E. loop over event times
    std::vector<uint32_t> cand;
    for (;;) {
        ++res.events;
        // E1. arrivals: a chunk that arrives at t may be forwarded at t
        for (uint32_t l = 0; l < L; ++l) {
            if (inflight[l] != NONE && free_t[l] == t) {
                insert_sorted(have[links[l].dst], inflight[l]);
                inflight[l] = NONE;
            }
        }
        // E2. match: destinations are independent; in-links of one destination are taken
        //     in ascending link id, each seeing the claims of the earlier ones (reading Q6)
        for (uint32_t v = 0; v < n; ++v) {
            for (uint32_t l : inl[v]) {
                if (free_t[l] > t) continue;           // link busy
                if (wants[v].empty()) continue;
                const std::vector<uint32_t>& hs = have[links[l].src];
                cand.clear();
                std::set_intersection(hs.begin(), hs.end(), wants[v].begin(), wants[v].end(),
                                      std::back_inserter(cand));
                if (cand.empty()) continue;            // link stays free
                if (pick_dist) {                       // keep the candidates with the largest c.dist (ascending chunk id)
                    uint64_t far = 0;
                    for (uint32_t c : cand) far = std::max(far, cdist[c]);
                    std::vector<uint32_t> tied;
                    for (uint32_t c : cand) if (cdist[c] == far) tied.push_back(c);
                    cand.swap(tied);
                }
                const uint32_t r = draw(seed, (uint32_t)(t & 0xFFFFFFFFull),
                                        (uint32_t)(t >> 32), l, 0);
                const uint32_t k = scale(r, cand.size());
                const uint32_t c = cand[k];            // k-th smallest chunk id
                erase_sorted(wants[v], c);
                inflight[l] = c;
                free_t[l] = t + w[l];
                res.recs.push_back(Rec{c, links[l].src, v, l, t, t + w[l]});
            }
        }
        // E3. advance to the next event time
        uint64_t tn = INF;
        for (uint32_t l = 0; l < L; ++l)
            if (free_t[l] > t && free_t[l] < tn) tn = free_t[l];
        if (tn == INF) break;
        t = tn;
    }

    // F. finish
    for (uint32_t v = 0; v < n; ++v)
        if (!wants[v].empty()) return OR_ERR_INTERNAL;
    for (uint32_t c = 0; c < C; ++c) {
        if (!conds[c].present) continue;
        for (uint32_t d : conds[c].dests)
            if (!contains(have[d], c)) return OR_ERR_INTERNAL;
    }
    std::sort(res.recs.begin(), res.recs.end(), [](const Rec& a, const Rec& b) {
        if (a.t_start_ps != b.t_start_ps) return a.t_start_ps < b.t_start_ps;
        return a.link < b.link;
    });
    res.T = 0;
    for (const Rec& r : res.recs) res.T = std::max(res.T, r.t_end_ps);
    return OR_OK;
}

// -------------------------------------------------------------------------------------
// synth_copy_dynamic: the same loop with the DYNAMIC relay rule (reading Q18, the
// forward-only analogue of the paper's "search the whole network, keep the useful paths",
// PAPER.md:294-300).  Instead of fixing one relay tree per chunk up front:
//   best[c][d]  = the smallest distance to dest d over the source and every node that has
//                 CLAIMED chunk c so far (0 once d itself has claimed it),
//   v wants c  <=>  for some dest d of c:  dist(v -> d) < best[c][d]      (strictly closer),
// and best / wants are updated at the END of each event from that event's claims, so that
// destinations stay independent within an event.  dist(v -> d) is the alpha-beta shortest
// path cost (reading Q3).  Everything else (arrivals, candidates, pick, conflict order,
// free-time advance) is step E of synth_copy unchanged.  A node claims a chunk at most once
// (after its claim it is no longer strictly closer than the best holder), several nodes
// may claim the same chunk, and some deliveries end up unused ("dead ends").
// -------------------------------------------------------------------------------------
int synth_copy_dynamic(uint32_t n, const std::vector<Link>& links, const std::vector<Cond>& conds,
                       uint64_t chunk_bytes, uint64_t seed, CopyResult& res,
                       std::vector<std::vector<uint32_t>>* wants_out = nullptr) {
    const uint32_t L = (uint32_t)links.size();
    const uint32_t C = (uint32_t)conds.size();
    std::vector<uint64_t> w(L);
    for (uint32_t l = 0; l < L; ++l) w[l] = link_cost(links[l], chunk_bytes);
    std::vector<std::vector<uint32_t>> inl(n);
    for (uint32_t l = 0; l < L; ++l) inl[links[l].dst].push_back(l);

    // distances TO every distinct dest: Dijkstra from d on the reversed links
    std::vector<Link> rev(links);
    for (Link& l : rev) std::swap(l.src, l.dst);
    std::vector<std::vector<uint64_t>> Dto(n);
    for (uint32_t c = 0; c < C; ++c) {
        if (!conds[c].present) continue;
        for (uint32_t d : conds[c].dests) {
            if (Dto[d].empty()) Dto[d] = dijkstra(n, rev, w, d);
            if (Dto[d][conds[c].src] == INF) return OR_ERR_UNREACHABLE;
        }
    }
    // best[c][i] for the i-th dest of c, and the wants relation it implies
    std::vector<std::vector<uint64_t>> best(C);
    std::vector<std::vector<uint32_t>> have(n), wants(n);
    auto wanted_by = [&](uint32_t c, uint32_t v) {
        for (size_t i = 0; i < conds[c].dests.size(); ++i)
            if (Dto[conds[c].dests[i]][v] < best[c][i]) return true;
        return false;
    };
    for (uint32_t c = 0; c < C; ++c) {
        if (!conds[c].present) continue;
        insert_sorted(have[conds[c].src], c);
        for (uint32_t d : conds[c].dests) best[c].push_back(Dto[d][conds[c].src]);
        for (uint32_t v = 0; v < n; ++v)
            if (wanted_by(c, v)) wants[v].push_back(c);   // c ascending: the lists stay sorted
    }
    res.wants_total = 0;
    for (uint32_t v = 0; v < n; ++v) res.wants_total += wants[v].size();
    if (wants_out) *wants_out = wants;

    std::vector<uint64_t> free_t(L, 0);
    std::vector<uint32_t> inflight(L, NONE);
    uint64_t t = 0;
    res.recs.clear();
    res.events = 0;
    std::vector<uint32_t> cand;
    for (;;) {
        ++res.events;
        for (uint32_t l = 0; l < L; ++l) {   // E1 arrivals
            if (inflight[l] != NONE && free_t[l] == t) {
                insert_sorted(have[links[l].dst], inflight[l]);
                inflight[l] = NONE;
            }
        }
        const size_t first_new = res.recs.size();
        for (uint32_t v = 0; v < n; ++v) {   // E2 match (identical to synth_copy)
            for (uint32_t l : inl[v]) {
                if (free_t[l] > t) continue;
                if (wants[v].empty()) continue;
                const std::vector<uint32_t>& hs = have[links[l].src];
                cand.clear();
                std::set_intersection(hs.begin(), hs.end(), wants[v].begin(), wants[v].end(),
                                      std::back_inserter(cand));
                if (cand.empty()) continue;
                const uint32_t r = draw(seed, (uint32_t)(t & 0xFFFFFFFFull), (uint32_t)(t >> 32), l, 0);
                const uint32_t c = cand[scale(r, cand.size())];
                erase_sorted(wants[v], c);
                inflight[l] = c;
                free_t[l] = t + w[l];
                res.recs.push_back(Rec{c, links[l].src, v, l, t, t + w[l]});
            }
        }
        // E2' end of the event: the claims tighten best, and every node that is no longer
        // strictly closer to some dest than the best holder stops wanting the chunk
        std::set<uint32_t> touched;
        for (size_t i = first_new; i < res.recs.size(); ++i) {
            const Rec& r = res.recs[i];
            for (size_t k = 0; k < conds[r.chunk].dests.size(); ++k)
                best[r.chunk][k] = std::min(best[r.chunk][k], Dto[conds[r.chunk].dests[k]][r.dst]);
            touched.insert(r.chunk);
        }
        for (uint32_t c : touched)
            for (uint32_t v = 0; v < n; ++v)
                if (contains(wants[v], c) && !wanted_by(c, v)) erase_sorted(wants[v], c);
        uint64_t tn = INF;   // E3
        for (uint32_t l = 0; l < L; ++l)
            if (free_t[l] > t && free_t[l] < tn) tn = free_t[l];
        if (tn == INF) break;
        t = tn;
    }
    for (uint32_t v = 0; v < n; ++v)
        if (!wants[v].empty()) return OR_ERR_INTERNAL;
    for (uint32_t c = 0; c < C; ++c) {
        if (!conds[c].present) continue;
        for (uint32_t d : conds[c].dests)
            if (!contains(have[d], c)) return OR_ERR_INTERNAL;
    }
    std::sort(res.recs.begin(), res.recs.end(), [](const Rec& a, const Rec& b) {
        if (a.t_start_ps != b.t_start_ps) return a.t_start_ps < b.t_start_ps;
        return a.link < b.link;
    });
    res.T = 0;
    for (const Rec& r : res.recs) res.T = std::max(res.T, r.t_end_ps);
    return OR_OK;
}

// -------------------------------------------------------------------------------------
// synth_copy_bfs: the PAPER'S OWN synthesizer, Algorithms 1-3 with the heterogeneous rules of
// section 4.6, condition by condition (readings Q19-Q22).
//
//   Alg. 3 lines 1-7  c.dist = max over dests of ShortestPath(c.src, dest) on the idle network
//                     (alpha-beta cost, reading Q3); conditions in DESCENDING c.dist.  Ties
//                     (paper silent, Q19): ascending Philox(seed; chunk, tag 2) draw, then chunk id.
//   Alg. 3 line 10    BFS(TEN, c): earliest-arrival search from c.src over the WHOLE network
//                     (PAPER.md:300).  Section 4.6 "Chunk Arrival Time": visited carries the time
//                     the chunk reaches each device, a device forwards only after that time.
//                     A link l = (u -> v) of cost w(l) may start at the earliest s >= arrival(u)
//                     such that [s, s + w(l)) overlaps no interval already taken on l
//                     (NextAvailableTime of Alg. 1 applied per link + Fig. 10);
//                     the chunk then reaches v at s + w(l).  arrival(v) is the minimum over v's
//                     in-links; devices are visited in order of arrival (the BFS of Alg. 2 visits
//                     them timestep by timestep).  Which of several links reaching v at the same
//                     earliest time is kept is not fixed by Alg. 2 (iteration order of a set):
//                     reading Q20 keeps the LOWEST LINK ID.
//   PAPER.md:298      filter: keep only the transfers on the recorded paths src -> dest.
//   Alg. 3 line 13    "Remove p from TEN": every kept transfer's interval [s, s + w) becomes busy
//                     on its link for all later conditions.
// A later condition may use a gap in front of an earlier one's interval if its transfer fits.
// -------------------------------------------------------------------------------------
struct BusyLink {                                         // disjoint intervals, ascending
    std::vector<std::pair<uint64_t, uint64_t>> iv;        // [start, end)
};

// earliest s >= a with [s, s + w) free on the link
uint64_t earliest_start(const BusyLink& b, uint64_t a, uint64_t w) {
    uint64_t s = a;
    // intervals are disjoint and ascending, so their ends ascend too: skip those ending at or before s
    auto it = std::upper_bound(b.iv.begin(), b.iv.end(), s,
                               [](uint64_t x, const std::pair<uint64_t, uint64_t>& p) { return x < p.second; });
    for (; it != b.iv.end(); ++it) {
        if (s + w <= it->first) break;   // fits in front of this interval (and of all later ones)
        s = it->second;                  // overlaps it: next try right behind it
    }
    return s;
}

void occupy(BusyLink& b, uint64_t s, uint64_t e) {
    auto it = std::lower_bound(b.iv.begin(), b.iv.end(), std::make_pair(s, e));
    b.iv.insert(it, std::make_pair(s, e));
}

// -------------------------------------------------------------------------------------
// Section 4.7 "Modeling Switches", readings Q23-Q25 of DESIGN.md.  Optional per-node
// parameters of the BFS mode:
//   buffer limit   "We track the number of chunks buffered at each switch node, and the BFS pathfinding
//                  algorithm skips visiting a TEN node at a given timestep if the switch node exceeds the
//                  provided buffer size."  A chunk is buffered at a node it is forwarded from, from its
//                  arrival there until the end of the last transfer that forwards it (store and forward,
//                  PAPER.md:338) -- a half-open stay [arrival, release).  Visiting node v at time t (the
//                  arrival of a transfer) is skipped while the stays of the conditions routed BEFORE hold
//                  limit(v) chunks or more at t; the link then starts at the earliest later time whose
//                  arrival finds a free buffer (and a free link interval).  The test is made at the visit
//                  time only, as the paper states it.
//   no multicast   "if the switch node does not support multicast, the BFS algorithm visits only one next
//                  neighbor ... visits next nodes one by one": such a node forwards over its out-links one
//                  after the other, in ascending link id, the next transfer starting no earlier than the end
//                  of the one before -- whether or not the visit is kept by the path filter afterwards.
// -------------------------------------------------------------------------------------
struct SwitchBuf {                                        // stays of the conditions routed so far
    std::vector<uint64_t> arr, rel;                       // sorted arrival / release times
    uint64_t occ(uint64_t t) const {                      // chunks buffered at time t: arrived by t, not released by t
        return (uint64_t)(std::upper_bound(arr.begin(), arr.end(), t) - arr.begin()) -
               (uint64_t)(std::upper_bound(rel.begin(), rel.end(), t) - rel.begin());
    }
    uint64_t next_free(uint64_t t, uint64_t limit) const { // earliest time >= t with fewer than `limit` chunks buffered
        while (occ(t) >= limit) t = *std::upper_bound(rel.begin(), rel.end(), t);   // occ > 0: a release after t exists
        return t;
    }
    void add(uint64_t a, uint64_t r) {
        arr.insert(std::upper_bound(arr.begin(), arr.end(), a), a);
        rel.insert(std::upper_bound(rel.begin(), rel.end(), r), r);
    }
};

// earliest s >= a with [s, s + w) free on the link AND a free buffer at the far node at the arrival s + w
uint64_t earliest_start_buffered(const BusyLink& b, uint64_t a, uint64_t w, const SwitchBuf* sb, uint64_t limit) {
    for (;;) {
        const uint64_t s = earliest_start(b, a, w);
        if (!sb || sb->occ(s + w) < limit) return s;
        a = sb->next_free(s + w, limit) - w;              // (> s: the buffer frees after s + w)
    }
}

int synth_copy_bfs(uint32_t n, const std::vector<Link>& links, const std::vector<Cond>& conds,
                   uint64_t chunk_bytes, uint64_t seed, CopyResult& res,
                   const uint32_t* buf_limit = nullptr, const uint8_t* no_mcast = nullptr,
                   const std::vector<BusyLink>* busy0 = nullptr, const std::vector<uint64_t>* ready = nullptr) {
    // busy0 / ready (pipelined All-Reduce, Q26): intervals already taken on every link when the first condition
    // is routed, and the time from which each chunk is available at its source
    const uint32_t L = (uint32_t)links.size();
    const uint32_t C = (uint32_t)conds.size();
    std::vector<uint64_t> w(L);
    for (uint32_t l = 0; l < L; ++l) w[l] = link_cost(links[l], chunk_bytes);
    std::vector<std::vector<uint32_t>> out(n);
    for (uint32_t l = 0; l < L; ++l) out[links[l].src].push_back(l);

    // Alg. 3 lines 1-7
    struct Key { uint64_t dist; uint32_t draw, chunk; };
    std::vector<Key> order;
    std::map<uint32_t, std::vector<uint64_t>> dist_from;
    for (uint32_t c = 0; c < C; ++c) {
        if (!conds[c].present || conds[c].dests.empty()) continue;
        auto f = dist_from.find(conds[c].src);
        if (f == dist_from.end()) f = dist_from.emplace(conds[c].src, dijkstra(n, links, w, conds[c].src)).first;
        uint64_t dmax = 0;
        for (uint32_t d : conds[c].dests) {
            if (f->second[d] == INF) return OR_ERR_UNREACHABLE;
            dmax = std::max(dmax, f->second[d]);
        }
        order.push_back(Key{dmax, draw(seed, c, 0, 0, 2), c});
    }
    std::sort(order.begin(), order.end(), [](const Key& a, const Key& b) {
        if (a.dist != b.dist) return a.dist > b.dist;
        if (a.draw != b.draw) return a.draw < b.draw;
        return a.chunk < b.chunk;
    });

    std::vector<BusyLink> busy(L);
    if (busy0) busy = *busy0;
    std::vector<SwitchBuf> sbuf(buf_limit ? n : 0);
    auto limited = [&](uint32_t v) { return buf_limit && buf_limit[v] != NONE; };
    res = CopyResult{};
    std::vector<uint64_t> arr(n);
    std::vector<uint32_t> pred(n);
    std::vector<char> done(n), keep(n);
    for (const Key& k : order) {                              // Alg. 3 line 9
        const Cond& c = conds[k.chunk];
        // Alg. 2 + section 4.6: visit devices in order of arrival
        std::fill(arr.begin(), arr.end(), INF);
        std::fill(pred.begin(), pred.end(), NONE);
        std::fill(done.begin(), done.end(), 0);
        using QE = std::pair<uint64_t, uint32_t>;
        std::priority_queue<QE, std::vector<QE>, std::greater<QE>> pq;
        const uint64_t t0 = ready ? (*ready)[k.chunk] : 0;
        arr[c.src] = t0;
        pq.push({t0, c.src});
        size_t left = c.dests.size();
        uint64_t last = 0;                                    // arrival at the last dest reached
        while (!pq.empty()) {
            auto [a, u] = pq.top();
            pq.pop();
            if (done[u] || a != arr[u]) continue;
            if (left == 0 && a > last) break;                 // Alg. 2 line 4: all dests visited
            done[u] = 1;
            if (left && std::binary_search(c.dests.begin(), c.dests.end(), u)) { --left; last = a; }
            uint64_t from = a;                                // a node without multicast: one out-link after the other (4.7)
            for (uint32_t l : out[u]) {                       // NextDevices(TEN, u, .), ascending link id
                const uint32_t v = links[l].dst;
                const bool serial = no_mcast && no_mcast[u];
                if (done[v] && !serial) continue;             // Alg. 2 line 7
                if (limited(v) && buf_limit[v] == 0) continue;   // a node that buffers nothing is never visited
                const uint64_t t = earliest_start_buffered(busy[l], from, w[l], limited(v) ? &sbuf[v] : nullptr,
                                                           limited(v) ? buf_limit[v] : 0) + w[l];
                if (serial) from = t;
                if (done[v]) continue;
                if (t < arr[v] || (t == arr[v] && l < pred[v])) {   // Q20
                    arr[v] = t;
                    pred[v] = l;
                    pq.push({t, v});
                }
            }
        }
        if (left) return OR_ERR_UNREACHABLE;
        // keep the paths to the dests only
        std::fill(keep.begin(), keep.end(), 0);
        for (uint32_t d : c.dests)
            for (uint32_t v = d; v != c.src && !keep[v]; v = links[pred[v]].src) keep[v] = 1;
        std::vector<uint64_t> release(buf_limit ? n : 0, 0);  // end of the last kept transfer out of each node
        for (uint32_t v = 0; v < n; ++v) {
            if (!keep[v]) continue;
            const uint32_t l = pred[v];
            res.recs.push_back(Rec{k.chunk, links[l].src, v, l, arr[v] - w[l], arr[v]});
            occupy(busy[l], arr[v] - w[l], arr[v]);           // Alg. 3 line 13
            res.T = std::max(res.T, arr[v]);
            if (buf_limit) release[links[l].src] = std::max(release[links[l].src], arr[v]);
        }
        if (buf_limit)                                        // the chunk was buffered at every limited node that forwarded it
            for (uint32_t v = 0; v < n; ++v)
                if (limited(v) && keep[v] && release[v] > 0) sbuf[v].add(arr[v], release[v]);
        ++res.events;                                         // here: conditions routed
    }
    std::sort(res.recs.begin(), res.recs.end(), [](const Rec& a, const Rec& b) {
        if (a.t_start_ps != b.t_start_ps) return a.t_start_ps < b.t_start_ps;
        return a.link < b.link;
    });
    res.wants_total = res.recs.size();
    return OR_OK;
}

// relay rule used by the dispatchers below: 0 = thin relay tree (step C), 1 = dynamic,
// 2 = the paper's per-condition BFS (no matching loop at all)
struct SwitchModel { const uint32_t* buf_limit = nullptr; const uint8_t* no_mcast = nullptr; };   // section 4.7, BFS mode only

int synth_copy_mode(int relay, uint32_t n, const std::vector<Link>& links, const std::vector<Cond>& conds,
                    uint64_t chunk_bytes, uint64_t seed, CopyResult& res, SwitchModel sw = SwitchModel()) {
    if (relay == 2) return synth_copy_bfs(n, links, conds, chunk_bytes, seed, res, sw.buf_limit, sw.no_mcast);
    if (relay == 3) return synth_copy(n, links, conds, chunk_bytes, seed, res, nullptr, true);   // thin tree, c.dist pick
    return relay == 1 ? synth_copy_dynamic(n, links, conds, chunk_bytes, seed, res)
                      : synth_copy(n, links, conds, chunk_bytes, seed, res);
}

// -------------------------------------------------------------------------------------
// REDUCE mode (reading Q10): synthesize the broadcast root -> holders on
// the TRANSPOSED topology, then reverse every transfer in direction and in time.
// -------------------------------------------------------------------------------------
int synth_reduce(uint32_t n, const std::vector<Link>& links, const std::vector<Cond>& bcast,
                 uint64_t chunk_bytes, uint64_t seed, CopyResult& res, int relay = 0, SwitchModel sw = SwitchModel()) {
    std::vector<Link> tr(links);
    for (Link& l : tr) std::swap(l.src, l.dst);
    CopyResult b;
    const int rc = synth_copy_mode(relay, n, tr, bcast, chunk_bytes, seed, b, sw);
    if (rc != OR_OK) return rc;
    res.recs.clear();
    for (const Rec& r : b.recs)   // (c, a, b, l, ts, te) -> (c, src=b, dst=a, l, T-te, T-ts)
        res.recs.push_back(Rec{r.chunk, r.dst, r.src, r.link, b.T - r.t_end_ps, b.T - r.t_start_ps});
    std::sort(res.recs.begin(), res.recs.end(), [](const Rec& a, const Rec& b2) {
        if (a.t_start_ps != b2.t_start_ps) return a.t_start_ps < b2.t_start_ps;
        return a.link < b2.link;
    });
    res.T = b.T;
    res.events = b.events;
    res.wants_total = b.wants_total;
    return OR_OK;
}

struct Result {
    std::vector<Rec> recs;
    uint64_t T = 0;
    uint64_t events = 0;
    uint64_t wants_total = 0;
    uint64_t T_phase1 = 0;   // all-reduce: time of the reduce phase
    int mode = 0;            // 0 copy, 1 reduce, 2 all-reduce
};

// -------------------------------------------------------------------------------------
// Step R + dispatch.  Pre/postcondition (NPU-centric) -> conditions
// (chunk-centric).  |pre(c)| > 1 marks a reduction chunk (reading Q12).
// -------------------------------------------------------------------------------------
int synthesize(uint32_t n_npus, const Link* links_p, uint32_t n_links, const uint32_t* group,
               uint32_t n_members, uint32_t n_chunks, const Pair* pre_p, uint64_t n_pre,
               const Pair* post_p, uint64_t n_post, uint64_t chunk_bytes, uint64_t seed,
               Result& out, int relay = 0, SwitchModel sw = SwitchModel(), bool pipeline = false) {
    if (n_links && !links_p) return OR_ERR_INVALID;
    if (n_members && !group) return OR_ERR_INVALID;
    if ((n_pre && !pre_p) || (n_post && !post_p)) return OR_ERR_INVALID;
    if (chunk_bytes == 0) return OR_ERR_INVALID;
    std::vector<Link> links(links_p, links_p + n_links);
    for (const Link& l : links) {
        if (l.src >= n_npus || l.dst >= n_npus || l.src == l.dst || l.bytes_per_ps == 0)
            return OR_ERR_INVALID;
    }
    std::vector<char> member(n_npus, 0);
    for (uint32_t i = 0; i < n_members; ++i) {
        if (group[i] >= n_npus || member[group[i]]) return OR_ERR_INVALID;
        member[group[i]] = 1;
    }
    std::vector<std::set<uint32_t>> pre(n_chunks), post(n_chunks);
    for (uint64_t i = 0; i < n_pre; ++i) {
        if (pre_p[i].chunk >= n_chunks || pre_p[i].npu >= n_npus || !member[pre_p[i].npu])
            return OR_ERR_INVALID;
        pre[pre_p[i].chunk].insert(pre_p[i].npu);
    }
    for (uint64_t i = 0; i < n_post; ++i) {
        if (post_p[i].chunk >= n_chunks || post_p[i].npu >= n_npus || !member[post_p[i].npu])
            return OR_ERR_INVALID;
        post[post_p[i].chunk].insert(post_p[i].npu);
    }
    bool all_single = true, all_multi_one = true, all_multi_many = true;
    for (uint32_t c = 0; c < n_chunks; ++c) {
        if (pre[c].empty() || post[c].empty()) return OR_ERR_INVALID;
        const bool single = pre[c].size() == 1;
        all_single &= single;
        all_multi_one &= (!single && post[c].size() == 1);
        all_multi_many &= (!single && post[c].size() > 1);
    }

    out = Result{};
    if (all_single) {                                        // COPY
        std::vector<Cond> conds(n_chunks);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            conds[c].present = true;
            conds[c].src = *pre[c].begin();
            for (uint32_t d : post[c]) if (d != conds[c].src) conds[c].dests.push_back(d);
        }
        CopyResult r;
        const int rc = synth_copy_mode(relay, n_npus, links, conds, chunk_bytes, seed, r, sw);
        if (rc != OR_OK) return rc;
        out.recs = std::move(r.recs); out.T = r.T; out.events = r.events;
        out.wants_total = r.wants_total; out.mode = 0;
        return OR_OK;
    }
    if (all_multi_one) {                                     // REDUCE / Reduce-Scatter
        std::vector<Cond> bc(n_chunks);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            bc[c].present = true;
            bc[c].src = *post[c].begin();
            for (uint32_t d : pre[c]) if (d != bc[c].src) bc[c].dests.push_back(d);
        }
        CopyResult r;
        const int rc = synth_reduce(n_npus, links, bc, chunk_bytes, seed, r, relay, sw);
        if (rc != OR_OK) return rc;
        out.recs = std::move(r.recs); out.T = r.T; out.events = r.events;
        out.wants_total = r.wants_total; out.mode = 1; out.T_phase1 = r.T;
        return OR_OK;
    }
    if (all_multi_many) {                                    // ALL-REDUCE = RS then AG (Q11)
        std::vector<Cond> bc(n_chunks), cp(n_chunks);
        for (uint32_t c = 0; c < n_chunks; ++c) {
            std::vector<uint32_t> I;
            for (uint32_t v : pre[c]) if (post[c].count(v)) I.push_back(v);
            if (I.empty()) I.assign(post[c].begin(), post[c].end());
            const uint32_t root = I[c % I.size()];           // std::set iterates ascending
            bc[c].present = cp[c].present = true;
            bc[c].src = cp[c].src = root;
            for (uint32_t d : pre[c]) if (d != root) bc[c].dests.push_back(d);
            for (uint32_t d : post[c]) if (d != root) cp[c].dests.push_back(d);
        }
        CopyResult r1, r2;
        int rc = synth_reduce(n_npus, links, bc, chunk_bytes, seed, r1, relay, sw);
        if (rc != OR_OK) return rc;
        if (pipeline) {
            // Pipelined All-Reduce (PAPER.md:330 composes the phases, reading Q26 lets them overlap): the
            // copy phase of chunk c may start as soon as root(c) holds the complete sum -- the end of the last transfer of
            // c into the root -- instead of at the end of the whole reduce phase.  Both phases share the links, so the
            // copy phase is routed by the per-condition search (BFS mode only) against the intervals the reduce phase took.
            if (relay != 2 || sw.buf_limit || sw.no_mcast) return OR_ERR_UNSUPPORTED;
            std::vector<BusyLink> busy(links.size());
            std::vector<uint64_t> ready(n_chunks, 0);
            for (const Rec& r : r1.recs) {
                occupy(busy[r.link], r.t_start_ps, r.t_end_ps);
                if (r.dst == cp[r.chunk].src) ready[r.chunk] = std::max(ready[r.chunk], r.t_end_ps);
            }
            rc = synth_copy_bfs(n_npus, links, cp, chunk_bytes, seed, r2, nullptr, nullptr, &busy, &ready);
            if (rc != OR_OK) return rc;
            out.recs = std::move(r1.recs);
            out.recs.insert(out.recs.end(), r2.recs.begin(), r2.recs.end());
            std::sort(out.recs.begin(), out.recs.end(), [](const Rec& a, const Rec& b) {
                if (a.t_start_ps != b.t_start_ps) return a.t_start_ps < b.t_start_ps;
                return a.link < b.link;
            });
            out.T_phase1 = r1.T;
            out.T = std::max(r1.T, r2.T);
            out.events = r1.events + r2.events;
            out.wants_total = r1.wants_total + r2.wants_total;
            out.mode = 2;
            return OR_OK;
        }
        rc = synth_copy_mode(relay, n_npus, links, cp, chunk_bytes, seed, r2, sw);
        if (rc != OR_OK) return rc;
        out.recs = std::move(r1.recs);
        for (const Rec& r : r2.recs)
            out.recs.push_back(Rec{r.chunk, r.src, r.dst, r.link, r.t_start_ps + r1.T, r.t_end_ps + r1.T});
        std::sort(out.recs.begin(), out.recs.end(), [](const Rec& a, const Rec& b) {
            if (a.t_start_ps != b.t_start_ps) return a.t_start_ps < b.t_start_ps;
            return a.link < b.link;
        });
        out.T_phase1 = r1.T;
        out.T = r1.T + r2.T;
        out.events = r1.events + r2.events;
        out.wants_total = r1.wants_total + r2.wants_total;
        out.mode = 2;
        return OR_OK;
    }
    return OR_ERR_UNSUPPORTED;
}

}  // namespace

// =====================================================================================
// C interface for ctypes (tests, smoke, bench cpu_baseline).  Host pointers only.
// =====================================================================================
extern "C" {

struct oracle_link { uint32_t src, dst; uint64_t alpha_ps, bytes_per_ps; };
struct oracle_pair { uint32_t npu, chunk; };
struct oracle_rec  { uint32_t chunk, src, dst, link; uint64_t t_start_ps, t_end_ps; };
static_assert(sizeof(oracle_link) == sizeof(Link), "layout");
static_assert(sizeof(oracle_pair) == sizeof(Pair), "layout");
static_assert(sizeof(oracle_rec) == sizeof(Rec) && sizeof(Rec) == 32, "layout");

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox4x32_10(ctr, key, out);
}

uint64_t oracle_link_cost(uint64_t alpha_ps, uint64_t bytes_per_ps, uint64_t chunk_bytes) {
    return link_cost(Link{0, 1, alpha_ps, bytes_per_ps}, chunk_bytes);
}

// distances from s under the alpha-beta cost; out[n_npus], UINT64_MAX = unreachable
int oracle_distances(uint32_t n_npus, const oracle_link* links, uint32_t n_links,
                     uint64_t chunk_bytes, uint32_t s, uint64_t* out) {
    std::vector<Link> ls((const Link*)links, (const Link*)links + n_links);
    std::vector<uint64_t> w(n_links);
    for (uint32_t l = 0; l < n_links; ++l) w[l] = link_cost(ls[l], chunk_bytes);
    std::vector<uint64_t> D = dijkstra(n_npus, ls, w, s);
    std::copy(D.begin(), D.end(), out);
    return OR_OK;
}

int oracle_synthesize(uint32_t n_npus, const oracle_link* links, uint32_t n_links,
                      const uint32_t* group, uint32_t n_members, uint32_t n_chunks,
                      const oracle_pair* pre, uint64_t n_pre, const oracle_pair* post,
                      uint64_t n_post, uint64_t chunk_bytes, uint64_t seed, void** handle) {
    if (!handle) return OR_ERR_INVALID;
    Result* r = new Result();
    const int rc = synthesize(n_npus, (const Link*)links, n_links, group, n_members, n_chunks,
                              (const Pair*)pre, n_pre, (const Pair*)post, n_post, chunk_bytes,
                              seed, *r);
    if (rc != OR_OK) { delete r; return rc; }
    *handle = r;
    return OR_OK;
}

int oracle_synthesize_relay(uint32_t n_npus, const oracle_link* links, uint32_t n_links,
                            const uint32_t* group, uint32_t n_members, uint32_t n_chunks,
                            const oracle_pair* pre, uint64_t n_pre, const oracle_pair* post,
                            uint64_t n_post, uint64_t chunk_bytes, uint64_t seed, int relay, void** handle) {
    if (!handle || relay < 0 || relay > 3) return OR_ERR_INVALID;
    Result* r = new Result();
    const int rc = synthesize(n_npus, (const Link*)links, n_links, group, n_members, n_chunks,
                              (const Pair*)pre, n_pre, (const Pair*)post, n_post, chunk_bytes,
                              seed, *r, relay);
    if (rc != OR_OK) { delete r; return rc; }
    *handle = r;
    return OR_OK;
}

// BFS mode with the switch model of section 4.7: buf_limit[n_npus] (0xFFFFFFFF = no limit) and no_mcast[n_npus]
// (non-zero = the node forwards one transfer at a time); either may be NULL
int oracle_synthesize_switches(uint32_t n_npus, const oracle_link* links, uint32_t n_links,
                               const uint32_t* group, uint32_t n_members, uint32_t n_chunks,
                               const oracle_pair* pre, uint64_t n_pre, const oracle_pair* post,
                               uint64_t n_post, uint64_t chunk_bytes, uint64_t seed,
                               const uint32_t* buf_limit, const uint8_t* no_mcast, void** handle) {
    if (!handle) return OR_ERR_INVALID;
    Result* r = new Result();
    SwitchModel sw;
    sw.buf_limit = buf_limit; sw.no_mcast = no_mcast;
    const int rc = synthesize(n_npus, (const Link*)links, n_links, group, n_members, n_chunks,
                              (const Pair*)pre, n_pre, (const Pair*)post, n_post, chunk_bytes,
                              seed, *r, 2, sw);
    if (rc != OR_OK) { delete r; return rc; }
    *handle = r;
    return OR_OK;
}

// BFS mode, All-Reduce with overlapping phases (reading Q26); anything but an all-reduce problem is synthesized as usual
int oracle_synthesize_pipelined(uint32_t n_npus, const oracle_link* links, uint32_t n_links,
                                const uint32_t* group, uint32_t n_members, uint32_t n_chunks,
                                const oracle_pair* pre, uint64_t n_pre, const oracle_pair* post,
                                uint64_t n_post, uint64_t chunk_bytes, uint64_t seed, void** handle) {
    if (!handle) return OR_ERR_INVALID;
    Result* r = new Result();
    const int rc = synthesize(n_npus, (const Link*)links, n_links, group, n_members, n_chunks,
                              (const Pair*)pre, n_pre, (const Pair*)post, n_post, chunk_bytes,
                              seed, *r, 2, SwitchModel(), true);
    if (rc != OR_OK) { delete r; return rc; }
    *handle = r;
    return OR_OK;
}

// wants relation of step C for a COPY-mode problem given directly as conditions:
// cond_src[c], dests CSR (dest_off[c]..dest_off[c+1]).  Writes pairs (node, chunk) sorted
// by (node, chunk) to out (capacity cap); returns the number of pairs or a negative error.
int64_t oracle_wants(uint32_t n_npus, const oracle_link* links, uint32_t n_links,
                     uint32_t n_chunks, const uint32_t* cond_src, const uint64_t* dest_off,
                     const uint32_t* dests, uint64_t chunk_bytes, uint64_t seed,
                     oracle_pair* out, uint64_t cap) {
    std::vector<Link> ls((const Link*)links, (const Link*)links + n_links);
    std::vector<Cond> conds(n_chunks);
    for (uint32_t c = 0; c < n_chunks; ++c) {
        conds[c].present = true;
        conds[c].src = cond_src[c];
        conds[c].dests.assign(dests + dest_off[c], dests + dest_off[c + 1]);
    }
    CopyResult r;
    std::vector<std::vector<uint32_t>> wants;
    const int rc = synth_copy(n_npus, ls, conds, chunk_bytes, seed, r, &wants);
    if (rc != OR_OK) return rc;
    uint64_t k = 0;
    for (uint32_t v = 0; v < n_npus; ++v)
        for (uint32_t c : wants[v]) { if (k < cap) out[k] = oracle_pair{v, c}; ++k; }
    return (int64_t)k;
}

uint64_t oracle_size(const void* h) { return ((const Result*)h)->recs.size(); }
const oracle_rec* oracle_records(const void* h) { return (const oracle_rec*)((const Result*)h)->recs.data(); }
uint64_t oracle_time(const void* h) { return ((const Result*)h)->T; }
uint64_t oracle_events(const void* h) { return ((const Result*)h)->events; }
uint64_t oracle_wants_total(const void* h) { return ((const Result*)h)->wants_total; }
uint64_t oracle_time_phase1(const void* h) { return ((const Result*)h)->T_phase1; }
int oracle_mode(const void* h) { return ((const Result*)h)->mode; }
void oracle_free(void* h) { delete (Result*)h; }

}  // extern "C"
