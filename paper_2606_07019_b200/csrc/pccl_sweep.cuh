// =========================================================================================
// pccl_sweep.cuh -- the candidate bitmap (row a5) as a streaming kernel.
//
//   cand(l) = have[src_l] & wants[dst_l]            (one chunk per link; north star: per-link bitmap)
//   gcnt[l][s] = popcount of cand(l) over segment s (64 words = 4096 chunks),  gtot[l] = their sum
//
// for EVERY link, destination by destination: the wants row of v is read once and ANDed with the have rows of its
// in-links' sources, (N + L) rows per sweep -- SURVEY 8(d)'s algorithmic byte count.  The barrier loops run it once
// per phase to seed the kept counts; pccl_device_candidate_sweep times it alone (bench.py's memory-bound leg, the
// kernel the HBM / L2 roofline is read on).
//
// Two forms, same result:
//   TMA = true   rows are staged in shared memory by bulk asynchronous copies (cp.async.bulk -> UBLKCP in SASS):
//                one elected thread issues, per 4 KB slice, one copy of the wants row and one per source row
//                (<= 9 copies of 4 KB) into a ring of STAGES stages, each guarded by an mbarrier that counts the
//                bytes (complete_tx); the 256 threads wait on the stage's barrier, AND + popcount from shared memory
//                (one 64-word segment per warp), and a block barrier hands the stage back.
//   TMA = false  every lane loads its 16 bytes of each row with ld.global.cg.v4 (the form of k_loop's dense sweep).
// =========================================================================================
#pragma once
#include "pccl_device.cuh"

namespace pccl {

constexpr int SW_THREADS = 256;
constexpr int SW_SLICE_U4 = 256;                 // uint4 per row and slice: 4 KB, one 512-byte segment per warp
constexpr int SW_STAGES = 2;
constexpr int SW_ROWS = NB + 1;                  // wants row + up to NB source rows per sweep of in-links

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
    asm volatile(
        "{\n .reg .pred p;\n"
        "W_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @!p bra W_%=;\n}"
        ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared bulk copy, completion counted in bytes on the mbarrier (bytes: a multiple of 16, both ends 16-byte aligned)
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <bool TMA>
__global__ void __launch_bounds__(SW_THREADS) k_count_sweep(LoopArgs a) {
    extern __shared__ __align__(128) unsigned char sw_smem[];    // [SW_STAGES][SW_ROWS][4 KB] (TMA form only)
    __shared__ __align__(8) unsigned long long full[SW_STAGES];
    __shared__ uint32_t s_src[NB], s_link[NB];
    __shared__ uint32_t s_tot[NB][SW_THREADS / 32];
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t Q = a.Wp >> 1;                                // uint4 per row
    const uint32_t nsl = (Q + SW_SLICE_U4 - 1) / SW_SLICE_U4;    // slices per row
    const uint4* have4 = reinterpret_cast<const uint4*>(a.have);
    const uint4* wants4 = reinterpret_cast<const uint4*>(a.wants);
    if (TMA) {
        if (tid == 0) {
            for (int s = 0; s < SW_STAGES; ++s) mbar_init(&full[s], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
    }
    uint32_t phase_bits = 0;                                     // parity of each stage's barrier (bit s)
    // work units: (destination v, sweep of NB in-links, part of the row) dealt round-robin to the CTAs -- `parts` row
    // parts per destination keep the CTAs balanced when there are only a few destinations per CTA
    const uint32_t parts = max(1u, a.flags);                      // (a.flags carries the number of parts here)
    const uint32_t per_part = (nsl + parts - 1) / parts;
    for (uint32_t unit = blockIdx.x; unit < a.N * parts; unit += gridDim.x) {
        const uint32_t v = unit / parts, part = unit - v * parts;
        const uint32_t k_lo = part * per_part, k_hi = min(nsl, k_lo + per_part);
        if (k_lo >= k_hi) continue;                               // block-uniform
        const uint32_t e0 = a.in_off[v], e1 = a.in_off[v + 1];
        for (uint32_t eb = e0; eb < e1; eb += NB) {              // in-links in sweeps of NB
            const uint32_t nb = min((uint32_t)NB, e1 - eb);
            __syncthreads();
            if (tid < nb) { const uint32_t l = a.in_link[eb + tid]; s_link[tid] = l; s_src[tid] = a.esrc[l]; }
            __syncthreads();
            uint32_t tot[NB];
#pragma unroll
            for (int j = 0; j < NB; ++j) tot[j] = 0;
            if (TMA) {
                auto issue = [&](uint32_t k) {                   // thread 0: slice k of all rows into stage (k - k_lo) % STAGES
                    const uint32_t st = (k - k_lo) % SW_STAGES;
                    const uint32_t q0 = k * SW_SLICE_U4, nq = min((uint32_t)SW_SLICE_U4, Q - q0);
                    unsigned char* base = sw_smem + (size_t)st * SW_ROWS * SW_SLICE_U4 * 16;
                    mbar_expect_tx(&full[st], (nb + 1) * nq * 16);
                    bulk_g2s(base, wants4 + (size_t)v * Q + q0, nq * 16, &full[st]);
                    for (uint32_t j = 0; j < nb; ++j)
                        bulk_g2s(base + (size_t)(j + 1) * SW_SLICE_U4 * 16, have4 + (size_t)s_src[j] * Q + q0, nq * 16, &full[st]);
                };
                if (tid == 0)
                    for (uint32_t k = k_lo; k < k_lo + SW_STAGES - 1 && k < k_hi; ++k) issue(k);
                for (uint32_t k = k_lo; k < k_hi; ++k) {
                    if (tid == 0 && k + SW_STAGES - 1 < k_hi) issue(k + SW_STAGES - 1);   // its stage was handed back at the end of slice k - 1
                    const uint32_t st = (k - k_lo) % SW_STAGES;
                    mbar_wait(&full[st], (phase_bits >> st) & 1u);
                    phase_bits ^= 1u << st;
                    const uint4* base = reinterpret_cast<const uint4*>(sw_smem + (size_t)st * SW_ROWS * SW_SLICE_U4 * 16);
                    const uint32_t q = k * SW_SLICE_U4 + tid;
                    const bool ok = q < Q;
                    const uint4 wv = ok ? base[tid] : make_uint4(0, 0, 0, 0);
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        if (j < (int)nb) {                        // block-uniform
                            const uint4 hv = ok ? base[(j + 1) * SW_SLICE_U4 + tid] : make_uint4(0, 0, 0, 0);
                            const uint32_t c = __reduce_add_sync(0xFFFFFFFFu, (uint32_t)popc128(and128(hv, wv)));
                            const uint32_t seg = k * (SW_SLICE_U4 / SEG_U4) + warp;
                            if (lane == 0 && seg < a.S) { a.gcnt[(size_t)s_link[j] * a.S + seg] = c; tot[j] += c; }
                        }
                    }
                    __syncthreads();                              // every thread is done with the stage: it may be refilled
                }
            } else {
                for (uint32_t k = k_lo; k < k_hi; ++k) {
                    const uint32_t q = k * SW_SLICE_U4 + tid;
                    const bool ok = q < Q;
                    uint4 wv = make_uint4(0, 0, 0, 0), hv[NB];
                    if (ok) wv = ldcg128(wants4 + (size_t)v * Q + q);
#pragma unroll
                    for (int j = 0; j < NB; ++j) {                // all loads of the slice in flight before the first use
                        hv[j] = make_uint4(0, 0, 0, 0);
                        if (j < (int)nb && ok) hv[j] = ldcg128(have4 + (size_t)s_src[j] * Q + q);
                    }
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        if (j < (int)nb) {
                            const uint32_t c = __reduce_add_sync(0xFFFFFFFFu, (uint32_t)popc128(and128(hv[j], wv)));
                            const uint32_t seg = k * (SW_SLICE_U4 / SEG_U4) + warp;
                            if (lane == 0 && seg < a.S) { a.gcnt[(size_t)s_link[j] * a.S + seg] = c; tot[j] += c; }
                        }
                    }
                }
            }
            if (lane == 0)
                for (uint32_t j = 0; j < nb; ++j) s_tot[j][warp] = tot[j];
            __syncthreads();
            if (tid < nb) {
                uint32_t t = 0;
                for (int w = 0; w < SW_THREADS / 32; ++w) t += s_tot[tid][w];
                if (parts == 1) a.gtot[s_link[tid]] = t;
                else if (t) atomicAdd(&a.gtot[s_link[tid]], t);  // (zeroed by the launcher)
            }
        }
    }
}

// sequential read of a buffer with the sweep's access pattern (128-bit ld.global.cg, grid-stride): the measured
// ceiling of the level that serves it -- L2 when the buffer fits there, HBM when it does not (bench.py's peak legs)
__global__ void __launch_bounds__(SW_THREADS) k_read_sweep(const uint4* __restrict__ buf, uint64_t n_u4, uint32_t* sink) {
    uint32_t acc = 0;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n_u4; i += 4 * stride) {   // four independent loads in flight per thread
        const uint4 x0 = ldcg128(buf + i), x1 = ldcg128(buf + i + stride), x2 = ldcg128(buf + i + 2 * stride),
                    x3 = ldcg128(buf + i + 3 * stride);
        acc += popc128(x0) + popc128(x1) + popc128(x2) + popc128(x3);
    }
    for (; i < n_u4; i += stride) acc += popc128(ldcg128(buf + i));
    if (acc == 0xFFFFFFFFu) *sink = acc;               // (keeps the loads alive)
}

}  // namespace pccl
