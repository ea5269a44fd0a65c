// append_tc2_body.cuh — the CTA body of append_prefill_attn for head_dim 128 on tcgen05 / TMEM (two 128-row tiles per
// CTA).  Used by append_tc2_kernel (append_attn_tc2.cu) and by tail_kernel (tail_fused.cu: the CTAs that take the append
// role of a mixed step, and the decode-role CTAs once their share is done).  Design notes: append_attn_tc2.cu.
#pragma once
#include <math.h>

#include "common.cuh"
#include "internal.h"
#include "tc5.cuh"


constexpr int kT2Threads = 352;
constexpr int kChunk = 64;                 // KV tokens per pipeline step
constexpr int kChunkBlocks = kChunk / 16;
constexpr uint32_t kTmemCols2 = 512;

struct AppendTc2Params {
    const AppendItem* items;
    int32_t n_items;
    const uint8_t* pool_layer;
    const uint16_t* q;
    const int32_t* tables;
    uint16_t* out;
    float* lse;
    float* po;
    float* pml;
    int32_t max_blocks, Hq, Hkv, G;
    float scale_log2;
    uint32_t* sched;   // [0] next item of the work queue (beyond the first gridDim.x), [1] unused, [2] next decode share of
                       // tail_kernel; zeroed by the launcher (cudaMemsetAsync) before every launch
};

constexpr uint32_t kOffQ2 = 0;                           // 2 tiles x [2 halves][128 rows][128 B]
constexpr uint32_t kOffK2 = 65536;                       // ST x [2 halves][4 blocks][2048 B]
__host__ __device__ constexpr uint32_t smem_bytes2(int ST) { return kOffK2 + 2u * ST * 16384u + 256u; }


template <int ST>
struct AppendTc2Smem {
    static constexpr int kKSt = ST, kVSt = ST;
    static constexpr uint32_t kOffV2 = kOffK2 + kKSt * 16384;       // kVSt x [4 blocks][4096 B]
    static constexpr uint32_t kOffBar2 = kOffV2 + kVSt * 16384;     // mbarriers + TMEM slot
};

// Barrier init + TMEM allocation; every thread of the CTA calls it (ends with a CTA barrier).  Returns the TMEM base.
template <int ST>
__device__ __forceinline__ uint32_t append_tc2_setup(uint8_t* smem) {
    constexpr uint32_t kOffBar2 = AppendTc2Smem<ST>::kOffBar2;
    const uint32_t sbase = smem_u32(smem);
    if (sbase & 1023u) __trap();   // SWIZZLE_128B operand tiles must be 1024-byte aligned
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kOffBar2);
    uint64_t *k_full = bars, *k_empty = bars + 4, *v_full = bars + 8, *v_empty = bars + 12;
    uint64_t *s_full = bars + 16, *p_full = bars + 20, *o_done = bars + 24;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 26);
    const int warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        for (int i = 0; i < 4; ++i) {
            mbar_init(&k_full[i], 1);
            mbar_init(&k_empty[i], 2);   // both MMA warps release a stage
            mbar_init(&v_full[i], 1);
            mbar_init(&v_empty[i], 2);
            mbar_init(&s_full[i], 1);
            mbar_init(&p_full[i], 128);
        }
        mbar_init(&o_done[0], 1);
        mbar_init(&o_done[1], 1);
        fence_mbar_init();
    }
    if (warp == 9) tmem_alloc(tmem_slot, kTmemCols2);   // warp 9 also frees it
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    return *tmem_slot;
}

template <int ST>
__device__ __forceinline__ void append_tc2_teardown(uint32_t tmem) {
    __syncthreads();
    if ((threadIdx.x >> 5) == 9) tmem_dealloc(tmem, kTmemCols2);
}

// Work items from the queue: this CTA starts with item `it_first` and then takes queue_base + (next ticket of p.sched).
// Items are sorted longest first, so this is LPT scheduling.  All kT2Threads threads of the CTA call it.
template <int ST>
__device__ __forceinline__ void append_tc2_items(const AppendTc2Params& p, uint8_t* smem, const uint32_t tmem, const int it_first,
                                                 const int queue_base) {
    constexpr int D = 128;
    constexpr int kKSt = ST, kVSt = ST;
    constexpr uint32_t kOffV2 = AppendTc2Smem<ST>::kOffV2;
    constexpr uint32_t kOffBar2 = AppendTc2Smem<ST>::kOffBar2;
    constexpr int TB = 4096;
    const uint32_t sbase = smem_u32(smem);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kOffBar2);
    uint64_t *k_full = bars, *k_empty = bars + 4, *v_full = bars + 8, *v_empty = bars + 12;
    uint64_t *s_full = bars + 16 /* [tile][buf] */, *p_full = bars + 20 /* [tile][buf] */, *o_done = bars + 24 /* [tile] */;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 26);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = p.G;
    const size_t kv_stride = (size_t)p.Hkv * TB;
    const size_t blk_stride = 2 * kv_stride;
    uint32_t kc = 0;             // K/V chunks pushed through the rings so far (all roles agree)
    uint32_t tcnA = 0, tcnB = 0;   // chunks each tile has processed so far (tile B skips items without rows for it)

    // Work queue: CTA c starts with item c and then takes the next unclaimed one (items are sorted longest first, so
    // this is LPT scheduling).  Thread 0 claims the NEXT item while the current one runs; the index travels through
    // shared memory under the barrier that ends the Q staging.
    uint32_t* next_slot = tmem_slot + 2;   // [2] in the barrier block
    int it = it_first, par = 0;
    while (it < p.n_items) {
        if (threadIdx.x == 0) next_slot[par] = queue_base + atomicAdd(p.sched, 1u);
        const int4 i0 = __ldg(reinterpret_cast<const int4*>(p.items + it));
        const int4 i1 = __ldg(reinterpret_cast<const int4*>(p.items + it) + 1);
        const int4 i2 = __ldg(reinterpret_cast<const int4*>(p.items + it) + 2);
        const int conv = i0.x, head = i0.y, row_begin = i0.z, q_start = i0.w;
        const int m = i1.x, kv_len = i1.y, blk_begin = i1.z, blk_end = i1.w;
        const int partial = i2.x, direct = i2.y;
        const int P = kv_len - m;
        const int rows_total = m * G;
        const int nblk = blk_end - blk_begin;
        const int nch = (nblk + kChunkBlocks - 1) / kChunkBlocks;
        const bool hasB = row_begin + 128 < rows_total;

        // ---- stage the Q rows of both tiles in the K-major SWIZZLE_128B image ------------------------
        if (warp < 8) {
            const int t = warp >> 2, r = threadIdx.x & 127, sr = row_begin + t * 128 + r;
            if (t == 0 || hasB) {
                const bool ok = sr < rows_total;
                const uint4* src = reinterpret_cast<const uint4*>(
                    p.q + ((size_t)(q_start + (ok ? sr / G : 0)) * p.Hq + (size_t)head * G + (ok ? sr % G : 0)) * D);
                uint4 v[16];
#pragma unroll
                for (int c = 0; c < 16; ++c) v[c] = ok ? __ldg(src + c) : make_uint4(0, 0, 0, 0);
#pragma unroll
                for (int c = 0; c < 16; ++c)
                    *reinterpret_cast<uint4*>(smem + kOffQ2 + t * 32768 + (c >> 3) * 16384 + r * 128 +
                                              (((c & 7) ^ (r & 7)) << 4)) = v[c];
                fence_proxy_async();
            }
        }
        tc_fence_before();
        __syncthreads();   // Q staged; the previous item's epilogues have finished reading O
        tc_fence_after();
        const int it_next = (int)next_slot[par];

        if (warp == 8) {
            // ================= producer =================
            if (lane == 0) {
                const int32_t* tab = p.tables + (size_t)conv * p.max_blocks + blk_begin;
                const uint8_t* head_base = p.pool_layer + (size_t)head * TB;
                int ids[kChunkBlocks], nids[kChunkBlocks];
#pragma unroll
                for (int jb = 0; jb < kChunkBlocks; ++jb) nids[jb] = jb < nblk ? __ldg(tab + jb) : 0;
                for (int j = 0; j < nch; ++j) {
                    const uint32_t c = kc + j, ks = c % kKSt, kph = (c / kKSt) & 1, vs = c % kVSt, vph = (c / kVSt) & 1;
                    const int nb = min(kChunkBlocks, nblk - j * kChunkBlocks);
#pragma unroll
                    for (int jb = 0; jb < kChunkBlocks; ++jb) {
                        ids[jb] = nids[jb];
                        const int nx = (j + 1) * kChunkBlocks + jb;
                        nids[jb] = nx < nblk ? __ldg(tab + nx) : 0;
                    }
                    uint8_t* kb = smem + kOffK2 + ks * 16384;
                    uint8_t* vb = smem + kOffV2 + vs * 16384;
                    mbar_wait(&k_empty[ks], kph ^ 1);
                    mbar_expect_tx(&k_full[ks], (uint32_t)nb * TB);
#pragma unroll
                    for (int jb = 0; jb < kChunkBlocks; ++jb)
                        if (jb < nb) {
                            const uint8_t* src = head_base + (size_t)ids[jb] * blk_stride;
                            bulk_g2s(kb + jb * 2048, src, 2048, &k_full[ks]);
                            bulk_g2s(kb + 8192 + jb * 2048, src + 2048, 2048, &k_full[ks]);
                        }
                    mbar_wait(&v_empty[vs], vph ^ 1);
                    mbar_expect_tx(&v_full[vs], (uint32_t)nb * TB);
#pragma unroll
                    for (int jb = 0; jb < kChunkBlocks; ++jb)
                        if (jb < nb)
                            bulk_g2s(vb + jb * TB, head_base + (size_t)ids[jb] * blk_stride + kv_stride, TB, &v_full[vs]);
                }
            }
        } else if (warp >= 9) {
            // ================= MMA issuers: warp 9 -> tile A, warp 10 -> tile B =================
            constexpr uint32_t idS = idesc_bf16(128, kChunk, 0, 0);
            constexpr uint32_t idO = idesc_bf16(128, D, 0, 1);
            const int t = warp - 9;
            const bool active = t == 0 || hasB;      // an idle issuer still releases the K/V stages
            const uint32_t tc0 = t ? tcnB : tcnA;
            // descriptors are built once; per MMA only (byte offset >> 4) is added to the low word (tc5.cuh)
            const uint64_t qd = smem_desc_sw128(sbase + kOffQ2 + t * 32768, 16, 1024);
            const uint64_t kd = smem_desc_sw128(sbase + kOffK2, 16, 1024);
            const uint64_t vd = smem_desc_sw128(sbase + kOffV2, 2048, 1024);
            // broadcast through a shuffle: tells the compiler these are warp-uniform, so the per-MMA descriptor words are
            // formed on the uniform datapath (UIADD3) instead of one R2UR chain per MMA
            const uint32_t q_lo = __shfl_sync(0xffffffffu, (uint32_t)qd, 0), qk_hi = __shfl_sync(0xffffffffu, (uint32_t)(qd >> 32), 0);
            const uint32_t k_lo = __shfl_sync(0xffffffffu, (uint32_t)kd, 0);
            const uint32_t v_lo = __shfl_sync(0xffffffffu, (uint32_t)vd, 0), v_hi = __shfl_sync(0xffffffffu, (uint32_t)(vd >> 32), 0);
            const uint32_t tm_t = __shfl_sync(0xffffffffu, tmem + t * 256, 0);
            const bool leader = lane == 0;
            auto issue_S = [&](int j) {
                const uint32_t c = kc + j, ks = c % kKSt, kph = (c / kKSt) & 1;
                mbar_wait(&k_full[ks], kph);
                tc_fence_after();
                const uint32_t bt = __shfl_sync(0xffffffffu, (tc0 + j) & 1, 0);
                const uint32_t dS = tm_t + bt * 64, kl = k_lo + __shfl_sync(0xffffffffu, ks, 0) * 1024;
                if (leader) {
                    if (active) {
#pragma unroll
                        for (int hk = 0; hk < 8; ++hk)   // hk = half * 4 + k-step inside the 64-element half
                            mma_ss_lohi(dS, q_lo + (hk >> 2) * 1024 + (hk & 3) * 2, qk_hi, kl + (hk >> 2) * 512 + (hk & 3) * 2,
                                        qk_hi, idS, hk != 0);
                        tc_commit(&s_full[t * 2 + bt]);
                    }
                    tc_commit(&k_empty[ks]);
                }
                __syncwarp();
            };
            issue_S(0);
            for (int j = 0; j < nch; ++j) {
                if (j + 1 < nch) issue_S(j + 1);
                const uint32_t c = kc + j, vs = c % kVSt, vph = (c / kVSt) & 1;
                const int nb = min(kChunkBlocks, nblk - j * kChunkBlocks);
                const uint32_t tcv = tc0 + j, bt = tcv & 1, pht = (tcv >> 1) & 1;
                if (active) mbar_wait(&p_full[t * 2 + bt], pht);
                mbar_wait(&v_full[vs], vph);
                const int tok0 = (blk_begin + j * kChunkBlocks) * 16;
                if (active && tok0 + nb * 16 > kv_len) {   // slots past kv_len may hold NaN patterns: 0 * NaN must not reach O
                    // (both issuers write the same zeros; each fences its own writes before its own MMAs)
                    const int nvalid = kv_len - (tok0 + (nb - 1) * 16);
                    uint8_t* vt = smem + kOffV2 + vs * 16384 + (nb - 1) * TB;
                    for (int cidx = lane; cidx < TB / 16; cidx += 32)
                        if (((cidx & 127) >> 3) >= nvalid) *reinterpret_cast<uint4*>(vt + cidx * 16) = make_uint4(0, 0, 0, 0);
                    fence_proxy_async();
                    __syncwarp();
                }
                tc_fence_after();
                const uint32_t dO = tm_t + 128, aP = tm_t + __shfl_sync(0xffffffffu, bt, 0) * 64;
                const uint32_t vl = v_lo + __shfl_sync(0xffffffffu, vs, 0) * 1024;
                if (leader) {
                    if (active) {
#pragma unroll
                        for (int kk = 0; kk < kChunkBlocks; ++kk)
                            if (kk < nb) mma_ts_lohi(dO, aP + kk * 8, vl + kk * (TB >> 4), v_hi, idO, (j | kk) != 0);
                        tc_commit(&o_done[t]);
                    }
                    tc_commit(&v_empty[vs]);
                }
                __syncwarp();
            }
        } else {
            // ================= softmax: warps 0-3 tile A, warps 4-7 tile B =================
            const int t = warp >> 2;
            if (t == 0 || hasB) {
                const int r = threadIdx.x & 127, sr = row_begin + t * 128 + r;
                const bool ok = sr < rows_total;
                const int lim = ok ? P + sr / G : kv_len - 1;   // last visible key; rows past the chunk see all (Q = 0)
                const uint32_t lane_base = tmem + t * 256 + ((uint32_t)((warp & 3) * 32) << 16);
                const uint32_t tc0 = t ? tcnB : tcnA;
                float m_used = -INFINITY, l_run = 0.f;
                for (int j = 0; j < nch; ++j) {
                    const uint32_t c = tc0 + j, b = c & 1, ph = (c >> 1) & 1;
                    mbar_wait(&s_full[t * 2 + b], ph);
                    tc_fence_after();
                    uint32_t s0[32], s1[32];
                    tmem_ld32(lane_base + b * 64, s0);
                    tmem_ld32(lane_base + b * 64 + 32, s1);
                    tmem_wait_ld();
                    const int tok0 = (blk_begin + j * kChunkBlocks) * 16;
                    const int nb = min(kChunkBlocks, nblk - j * kChunkBlocks);
                    const int nvis = min(lim - tok0 + 1, nb * 16);   // visible columns (<= 0: none); stale columns masked too
                    float x[64];
#pragma unroll
                    for (int k = 0; k < 32; ++k) {
                        x[k] = __uint_as_float(s0[k]);
                        x[32 + k] = __uint_as_float(s1[k]);
                    }
                    if (nvis < kChunk) {
#pragma unroll
                        for (int k = 0; k < 64; ++k)
                            if (k >= nvis) x[k] = -INFINITY;
                    }
                    float mraw = x[0];
#pragma unroll
                    for (int k = 1; k < 63; k += 2) mraw = fmax3(mraw, x[k], x[k + 1]);
                    mraw = fmaxf(mraw, x[63]);
                    const float mx = mraw * p.scale_log2;   // -inf stays -inf
                    bool need = false;
                    float alpha = 1.f;
                    if (j == 0) {
                        m_used = mx;   // PV_0 overwrites O (accumulate = 0): nothing to rescale
                    } else {
                        need = mx > m_used + 8.f;   // lazy rescale: exponents stay below 2^8 otherwise
                        if (need) {
                            alpha = fast_exp2(m_used - mx);   // exp2(-inf) = 0 for a row with no key yet
                            m_used = mx;
                            l_run *= alpha;
                        }
                    }
                    const float ref = m_used == -INFINITY ? 0.f : m_used;
                    // The XU (ex2) pipe of an SM sub-partition is shared by warp w (tile A) and warp w + 4 (tile B).  Left
                    // alone the two drift into running their exponential phases together at half rate each; a token
                    // passed between the pair makes them alternate (A first in every chunk).
                    if (hasB) {
                        if (t == 0) {
                            if (j > 0) asm volatile("bar.sync %0, 64;" ::"r"(1 + (warp & 3)) : "memory");
                        } else {
                            asm volatile("bar.sync %0, 64;" ::"r"(5 + (warp & 3)) : "memory");
                        }
                    }
                    uint32_t pk[32];
                    const float2 sc2 = make_float2(p.scale_log2, p.scale_log2), nref2 = make_float2(-ref, -ref);
                    float2 acc2 = make_float2(0.f, 0.f);
#pragma unroll
                    for (int k = 0; k < 32; ++k) {
                        const float2 tt = ffma2(make_float2(x[2 * k], x[2 * k + 1]), sc2, nref2);
                        const float p0 = fast_exp2(tt.x), p1 = fast_exp2(tt.y);
                        acc2 = fadd2(acc2, make_float2(p0, p1));
                        pk[k] = pack_bf16(p0, p1);
                    }
                    l_run += acc2.x + acc2.y;
                    if (hasB) {
                        if (t == 0) {
                            asm volatile("bar.arrive %0, 64;" ::"r"(5 + (warp & 3)) : "memory");
                        } else if (j + 1 < nch) {
                            asm volatile("bar.arrive %0, 64;" ::"r"(1 + (warp & 3)) : "memory");
                        }
                    }
                    if (j > 0) {
                        mbar_wait(&o_done[t], (c - 1) & 1);   // PV_{j-1} of this tile has finished: O is stable
                        tc_fence_after();
                        if (__any_sync(0xffffffffu, need)) {
#pragma unroll
                            for (int piece = 0; piece < 4; ++piece) {
                                uint32_t o[32];
                                tmem_ld32(lane_base + 128 + piece * 32, o);
                                tmem_wait_ld();
#pragma unroll
                                for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * alpha);
                                tmem_st32(lane_base + 128 + piece * 32, o);
                            }
                            tmem_wait_st();
                        }
                    }
                    tmem_st32(lane_base + b * 64, pk);   // P_j over the first 32 columns of S_j (this lane's row only)
                    tmem_wait_st();
                    tc_fence_before();
                    mbar_arrive(&p_full[t * 2 + b]);
                }
                // ---- epilogue: wait for this tile's last PV, normalise, write ----
                mbar_wait(&o_done[t], (tc0 + nch - 1) & 1);
                tc_fence_after();
                const float inv = direct ? 1.f / l_run : 1.f;
                const size_t orow = (size_t)(q_start + (ok ? sr / G : 0)) * p.Hq + (size_t)head * G + (ok ? sr % G : 0);
                const size_t prow = (size_t)partial * 256 + t * 128 + r;
#pragma unroll
                for (int piece = 0; piece < 4; ++piece) {
                    uint32_t o[32];
                    tmem_ld32(lane_base + 128 + piece * 32, o);
                    tmem_wait_ld();
                    if (direct) {
                        if (ok) {
                            uint4* dst = reinterpret_cast<uint4*>(p.out + orow * D + piece * 32);
#pragma unroll
                            for (int q4 = 0; q4 < 4; ++q4) {
                                uint4 w;
                                w.x = pack_bf16(__uint_as_float(o[8 * q4 + 0]) * inv, __uint_as_float(o[8 * q4 + 1]) * inv);
                                w.y = pack_bf16(__uint_as_float(o[8 * q4 + 2]) * inv, __uint_as_float(o[8 * q4 + 3]) * inv);
                                w.z = pack_bf16(__uint_as_float(o[8 * q4 + 4]) * inv, __uint_as_float(o[8 * q4 + 5]) * inv);
                                w.w = pack_bf16(__uint_as_float(o[8 * q4 + 6]) * inv, __uint_as_float(o[8 * q4 + 7]) * inv);
                                dst[q4] = w;
                            }
                        }
                    } else {
                        uint4* dst = reinterpret_cast<uint4*>(p.po + prow * D + piece * 32);
#pragma unroll
                        for (int q4 = 0; q4 < 8; ++q4) dst[q4] = make_uint4(o[4 * q4], o[4 * q4 + 1], o[4 * q4 + 2], o[4 * q4 + 3]);
                    }
                }
                if (direct) {
                    if (ok) p.lse[orow] = (m_used + log2f(l_run)) * 0.6931471805599453f;
                } else {
                    *reinterpret_cast<float2*>(p.pml + prow * 2) = make_float2(m_used, l_run);
                }
            } else if (!direct) {
                // tile B has no rows in this item: its partial slots must still read as "no key seen"
                const size_t prow = (size_t)partial * 256 + 128 + (threadIdx.x & 127);
                *reinterpret_cast<float2*>(p.pml + prow * 2) = make_float2(-INFINITY, 0.f);
            }
        }
        kc += nch;
        tcnA += nch;
        if (hasB) tcnB += nch;
        tc_fence_before();   // order this item's TMEM traffic before the next item's barrier
        it = it_next;
        par ^= 1;
    }
}
