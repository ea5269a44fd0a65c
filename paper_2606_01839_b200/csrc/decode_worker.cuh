// decode_worker.cuh — the warp-worker of paged_decode_attn (a4): one warp streams its share of the flattened
// (conversation, KV head, block) list through a private shared-memory ring.  Used by decode_kernel (decode_attn.cu: every
// warp of the grid is a worker) and by tail_kernel (tail_fused.cu: the warps of the CTAs that take the decode role of a
// mixed step).  See decode_attn.cu for the design notes.
#pragma once
#include <math.h>

#include "common.cuh"
#include "internal.h"

struct DecodeParams {
    const DecodeItem* items;
    const int32_t* worker_begin;
    const uint8_t* pool_layer;   // first tile of this layer
    const uint16_t* q;
    const int32_t* tables;
    uint16_t* out;
    float* lse;
    float* po;
    float* pml;
    const uint8_t* k_new;   // fused step only: this layer's new-token K / V, [total_q][Hkv][d] bf16, else NULL
    const uint8_t* v_new;
    uint8_t* pool_layer_w;  // same address as pool_layer, writable (fused step)
    int32_t max_blocks, Hq, Hkv, G;
    float scale_log2;
};

// worker: index into p.worker_begin; ring: STAGES x (K tile + V tile) of this warp; bars: STAGES mbarriers of this warp.
// PDL: wait for the previous kernel (and let the next one be scheduled) after the first plan reads, as decode_kernel
// does; false when the caller has already done so.
// cnt: blocks this warp has pushed through its ring so far.  A warp that runs several shares (tail_kernel) passes the same
// variable every time: the barriers are initialised on the first call only (cnt == 0) and keep their phase afterwards.
template <int D, int STAGES, bool PDL>
__device__ __forceinline__ void decode_worker(const DecodeParams& p, const int worker, uint8_t* ring, uint64_t* bars, uint32_t& cnt) {
    constexpr int TB = 16 * D * 2;   // tile bytes
    constexpr int KS = D / 16;       // k-steps of Q K^T
    constexpr int NT = D / 8;        // n-tiles of P V
    const int lane = threadIdx.x & 31;
    if (cnt == 0) {
        if (lane == 0) {
            for (int s = 0; s < STAGES; ++s) mbar_init(&bars[s], 1);
            fence_mbar_init();
        }
        __syncwarp();
    }

    const int G = p.G;
    const int row = lane >> 2, t4 = lane & 3;
    const size_t kv_stride = (size_t)p.Hkv * TB;   // K tile -> V tile of the same head
    const size_t blk_stride = 2 * kv_stride;

    // per-lane ldmatrix offsets inside a tile (see conserve_kv.h "Inside a tile")
    const int mi = lane >> 3, r8 = lane & 7;
    const uint32_t k_lane_off = (uint32_t)((r8 + 8 * (mi >> 1)) * 128 + (((mi & 1) ^ r8) << 4));
    const uint32_t v_lane_off = (uint32_t)((r8 + 8 * (mi & 1)) * 128 + (((mi >> 1) ^ r8) << 4));
    const uint32_t ring_u32 = smem_u32(ring);

    const int item_begin = __ldg(p.worker_begin + worker), item_end = __ldg(p.worker_begin + worker + 1);
    int4 c0 = make_int4(0, 0, 0, 0), c1 = c0, c2 = c0, n0 = c0, n1 = c0, n2 = c0;
    if (item_begin < item_end) {
        c0 = __ldg(reinterpret_cast<const int4*>(p.items + item_begin));
        c1 = __ldg(reinterpret_cast<const int4*>(p.items + item_begin) + 1);
        c2 = __ldg(reinterpret_cast<const int4*>(p.items + item_begin) + 2);
    }
    int ids_pref = 0;
    bool have_pref = false;
    if (PDL) {
        // Plan data (work lists) was read above; tables, Q and the pool may come from the previous kernel.
        pdl_wait();
        pdl_trigger();   // decode_merge_kernel may be scheduled now; it waits for this grid to finish
    }
    for (int ii = item_begin; ii < item_end; ++ii) {
        const int conv = c0.x, head = c0.y, blk_begin = c0.z, blk_end = c0.w;
        const int kv_len = c1.x, partial = c1.y, direct = c1.z, q_row = c1.w;
        const int nblk = blk_end - blk_begin;
        const int32_t* tab = p.tables + (size_t)conv * p.max_blocks + blk_begin;
        int ids_cur = have_pref ? ids_pref : (lane < nblk ? __ldg(tab + lane) : 0);
        have_pref = false;
        const bool has_next = ii + 1 < item_end;
        if (has_next) {   // next item's record: lands while this item streams
            n0 = __ldg(reinterpret_cast<const int4*>(p.items + ii + 1));
            n1 = __ldg(reinterpret_cast<const int4*>(p.items + ii + 1) + 1);
            n2 = __ldg(reinterpret_cast<const int4*>(p.items + ii + 1) + 2);
        }
        const int pf_at = nblk > 3 ? nblk - 3 : 0;   // when to fetch the next item's first 32 block ids
        int ids_nxt = 32 + lane < nblk ? __ldg(tab + 32 + lane) : 0;
        int grp_cur = 0;

        // Q fragments: row `row` of the group (zero beyond G); rows 8..15 of the MMA are zero
        uint32_t qa[KS][2];
        {
            const uint16_t* qrow = p.q + ((size_t)q_row * p.Hq + (size_t)head * G + row) * D;
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                qa[ks][0] = row < G ? *reinterpret_cast<const uint32_t*>(qrow + ks * 16 + 2 * t4) : 0u;
                qa[ks][1] = row < G ? *reinterpret_cast<const uint32_t*>(qrow + ks * 16 + 8 + 2 * t4) : 0u;
            }
        }
        float o[NT][2];
#pragma unroll
        for (int n = 0; n < NT; ++n) o[n][0] = o[n][1] = 0.f;
        float m_run = -INFINITY, l_run = 0.f;

        const uint8_t* head_base = p.pool_layer + (size_t)head * TB;
        const uint32_t cnt0 = cnt;
        // prologue: fill the ring
        const int npro = nblk < STAGES ? nblk : STAGES;
        for (int j = 0; j < npro; ++j) {
            const int id = __shfl_sync(0xffffffffu, ids_cur, j);
            if (lane == 0) {
                const uint32_t stage = (cnt0 + j) % STAGES;
                const uint8_t* src = head_base + (size_t)id * blk_stride;
                uint8_t* dst = ring + (size_t)stage * 2 * TB;
                mbar_expect_tx(&bars[stage], 2 * TB);
                bulk_g2s(dst, src, TB, &bars[stage]);
                bulk_g2s(dst + TB, src + kv_stride, TB, &bars[stage]);
            }
        }

        for (int i = 0; i < nblk; ++i) {
            const uint32_t stage = cnt % STAGES, parity = (cnt / STAGES) & 1u;
            mbar_wait(&bars[stage], parity);
            const uint32_t kt = ring_u32 + stage * 2 * TB, vt = kt + TB;
            const int nvalid = kv_len - (blk_begin + i) * 16;   // >= 1; < 16 only in the conversation's last block
            if (p.k_new != nullptr && nvalid <= 16) {
                // Fused tail step ("reading the full KV cache and appending one new entry"): this warp owns
                // the conversation's last block for this head.  The new token's K / V rows go into the landed tiles
                // (so this step attends to them) and into the pool (so the cache has grown).  Nobody else reads this
                // (block, head) in this launch, and the bulk copy that read the old bytes has completed.
                const int slot = nvalid - 1;
                const int c = lane & 15, kv = lane >> 4;   // lanes 0-15: K row chunks, 16-31: V row chunks
                const int id = __shfl_sync(0xffffffffu, ids_cur, i & 31);   // block i is in the current id group
                if (c < D / 8) {
                    const uint4 val = *reinterpret_cast<const uint4*>((kv ? p.v_new : p.k_new) +
                                                                      ((size_t)q_row * p.Hkv + head) * (D * 2) + c * 16);
                    const uint32_t off = (uint32_t)((c >> 3) * 2048 + slot * 128 + (((c & 7) ^ (slot & 7)) << 4));
                    *reinterpret_cast<uint4*>(ring + (size_t)stage * 2 * TB + kv * TB + off) = val;
                    *reinterpret_cast<uint4*>(p.pool_layer_w + (size_t)head * TB + (size_t)id * blk_stride + kv * kv_stride + off) = val;
                }
                fence_proxy_async();
                __syncwarp();
            }
            if (nvalid < 16) {
                // slots past kv_len may hold anything (NaN patterns): 0 * NaN must not reach the PV accumulators
                uint8_t* vtile = ring + (size_t)stage * 2 * TB + TB;
                for (int c = lane; c < TB / 16; c += 32)
                    if (((c & 127) >> 3) >= nvalid) *reinterpret_cast<uint4*>(vtile + c * 16) = make_uint4(0, 0, 0, 0);
                fence_proxy_async();   // these generic writes precede the next bulk copy into this stage
                __syncwarp();
            }
            // S = Q K^T : 16 (G real) rows x 16 tokens
            float s0[2] = {0.f, 0.f}, s1[2] = {0.f, 0.f};
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                uint32_t b[4];
                ldsm_x4(b, kt + (ks >> 2) * 2048 + (k_lane_off ^ (((2 * ks) & 7) << 4)));
                mma_bf16_top(s0, qa[ks][0], qa[ks][1], b[0], b[1]);
                mma_bf16_top(s1, qa[ks][0], qa[ks][1], b[2], b[3]);
            }
            // scale to the log2 domain, mask by index
            float sv[4] = {s0[0] * p.scale_log2, s0[1] * p.scale_log2, s1[0] * p.scale_log2, s1[1] * p.scale_log2};
            if (nvalid < 16) {
                const int c = 2 * t4;
                if (c >= nvalid) sv[0] = -INFINITY;
                if (c + 1 >= nvalid) sv[1] = -INFINITY;
                if (c + 8 >= nvalid) sv[2] = -INFINITY;
                if (c + 9 >= nvalid) sv[3] = -INFINITY;
            }
            float mx = fmaxf(fmaxf(sv[0], sv[1]), fmaxf(sv[2], sv[3]));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
            const float m_new = fmaxf(m_run, mx);   // finite: slot 0 of every block is valid
            if (__any_sync(0xffffffffu, m_new > m_run)) {
                const float alpha = fast_exp2(m_run - m_new);   // exp2(-inf) = 0 on the first block
                l_run *= alpha;
#pragma unroll
                for (int n = 0; n < NT; ++n) {
                    o[n][0] *= alpha;
                    o[n][1] *= alpha;
                }
                m_run = m_new;
            }
            const float p0 = fast_exp2(sv[0] - m_run), p1 = fast_exp2(sv[1] - m_run);
            const float p2 = fast_exp2(sv[2] - m_run), p3 = fast_exp2(sv[3] - m_run);
            l_run += (p0 + p1) + (p2 + p3);
            const uint32_t pa0 = pack_bf16(p0, p1), pa2 = pack_bf16(p2, p3);
            // O += P V
#pragma unroll
            for (int n2 = 0; n2 < NT / 2; ++n2) {
                uint32_t b[4];
                ldsm_x4_trans(b, vt + (n2 >> 2) * 2048 + (v_lane_off ^ (((2 * n2) & 7) << 4)));
                mma_bf16_top(o[2 * n2], pa0, pa2, b[0], b[1]);
                mma_bf16_top(o[2 * n2 + 1], pa0, pa2, b[2], b[3]);
            }
            __syncwarp();   // every lane is done reading this stage
            ++cnt;
            const int nxt = i + STAGES;
            if (nxt < nblk) {
                const int id = (nxt >> 5) == grp_cur ? __shfl_sync(0xffffffffu, ids_cur, nxt & 31)
                                                     : __shfl_sync(0xffffffffu, ids_nxt, nxt & 31);
                if (lane == 0) {
                    const uint8_t* src = head_base + (size_t)id * blk_stride;
                    uint8_t* dst = ring + (size_t)stage * 2 * TB;
                    mbar_expect_tx(&bars[stage], 2 * TB);
                    bulk_g2s(dst, src, TB, &bars[stage]);
                    bulk_g2s(dst + TB, src + kv_stride, TB, &bars[stage]);
                }
            }
            if (i == pf_at && has_next) {
                const int nn = n0.w - n0.z;
                ids_pref = lane < nn ? __ldg(p.tables + (size_t)n0.x * p.max_blocks + n0.z + lane) : 0;
                have_pref = true;
            }
            if (((i + 1) & 31) == 0) {
                ids_cur = ids_nxt;
                ++grp_cur;
                const int e = (grp_cur + 1) * 32 + lane;
                ids_nxt = e < nblk ? __ldg(tab + e) : 0;
            }
        }

        // epilogue
        l_run += __shfl_xor_sync(0xffffffffu, l_run, 1);
        l_run += __shfl_xor_sync(0xffffffffu, l_run, 2);
        if (direct) {
            if (row < G) {
                const float inv = 1.f / l_run;
                uint16_t* orow = p.out + ((size_t)q_row * p.Hq + (size_t)head * G + row) * D;
#pragma unroll
                for (int n = 0; n < NT; ++n)
                    *reinterpret_cast<uint32_t*>(orow + n * 8 + 2 * t4) = pack_bf16(o[n][0] * inv, o[n][1] * inv);
                if (t4 == 0) p.lse[(size_t)q_row * p.Hq + (size_t)head * G + row] = (m_run + log2f(l_run)) * 0.6931471805599453f;
            }
        } else {
            if (row < G) {
                float* orow = p.po + ((size_t)partial * G + row) * D;
#pragma unroll
                for (int n = 0; n < NT; ++n) *reinterpret_cast<float2*>(orow + n * 8 + 2 * t4) = make_float2(o[n][0], o[n][1]);
                if (t4 == 0) *reinterpret_cast<float2*>(p.pml + ((size_t)partial * G + row) * 2) = make_float2(m_run, l_run);
            }
        }
        c0 = n0, c1 = n1, c2 = n2;
    }
}
