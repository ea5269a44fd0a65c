// decode_attn.cu — paged_decode_attn (a4): split-K flash-decoding over block tables with GQA
// head grouping and a log-sum-exp merge.  PAPER.md:50 §2.1: decode "generates each subsequent
// token by reading the full KV cache"; §3.2: the tail is bandwidth-bound.
//
// Roofline: HBM.  Algorithmic bytes = sum_b kv_len_b * Hkv * d * 2 * 2 per layer.
//
// Design (sm_100a):
//  * The unit of execution is a WARP, not a CTA.  Every warp of the grid is an independent
//    worker with a private ring of STAGES x (K tile + V tile) in shared memory, private
//    mbarriers and its own contiguous share of the flattened (conversation, KV head, block)
//    stream (plan.cpp).  No __syncthreads anywhere; a long conversation never holds a CTA.
//  * Lane 0 feeds the ring with 1-D bulk copies (cp.async.bulk, SASS UBLKCP): one 4 KiB K
//    tile and one 4 KiB V tile per block, each contiguous in HBM and already in the 128-byte
//    XOR-swizzled image ldmatrix wants (pool layout, conserve_kv.h).  8 warps x 3 stages x
//    8 KiB = 192 KiB in flight per SM, well past the ~45 KiB/SM Little's law asks for.
//  * The G query heads of the group are the (zero-padded) M rows of mma.sync.m16n8k16: one
//    K/V tile read serves all G heads.  CUDA-core FMAs would need 2*d*(G+1) lane-ops per
//    512 B of KV, 68-99 % of the FP32 issue rate at G = 8; HMMA makes
//    the arithmetic ~8 % of issue slots so the kernel stays on the HBM roofline.
//  * Online softmax in fp32 in the log2 domain; P rounded to bf16 for the PV product; each
//    partition leaves (o, m, l) fp32 partials, merged in partial-index order (deterministic, no
//    float atomics) by decode_merge_kernel.  (An in-kernel last-arriver merge was measured slower:
//    the __threadfence + atomic per partition cost 12 us on config 2 against 6 us for the launch.)
//    Single-partition (conversation, head) pairs write O / LSE directly.
#include <math.h>
#include <stdlib.h>

#include <algorithm>

#include "common.cuh"
#include "internal.h"

namespace {

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
    int32_t l2_prefetch;   // blocks ahead of the ring that lane 0 asks the L2 to fetch (0 = off)
};

// One warp per (merge group, query head of the group): log-sum-exp merge of the group's partials in
// partial-index order (deterministic, no float atomics).
template <int D>
__global__ void __launch_bounds__(128) decode_merge_kernel(const MergeGroup* __restrict__ groups, int n_groups, int G,
                                                           int Hq, const float* __restrict__ po,
                                                           const float* __restrict__ pml, uint16_t* out, float* lse) {
    constexpr int VEC = D / 32;
    const int w = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    MergeGroup g = {};
    if (w < n_groups * G) g = groups[w / G];   // plan data, not decode_kernel output
    pdl_wait();                                // partials are complete and visible
    if (w >= n_groups * G) return;
    const int hh = w % G;
    float M = -INFINITY;
    for (int k = 0; k < g.count; ++k) M = fmaxf(M, __ldg(pml + ((size_t)(g.first + k) * G + hh) * 2));
    float L = 0.f, acc[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) acc[v] = 0.f;
    for (int k = 0; k < g.count; ++k) {
        const float2 ml = __ldg(reinterpret_cast<const float2*>(pml + ((size_t)(g.first + k) * G + hh) * 2));
        const float wgt = fast_exp2(ml.x - M);
        L += ml.y * wgt;
        const float* src = po + ((size_t)(g.first + k) * G + hh) * D + lane * VEC;
#pragma unroll
        for (int v = 0; v < VEC; ++v) acc[v] += __ldg(src + v) * wgt;
    }
    const float inv = 1.f / L;
    uint16_t* orow = out + ((size_t)g.q_start * Hq + (size_t)g.head * G + hh) * D + lane * VEC;
#pragma unroll
    for (int v = 0; v < VEC; v += 2) *reinterpret_cast<uint32_t*>(orow + v) = pack_bf16(acc[v] * inv, acc[v + 1] * inv);
    if (lane == 0) lse[(size_t)g.q_start * Hq + (size_t)g.head * G + hh] = (M + log2f(L)) * 0.6931471805599453f;
}

// Decode rows on an empty cache (q_len = 1, kv_len = 0): O = 0, LSE = -inf.  One CTA per row.
__global__ void decode_zero_rows_kernel(const int32_t* __restrict__ rows, int row_elems, int Hq, uint16_t* out, float* lse) {
    const int32_t r = rows[blockIdx.x];   // plan data
    pdl_wait();
    for (int i = threadIdx.x; i < row_elems / 2; i += blockDim.x) reinterpret_cast<uint32_t*>(out + (size_t)r * row_elems)[i] = 0u;
    for (int h = threadIdx.x; h < Hq; h += blockDim.x) lse[(size_t)r * Hq + h] = -INFINITY;
}

template <int D, int STAGES, int WARPS>
__global__ void __launch_bounds__(WARPS * 32, WARPS == 8 ? 1 : 512 / (WARPS * 32)) decode_kernel(const __grid_constant__ DecodeParams p) {
    constexpr int TB = 16 * D * 2;   // tile bytes
    constexpr int KS = D / 16;       // k-steps of Q K^T
    constexpr int NT = D / 8;        // n-tiles of P V
    extern __shared__ __align__(1024) uint8_t smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int worker = blockIdx.x * WARPS + warp;
    uint8_t* ring = smem + (size_t)warp * STAGES * 2 * TB;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)WARPS * STAGES * 2 * TB) + warp * STAGES;
    if (lane == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(&bars[s], 1);
        fence_mbar_init();
    }
    __syncwarp();

    const int G = p.G;
    const int row = lane >> 2, t4 = lane & 3;
    const size_t kv_stride = (size_t)p.Hkv * TB;   // K tile -> V tile of the same head
    const size_t blk_stride = 2 * kv_stride;

    // per-lane ldmatrix offsets inside a tile (see conserve_kv.h "Inside a tile")
    const int mi = lane >> 3, r8 = lane & 7;
    const uint32_t k_lane_off = (uint32_t)((r8 + 8 * (mi >> 1)) * 128 + (((mi & 1) ^ r8) << 4));
    const uint32_t v_lane_off = (uint32_t)((r8 + 8 * (mi & 1)) * 128 + (((mi >> 1) ^ r8) << 4));
    const uint32_t ring_u32 = smem_u32(ring);

    uint32_t cnt = 0;   // blocks consumed so far by this warp (ring position)
    const int item_begin = __ldg(p.worker_begin + worker), item_end = __ldg(p.worker_begin + worker + 1);
    int4 c0 = make_int4(0, 0, 0, 0), c1 = c0, c2 = c0, n0 = c0, n1 = c0, n2 = c0;
    if (item_begin < item_end) {
        c0 = __ldg(reinterpret_cast<const int4*>(p.items + item_begin));
        c1 = __ldg(reinterpret_cast<const int4*>(p.items + item_begin) + 1);
        c2 = __ldg(reinterpret_cast<const int4*>(p.items + item_begin) + 2);
    }
    int ids_pref = 0;
    bool have_pref = false;
    // Plan data (work lists) was read above; tables, Q and the pool may come from the previous kernel.
    pdl_wait();
    pdl_trigger();   // decode_merge_kernel may be scheduled now; it waits for this grid to finish
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
            if (p.l2_prefetch > 0) {
                // the shared-memory ring covers the L2 -> SM latency only; the HBM -> L2 leg is started l2_prefetch blocks early
                const int far = nxt + p.l2_prefetch;
                if (far < nblk && (far >> 5) <= grp_cur + 1) {
                    const int id = (far >> 5) == grp_cur ? __shfl_sync(0xffffffffu, ids_cur, far & 31)
                                                         : __shfl_sync(0xffffffffu, ids_nxt, far & 31);
                    if (lane == 0) {
                        const uint8_t* src = head_base + (size_t)id * blk_stride;
                        l2_prefetch(src, TB);
                        l2_prefetch(src + kv_stride, TB);
                    }
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

template <int D, int STAGES, int WARPS>
int launch_decode_t(const csv_plan* plan, const DecodeParams& p, cudaStream_t stream) {
    constexpr int TB = 16 * D * 2;
    const size_t smem = (size_t)WARPS * STAGES * 2 * TB + (size_t)WARPS * STAGES * 8;
    static PerDeviceOnce attr;
    CSV_CUDA_TRY(once_per_device(attr, [&] {
        cudaError_t e = cudaFuncSetAttribute(decode_kernel<D, STAGES, WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        // the slim variant runs BESIDE the append CTA: the SM must be carved for both kernels' shared memory at once
        if (e == cudaSuccess && WARPS != 8)
            e = cudaFuncSetAttribute(decode_kernel<D, STAGES, WARPS>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        return e;
    }));
    CSV_CUDA_TRY(launch_pdl(decode_kernel<D, STAGES, WARPS>, dim3(plan->decode_grid), dim3(WARPS * 32), smem, stream, p));
    const int ng = (int)plan->decode_groups.size();
    if (ng > 0) {
        const int warps = ng * p.G;
        CSV_CUDA_TRY(launch_pdl(decode_merge_kernel<D>, dim3((warps + 3) / 4), dim3(128), 0, stream,
                                reinterpret_cast<const MergeGroup*>(plan->d_ws + plan->lay.decode_groups), ng, p.G, p.Hq,
                                (const float*)p.po, (const float*)p.pml, p.out, p.lse));
    }
    return CSV_OK;
}

}   // namespace

int launch_decode(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                  int max_blocks, void* out, float* lse, void* stream, const void* k_new, const void* v_new) {
    const kv_pool_desc& s = pool->desc;
    if (!plan->zero_rows.empty())
        CSV_CUDA_TRY(launch_pdl(decode_zero_rows_kernel, dim3((unsigned)plan->zero_rows.size()), dim3(128), 0, (cudaStream_t)stream,
                                reinterpret_cast<const int32_t*>(plan->d_ws + plan->lay.zero_rows),
                                plan->shape.num_q_heads * s.head_dim, plan->shape.num_q_heads, (uint16_t*)out, lse));
    if (plan->decode_items.empty()) return CSV_OK;
    DecodeParams p;
    p.items = reinterpret_cast<const DecodeItem*>(plan->d_ws + plan->lay.decode_items);
    p.worker_begin = reinterpret_cast<const int32_t*>(plan->d_ws + plan->lay.worker_begin);
    p.pool_layer = pool->d_base + (size_t)layer * s.num_blocks * 2 * s.num_kv_heads * csv_tile_bytes(s.head_dim);
    p.q = (const uint16_t*)q;
    p.tables = tables;
    p.out = (uint16_t*)out;
    p.lse = lse;
    p.po = reinterpret_cast<float*>(plan->d_ws + plan->lay.decode_po);
    p.pml = reinterpret_cast<float*>(plan->d_ws + plan->lay.decode_pml);
    p.k_new = (const uint8_t*)k_new;
    p.v_new = (const uint8_t*)v_new;
    p.pool_layer_w = const_cast<uint8_t*>(p.pool_layer);
    p.max_blocks = max_blocks;
    p.Hq = plan->shape.num_q_heads;
    p.Hkv = plan->shape.num_kv_heads;
    p.G = p.Hq / p.Hkv;
    p.scale_log2 = (float)(1.4426950408889634 / sqrt((double)s.head_dim));
    p.l2_prefetch = 0;
    if (const char* e = getenv("CSV_X_DECODE_PF")) p.l2_prefetch = std::max(0, std::min(24, atoi(e)));   // experiment knob
    if (s.head_dim == 128) {
        if (plan->decode_warps == 2) return launch_decode_t<128, 4, 2>(plan, p, (cudaStream_t)stream);
        return launch_decode_t<128, 3, 8>(plan, p, (cudaStream_t)stream);
    }
    return launch_decode_t<64, 6, 8>(plan, p, (cudaStream_t)stream);
}
