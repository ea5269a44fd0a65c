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
//    XOR-swizzled image ldmatrix wants (pool layout, conserve_kv.h).  At d = 128: 7 warps x
//    2 stages x 8 KiB = 112 KiB in flight per SM (Little's law asks for ~45 KiB/SM).  Round 1
//    ran 8 x 3 = 192 KiB: measured slower by 4-8 % on every config: bytes
//    in flight beyond what the latency needs only queue up in the memory system.
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
#include "decode_worker.cuh"
#include "internal.h"

namespace {

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
__global__ void __launch_bounds__(WARPS * 32, 1) decode_kernel(const __grid_constant__ DecodeParams p) {
    constexpr int TB = 16 * D * 2;   // tile bytes
    extern __shared__ __align__(1024) uint8_t smem[];
    const int warp = threadIdx.x >> 5;
    uint8_t* ring = smem + (size_t)warp * STAGES * 2 * TB;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)WARPS * STAGES * 2 * TB) + warp * STAGES;
    uint32_t cnt = 0;
    decode_worker<D, STAGES, true>(p, blockIdx.x * WARPS + warp, ring, bars, cnt);
}

template <int D, int STAGES, int WARPS>
int launch_decode_t(const csv_plan* plan, const DecodeParams& p, cudaStream_t stream) {
    constexpr int TB = 16 * D * 2;
    const size_t smem = (size_t)WARPS * STAGES * 2 * TB + (size_t)WARPS * STAGES * 8;
    static PerDeviceOnce attr;
    CSV_CUDA_TRY(once_per_device(attr, [&] {
        return cudaFuncSetAttribute(decode_kernel<D, STAGES, WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
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

// Merge of the partials of `ng` groups (list at d_groups in the plan workspace), chained to the producing kernel by
// programmatic dependent launch.  Used by paged_decode_attn and by the mixed step's tail_kernel (its own group list).
int launch_decode_merge_128(const csv_plan* plan, size_t groups_off, int ng, void* out, float* lse, void* stream) {
    if (ng <= 0) return CSV_OK;
    const int G = plan->shape.num_q_heads / plan->shape.num_kv_heads;
    CSV_CUDA_TRY(launch_pdl(decode_merge_kernel<128>, dim3((ng * G + 3) / 4), dim3(128), 0, (cudaStream_t)stream,
                            reinterpret_cast<const MergeGroup*>(plan->d_ws + groups_off), ng, G, (int)plan->shape.num_q_heads,
                            reinterpret_cast<const float*>(plan->d_ws + plan->lay.decode_po),
                            reinterpret_cast<const float*>(plan->d_ws + plan->lay.decode_pml), (uint16_t*)out, lse));
    return CSV_OK;
}

// Decode rows on an empty cache: O = 0, LSE = -inf.
int launch_decode_zero_rows(const csv_plan* plan, const kv_pool* pool, void* out, float* lse, void* stream) {
    if (plan->zero_rows.empty()) return CSV_OK;
    CSV_CUDA_TRY(launch_pdl(decode_zero_rows_kernel, dim3((unsigned)plan->zero_rows.size()), dim3(128), 0, (cudaStream_t)stream,
                            reinterpret_cast<const int32_t*>(plan->d_ws + plan->lay.zero_rows),
                            plan->shape.num_q_heads * pool->desc.head_dim, (int)plan->shape.num_q_heads, (uint16_t*)out, lse));
    return CSV_OK;
}

int launch_decode(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                  int max_blocks, void* out, float* lse, void* stream, const void* k_new, const void* v_new) {
    const kv_pool_desc& s = pool->desc;
    {
        const int rc = launch_decode_zero_rows(plan, pool, out, lse, stream);
        if (rc != CSV_OK) return rc;
    }
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
    if (s.head_dim == 128) {
        // 7 warp-workers x 2 ring stages (the measured sweep of workers x stages)
        return launch_decode_t<128, 2, kDecodeWarps128>(plan, p, (cudaStream_t)stream);
    }
    return launch_decode_t<64, 6, 8>(plan, p, (cudaStream_t)stream);
}
