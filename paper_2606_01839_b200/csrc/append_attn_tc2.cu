// append_attn_tc2.cu — append_prefill_attn for head_dim 128 on tcgen05 / TMEM, two row tiles per CTA.
// PAPER.md:94 §3.1 / PAPER.md:60 §2.2 (see append_attn.cu).  Roofline: tensor (bf16, fp32 accumulate).
//
// One CTA per SM works on 256 stacked rows (token-major: row = token*G + head) of one KV head: two
// 128-row tiles A and B that SHARE every K/V chunk.  Measured on the one-tile-per-CTA predecessor
// (DESIGN.md §5): with two independent CTAs per SM the 2-stage K/V rings gave a stage one softmax
// period of lead (< loaded L2/HBM latency) and every CTA re-read its own K/V.  Here the rings are 4
// deep (two to three periods of lead), K/V traffic per row is halved, and the tensor pipe alternates
// between the two tiles while the other tile's softmax runs.
//   warps 0-3  softmax of tile A, warps 4-7 softmax of tile B (thread r owns row r = TMEM lane r % 128)
//   warp 8     producer: 1-D bulk copies of K half-tiles / V tiles into the rings
//   warps 9,10 MMA issuers, one per tile (one issuer for both tiles serialises their dependent chains: measured 563
//              against 957 TFLOP/s): S_t = Q_t K^T (SS, M=128, N=64), O_t += P_t V (A = P from TMEM)
// TMEM (all 512 columns): tile t at t*256: S/P buffer 0 [0,64), buffer 1 [64,128), O [128,256).
#include <math.h>
#include <stdlib.h>

#include <algorithm>

#include "append_tc2_body.cuh"

namespace {

// ST = depth of the K and V rings (16 KiB stages): 4.  (3 stages, which would leave 64 KB of the SM free, measured 7-20 % slower.)
template <int ST>
__global__ void __launch_bounds__(kT2Threads, 1) append_tc2_kernel(const __grid_constant__ AppendTc2Params p) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t tmem = append_tc2_setup<ST>(smem);
    append_tc2_items<ST>(p, smem, tmem, (int)blockIdx.x, (int)gridDim.x);
    append_tc2_teardown<ST>(tmem);
}

}   // namespace

int launch_append_attn_tc2(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                           int max_blocks, void* out, float* lse, void* stream) {
    const kv_pool_desc& s = pool->desc;
    AppendTc2Params p;
    p.items = reinterpret_cast<const AppendItem*>(plan->d_ws + plan->lay.append_items);
    p.n_items = (int32_t)plan->append_items.size();
    p.pool_layer = pool->d_base + (size_t)layer * s.num_blocks * 2 * s.num_kv_heads * csv_tile_bytes(s.head_dim);
    p.q = (const uint16_t*)q;
    p.tables = tables;
    p.out = (uint16_t*)out;
    p.lse = lse;
    p.po = reinterpret_cast<float*>(plan->d_ws + plan->lay.append_po);
    p.pml = reinterpret_cast<float*>(plan->d_ws + plan->lay.append_pml);
    p.max_blocks = max_blocks;
    p.Hq = plan->shape.num_q_heads;
    p.Hkv = plan->shape.num_kv_heads;
    p.G = p.Hq / p.Hkv;
    p.scale_log2 = (float)(1.4426950408889634 / sqrt((double)s.head_dim));
    p.sched = reinterpret_cast<uint32_t*>(plan->d_ws + plan->lay.append_sched);
    int grid = p.n_items < plan->num_sms ? p.n_items : plan->num_sms;
    // the work queue must start at zero whatever happened to an earlier launch on this plan
    CSV_CUDA_TRY(cudaMemsetAsync(p.sched, 0, 8, (cudaStream_t)stream));
    static PerDeviceOnce attr4;
    CSV_CUDA_TRY(once_per_device(attr4, [] {
        return cudaFuncSetAttribute(append_tc2_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes2(4));
    }));
    append_tc2_kernel<4><<<grid, kT2Threads, smem_bytes2(4), (cudaStream_t)stream>>>(p);
    CSV_CUDA_TRY(cudaGetLastError());
    return CSV_OK;
}
