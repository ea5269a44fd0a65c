// tail_fused.cu — csv_tail_step's attention in ONE launch for a mixed batch at head_dim 128: decode rows and appended
// chunks are work items of one persistent grid (Fig. 5: the collocated iteration runs the
// decode rows and the appended chunks of a decoder in the same step; the decode rows are HBM-bound;
// the chunks only compute their own rows against the cached prefix).
//
// One CTA per SM, 352 threads, the shared-memory footprint of either role (197 KB).  Two queues in the plan workspace:
//   decode SHARES: the decode rows' (conversation, KV head, block) stream cut into n_shares x 8 equal worker shares; a CTA
//     that claims share s runs the 8 warp-workers of decode_worker.cuh on workers [8 s, 8 s + 8) (private 3-stage rings);
//   append ITEMS: the longest-first item list of the two-tile tcgen05 body (append_tc2_body.cuh).
// The first `n_dec` CTAs start on decode shares, the others on append items, and a CTA whose own queue is empty takes work
// from the other one, so the split chosen by the plan (from the two roles' measured per-SM rates, 61-79 GB/s per SM in the
// decode role; HBM saturates near three quarters of the SMs streaming, which is where plan_tail caps the decode side) only
// has to be roughly right and every share is processed whichever CTAs
// run.  (Choosing the decode SMs evenly by SM id instead of by CTA index was measured and is slower: 4.94 against 4.64 ms
// on configs[2].)  Why roles per SM and not both kinds on every SM: the append CTA leaves
// 4 K registers and 30 KB of shared memory on its SM (measured: a co-resident decode CTA would have to fit in 64 registers
// x 64 threads, and with a 64 KB ring it pulls 2.7 TB/s).  Roofline: decode role HBM, append role tensor.
// Results are bit-identical from run to run and under block permutation for a fixed plan: which CTA computes an item or a
// share does not change its arithmetic (S8).
#include <math.h>
#include <stdlib.h>

#include <algorithm>

#include "append_tc2_body.cuh"
#include "decode_worker.cuh"

namespace {

constexpr int kTailDecStages = 3;
constexpr uint32_t kTailDecBarOff = smem_bytes2(4);                       // after the append role's barrier block
constexpr uint32_t kTailSmem = kTailDecBarOff + 8 * kTailDecStages * 8 + 64;
static_assert(8u * kTailDecStages * 2u * 4096u <= AppendTc2Smem<4>::kOffBar2, "decode rings must fit in front of the barrier block");

__global__ void __launch_bounds__(kT2Threads, 1) tail_kernel(const __grid_constant__ AppendTc2Params pa,
                                                             const __grid_constant__ DecodeParams pd, const int n_dec,
                                                             const int n_shares) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t tmem = append_tc2_setup<4>(smem);
    const int warp = threadIdx.x >> 5;
    uint64_t* dec_bars = reinterpret_cast<uint64_t*>(smem + kTailDecBarOff) + warp * kTailDecStages;
    uint32_t* slot = reinterpret_cast<uint32_t*>(smem + kTailDecBarOff + 8 * kTailDecStages * 8);
    uint32_t dec_cnt = 0;   // this warp's ring position across the decode shares it runs
    // plan data only above; tables, Q and the pool may come from the previous kernel (the KV write of this step)
    pdl_wait();
    pdl_trigger();   // the merge kernels may be scheduled; they wait for this grid to finish

    // decode shares until that queue is empty (sched[2] = next unclaimed share)
    auto decode_shares = [&]() {
        for (;;) {
            __syncthreads();   // the rings are free (earlier share or append items done), slot has been read
            if (threadIdx.x == 0) *slot = atomicAdd(pa.sched + 2, 1u);
            __syncthreads();
            const uint32_t sh = *slot;
            if (sh >= (uint32_t)n_shares) break;
            if (warp < 8)
                decode_worker<128, kTailDecStages, false>(pd, (int)sh * 8 + warp, smem + (size_t)warp * kTailDecStages * 8192, dec_bars,
                                                          dec_cnt);
            fence_proxy_async();   // the rings go back to the bulk-copy (async) proxy of whoever uses them next
        }
    };
    if ((int)blockIdx.x < n_dec) decode_shares();   // the first n_dec CTAs start in the decode role
    // append items (sched[0] = next unclaimed item)
    __syncthreads();
    if (threadIdx.x == 0) *slot = atomicAdd(pa.sched, 1u);
    __syncthreads();
    const int it_first = (int)*slot;
    __syncthreads();   // slot is rewritten by the next claim
    append_tc2_items<4>(pa, smem, tmem, it_first, 0);
    // whatever decode shares are left (append-role SMs that ran out of items; SMs the spread did not reach)
    decode_shares();
    append_tc2_teardown<4>(tmem);
}

}   // namespace

int launch_tail_zero_queue(const csv_plan* plan, void* stream) {
    CSV_CUDA_TRY(cudaMemsetAsync(plan->d_ws + plan->lay.append_sched, 0, 16, (cudaStream_t)stream));   // [0] items, [2] shares
    return CSV_OK;
}

int launch_tail_fused(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                      int max_blocks, void* out, float* lse, void* stream, bool pdl) {
    const kv_pool_desc& s = pool->desc;
    const uint8_t* pool_layer = pool->d_base + (size_t)layer * s.num_blocks * 2 * s.num_kv_heads * csv_tile_bytes(s.head_dim);
    const float scale_log2 = (float)(1.4426950408889634 / sqrt((double)s.head_dim));
    AppendTc2Params pa;
    pa.items = reinterpret_cast<const AppendItem*>(plan->d_ws + plan->lay.append_items);
    pa.n_items = (int32_t)plan->append_items.size();
    pa.pool_layer = pool_layer;
    pa.q = (const uint16_t*)q;
    pa.tables = tables;
    pa.out = (uint16_t*)out;
    pa.lse = lse;
    pa.po = reinterpret_cast<float*>(plan->d_ws + plan->lay.append_po);
    pa.pml = reinterpret_cast<float*>(plan->d_ws + plan->lay.append_pml);
    pa.max_blocks = max_blocks;
    pa.Hq = plan->shape.num_q_heads;
    pa.Hkv = plan->shape.num_kv_heads;
    pa.G = pa.Hq / pa.Hkv;
    pa.scale_log2 = scale_log2;
    pa.sched = reinterpret_cast<uint32_t*>(plan->d_ws + plan->lay.append_sched);
    DecodeParams pd;
    pd.items = reinterpret_cast<const DecodeItem*>(plan->d_ws + plan->lay.tail_items);
    pd.worker_begin = reinterpret_cast<const int32_t*>(plan->d_ws + plan->lay.tail_worker_begin);
    pd.pool_layer = pool_layer;
    pd.q = (const uint16_t*)q;
    pd.tables = tables;
    pd.out = (uint16_t*)out;
    pd.lse = lse;
    pd.po = reinterpret_cast<float*>(plan->d_ws + plan->lay.decode_po);
    pd.pml = reinterpret_cast<float*>(plan->d_ws + plan->lay.decode_pml);
    pd.k_new = nullptr;   // the step's KV write is its own kernel in a mixed step (kv_append_tokens)
    pd.v_new = nullptr;
    pd.pool_layer_w = nullptr;
    pd.max_blocks = max_blocks;
    pd.Hq = pa.Hq;
    pd.Hkv = pa.Hkv;
    pd.G = pa.G;
    pd.scale_log2 = scale_log2;
    const int n_dec = plan->tail_n_dec, n_shares = plan->tail_n_shares, grid = plan->num_sms;
    // the work queues must start at zero whatever happened to an earlier launch on this plan; with pdl the caller has
    // enqueued launch_tail_zero_queue BEFORE the kernel this one is chained to (a memset between them would break the chain)
    if (!pdl) {
        const int rz = launch_tail_zero_queue(plan, stream);
        if (rz != CSV_OK) return rz;
    }
    static PerDeviceOnce attr;
    CSV_CUDA_TRY(once_per_device(attr, [] {
        return cudaFuncSetAttribute(tail_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTailSmem);
    }));
    if (pdl)
        CSV_CUDA_TRY(launch_pdl(tail_kernel, dim3(grid), dim3(kT2Threads), kTailSmem, (cudaStream_t)stream, pa, pd, n_dec, n_shares));
    else
        tail_kernel<<<grid, kT2Threads, kTailSmem, (cudaStream_t)stream>>>(pa, pd, n_dec, n_shares);
    CSV_CUDA_TRY(cudaGetLastError());
    // two merges behind it: the decode groups of the tail share list, the append groups
    int rc = launch_decode_merge_128(plan, plan->lay.tail_groups, (int)plan->tail_groups.size(), out, lse, stream);
    if (rc == CSV_OK) rc = launch_append_merge_128(plan, out, lse, stream);
    return rc;
}
