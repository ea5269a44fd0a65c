// noalloc.cu — paged_decode_attn_static: paged_decode_attn (a4, §2.1) for callers that have no device
// memory to give the library as a plan workspace and cannot allocate any.
//
// Who that is.  A ConServe decoder hands its whole HBM to the KV pool when it starts (§5.1: a decoder
// holds ~300k tokens of KV), so by the time it serves a step there may be nothing left for cudaMalloc to return;
// and a decode step that lives inside somebody else's engine (a plugin called from a serving loop that owns the
// device allocator) must not call cudaMalloc / cudaFree at all, because both can fail late and both make the
// device wait for every stream.  Every other attention call of this library needs a caller-provided workspace
// (csv_plan_create) for the split-K work lists and the fp32 partial results.  This one keeps that scratch in a
// fixed array that is part of the library image instead.
//
// What it costs.  CSV_STATIC_SCRATCH_BYTES (8 MiB) of device memory on EVERY GPU the process touches with this
// library loaded, from the moment the module is loaded on that GPU until the process exits, whether or not the
// entry point is ever called.  A step whose plan needs more is refused (CSV_E_NOMEM), never truncated.
//
// What is shared.  There is one array per GPU and every call on that GPU uses it from offset 0.  Each call uploads
// its own work lists over whatever the previous call left (queue words included, so nothing has to be cleared by
// hand), and the merge only reads partial slots that the decode kernel of the same call has written, so stale
// contents are harmless.  Two calls that are in flight on one GPU at the same time (different streams, or two
// host threads) overwrite each other's lists and partials: keep calls on one stream, or order them with events.
#include <algorithm>
#include <vector>

#include "common.cuh"
#include "internal.h"

// The scratch itself.  In host code this name is only a handle for cudaGetSymbolAddress: it is not a device
// address and must never be handed to a kernel or to cudaMemcpy as a pointer.
static __device__ __align__(256) uint8_t g_static_scratch[CSV_STATIC_SCRATCH_BYTES];

// Device address of g_static_scratch on the CURRENT device; looked up once per device ordinal.
static int static_scratch_ptr(uint8_t** out) {
    static PerDeviceOnce once;
    static uint8_t* cached[64];
    int dev = 0;
    CSV_CUDA_TRY(cudaGetDevice(&dev));
    uint8_t* fresh = nullptr;
    CSV_CUDA_TRY(once_per_device(once, [&] {
        const cudaError_t e = cudaGetSymbolAddress((void**)&fresh, g_static_scratch);
        if (e == cudaSuccess && dev >= 0 && dev < 64) cached[dev] = fresh;
        return e;
    }));
    *out = (dev >= 0 && dev < 64) ? cached[dev] : fresh;   // ordinals >= 64 are looked up on every call
    return *out ? CSV_OK : csv_set_cuda_error((int)cudaErrorInvalidSymbol);
}

extern "C" int paged_decode_attn_static(const kv_pool_t* pool, int32_t layer, const csv_attn_shape* shape, int32_t batch,
                                        const int32_t* h_kv_lens, int32_t max_partition_tokens, const void* d_q,
                                        const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse,
                                        void* stream) {
    auto aligned = [](const void* p, size_t a) { return ((uintptr_t)p & (a - 1)) == 0; };
    if (!pool || !shape || batch <= 0 || !h_kv_lens) return CSV_E_INVAL;
    if (pool->desc.num_kv_heads != shape->num_kv_heads || pool->desc.head_dim != shape->head_dim ||
        pool->desc.block_size != shape->block_size)
        return CSV_E_INVAL;
    if (layer < 0 || layer >= pool->desc.num_layers) return CSV_E_INVAL;
    if (!d_q || !d_block_tables || !d_out || !d_lse || !aligned(d_q, 16) || !aligned(d_out, 16) || !aligned(d_lse, 4))
        return CSV_E_INVAL;
    int64_t need_blocks = 0;
    for (int b = 0; b < batch; ++b) {
        if (h_kv_lens[b] < 0) return CSV_E_INVAL;
        need_blocks = std::max<int64_t>(need_blocks, ((int64_t)h_kv_lens[b] + CSV_BLOCK_SIZE - 1) / CSV_BLOCK_SIZE);
    }
    if ((int64_t)max_blocks < need_blocks) return CSV_E_INVAL;

    // Host side of the plan (host heap only): every conversation contributes one decode row.
    const std::vector<int32_t> ones((size_t)batch, 1);
    int err = CSV_E_INVAL;
    csv_plan* plan = csv_plan_build_host(shape, ones.data(), h_kv_lens, batch, max_partition_tokens, &err);
    if (!plan) return err;
    int rc = CSV_OK;
    if (plan->lay.total > (size_t)CSV_STATIC_SCRATCH_BYTES) rc = CSV_E_NOMEM;   // the documented limit: refuse, do not truncate
    uint8_t* scratch = nullptr;
    if (rc == CSV_OK) rc = static_scratch_ptr(&scratch);
    if (rc == CSV_OK && !plan->h_image.empty()) {
        // Work lists over the previous call's.  Stream order puts this copy after that call's kernels.  The source is
        // pageable, so the runtime has taken its own copy of it when this returns and the plan may be freed below.
        const cudaError_t e = cudaMemcpyAsync(scratch, plan->h_image.data(), plan->h_image.size(), cudaMemcpyHostToDevice,
                                              (cudaStream_t)stream);
        if (e != cudaSuccess) rc = csv_set_cuda_error((int)e);
    }
    if (rc == CSV_OK) {
        plan->d_ws = scratch;
        rc = launch_decode(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse, stream);
    }
    delete plan;   // launch parameters were passed by value; nothing on the device refers to the host object
    return rc;
}
