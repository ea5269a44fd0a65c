// api.cu — the extern "C" entry points of include/conserve_kv.h that touch CUDA: argument
// validation, plan upload, launches, and the host-buffer tail step.  No kernels here.
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <new>
#include <vector>

#include "common.cuh"
#include "internal.h"

static thread_local int g_last_cuda_error = 0;
int csv_set_cuda_error(int err) {
    g_last_cuda_error = err;
    return CSV_E_CUDA;
}

int csv_query_num_sms() {
    // per device: a process may drive several GPUs (conserve_kv.h "Devices")
    static std::atomic<int> cached[64];
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return 148;   // B200; lets the planner run on a box without a GPU (host tests, host-only plans)
    }
    const bool slot = dev >= 0 && dev < 64;
    if (slot && (n = cached[dev].load(std::memory_order_relaxed)) > 0) return n;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
        (void)cudaGetLastError();
        return 148;
    }
    if (slot) cached[dev].store(n, std::memory_order_relaxed);
    return n;
}

static bool aligned(const void* p, size_t a) { return ((uintptr_t)p & (a - 1)) == 0; }

static bool same_shape(const kv_pool_desc& a, const csv_attn_shape& s) {
    return a.num_kv_heads == s.num_kv_heads && a.head_dim == s.head_dim && a.block_size == s.block_size;
}

extern "C" {

int csv_last_cuda_error(void) { return g_last_cuda_error; }

size_t kv_staging_bytes(const kv_pool_desc* shape, int32_t tokens, int32_t token_offset) {
    if (!csv_shape_ok(shape, false) || tokens <= 0 || token_offset < 0) return 0;
    const int slot0 = token_offset & 15;
    const size_t ntb = (size_t)(slot0 + tokens + 15) / 16;
    return (size_t)shape->num_layers * ntb * 2u * shape->num_kv_heads * csv_tile_bytes(shape->head_dim);
}

int kv_pack_batch(const kv_pool_desc* shape, int32_t n, const void* const* h_d_k, const void* const* h_d_v,
                  const int32_t* h_tokens, const int32_t* h_token_offsets, void* const* h_d_staging, void* stream) {
    if (!csv_shape_ok(shape, false) || n < 0) return CSV_E_INVAL;
    if (n > 0 && (!h_d_k || !h_d_v || !h_tokens || !h_token_offsets || !h_d_staging)) return CSV_E_INVAL;
    for (int i = 0; i < n; ++i) {
        if (h_tokens[i] < 0 || h_token_offsets[i] < 0) return CSV_E_INVAL;
        if (h_tokens[i] == 0) continue;
        if (!h_d_k[i] || !h_d_v[i] || !h_d_staging[i]) return CSV_E_INVAL;
        if (!aligned(h_d_k[i], 16) || !aligned(h_d_v[i], 16) || !aligned(h_d_staging[i], 128)) return CSV_E_INVAL;
    }
    return launch_pack(*shape, n, h_d_k, h_d_v, h_tokens, h_token_offsets, h_d_staging, stream);
}

int kv_pack(const kv_pool_desc* shape, const void* d_k, const void* d_v, int32_t tokens, int32_t token_offset,
            void* d_staging, void* stream) {
    if (tokens <= 0) return CSV_E_INVAL;
    return kv_pack_batch(shape, 1, &d_k, &d_v, &tokens, &token_offset, &d_staging, stream);
}

int kv_unpack_batch(kv_pool_t* dst, int32_t n, const void* const* h_d_staging, const int32_t* h_tokens,
                    const int32_t* h_token_offsets, const int32_t* const* h_d_block_ids, const int32_t* h_n_ids,
                    void* stream) {
    if (!dst || n < 0) return CSV_E_INVAL;
    if (n > 0 && (!h_d_staging || !h_tokens || !h_token_offsets || !h_d_block_ids || !h_n_ids)) return CSV_E_INVAL;
    for (int i = 0; i < n; ++i) {
        if (h_tokens[i] < 0 || h_token_offsets[i] < 0) return CSV_E_INVAL;
        if (h_tokens[i] == 0) continue;
        if (!h_d_staging[i] || !h_d_block_ids[i] || !aligned(h_d_staging[i], 128) || !aligned(h_d_block_ids[i], 4))
            return CSV_E_INVAL;
        const int64_t need = ((int64_t)h_token_offsets[i] + h_tokens[i] + 15) / 16;
        if ((int64_t)h_n_ids[i] < need) return CSV_E_INVAL;
    }
    return launch_unpack(dst, n, h_d_staging, h_tokens, h_token_offsets, h_d_block_ids, stream);
}

int kv_unpack(kv_pool_t* dst, const void* d_staging, int32_t tokens, int32_t token_offset, const int32_t* d_block_ids,
              int32_t n_ids, void* stream) {
    if (tokens <= 0) return CSV_E_INVAL;
    return kv_unpack_batch(dst, 1, &d_staging, &tokens, &token_offset, &d_block_ids, &n_ids, stream);
}

int kv_handoff_direct_batch(kv_pool_t* dst, int32_t n, const void* const* h_d_k, const void* const* h_d_v,
                            const int32_t* h_tokens, const int32_t* h_token_offsets,
                            const int32_t* const* h_d_block_ids, const int32_t* h_n_ids, void* stream) {
    if (!dst || n < 0) return CSV_E_INVAL;
    if (n > 0 && (!h_d_k || !h_d_v || !h_tokens || !h_token_offsets || !h_d_block_ids || !h_n_ids)) return CSV_E_INVAL;
    for (int i = 0; i < n; ++i) {
        if (h_tokens[i] < 0 || h_token_offsets[i] < 0) return CSV_E_INVAL;
        if (h_tokens[i] == 0) continue;
        if (!h_d_k[i] || !h_d_v[i] || !h_d_block_ids[i]) return CSV_E_INVAL;
        if (!aligned(h_d_k[i], 16) || !aligned(h_d_v[i], 16) || !aligned(h_d_block_ids[i], 4)) return CSV_E_INVAL;
        const int64_t need = ((int64_t)h_token_offsets[i] + h_tokens[i] + 15) / 16;
        if ((int64_t)h_n_ids[i] < need) return CSV_E_INVAL;
    }
    return launch_handoff_direct(dst, n, h_d_k, h_d_v, h_tokens, h_token_offsets, h_d_block_ids, stream);
}

int kv_handoff_direct(kv_pool_t* dst, const void* d_k, const void* d_v, int32_t tokens, int32_t token_offset,
                      const int32_t* d_block_ids, int32_t n_ids, void* stream) {
    if (tokens <= 0) return CSV_E_INVAL;
    return kv_handoff_direct_batch(dst, 1, &d_k, &d_v, &tokens, &token_offset, &d_block_ids, &n_ids, stream);
}

// ---- peer mapping of a decoder's pool (one process per GPU: CUDA IPC) ----
// cuMemGetAddressRange comes from the driver through the runtime's entry-point query: the library links no libcuda.
typedef int (*cu_get_range_fn)(unsigned long long*, size_t*, unsigned long long);

static cu_get_range_fn driver_get_range() {
    static cu_get_range_fn fn = nullptr;
    if (!fn) {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult st;
        if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &f, cudaEnableDefault, &st) == cudaSuccess &&
            st == cudaDriverEntryPointSuccess)
            fn = (cu_get_range_fn)f;
    }
    return fn;
}

// One entry per allocation opened in this process.  The driver refuses to map the same handle twice, and several
// exported pointers often share one cudaMalloc allocation (the caller's caching allocator), so opens are counted.
struct ipc_region {
    uint8_t handle[CSV_IPC_HANDLE_BYTES];
    int device;                 // the device that was current at the open: the mapping belongs to its context
    void* base;                 // what cudaIpcOpenMemHandle returned
    std::vector<void*> users;   // pointers csv_ipc_open handed out (base + offset), one per open
};
static std::vector<ipc_region> g_ipc;   // host calls are thread-compatible, not thread-safe (header)

int csv_ipc_export(const void* d_ptr, void* out_handle, uint64_t* out_offset) {
    if (!d_ptr || !out_handle || !out_offset) return CSV_E_INVAL;
    static_assert(sizeof(cudaIpcMemHandle_t) == CSV_IPC_HANDLE_BYTES, "handle size");
    cu_get_range_fn get_range = driver_get_range();
    if (!get_range) return csv_set_cuda_error((int)cudaErrorNotSupported);
    unsigned long long base = 0;
    size_t size = 0;
    if (get_range(&base, &size, (unsigned long long)(uintptr_t)d_ptr) != 0) return csv_set_cuda_error((int)cudaErrorInvalidValue);
    cudaIpcMemHandle_t h;
    CSV_CUDA_TRY(cudaIpcGetMemHandle(&h, (void*)(uintptr_t)base));
    memcpy(out_handle, &h, sizeof(h));
    *out_offset = (uint64_t)((uintptr_t)d_ptr - (uintptr_t)base);
    return CSV_OK;
}

int csv_ipc_open(const void* handle, uint64_t offset, void** out_d_ptr) {
    if (!handle || !out_d_ptr) return CSV_E_INVAL;
    int dev = 0;
    CSV_CUDA_TRY(cudaGetDevice(&dev));
    for (ipc_region& r : g_ipc) {
        if (r.device == dev && memcmp(r.handle, handle, CSV_IPC_HANDLE_BYTES) == 0) {
            r.users.push_back((uint8_t*)r.base + offset);
            *out_d_ptr = r.users.back();
            return CSV_OK;
        }
    }
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, sizeof(h));
    void* base = nullptr;
    CSV_CUDA_TRY(cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
    ipc_region r;
    memcpy(r.handle, handle, CSV_IPC_HANDLE_BYTES);
    r.device = dev;
    r.base = base;
    r.users.push_back((uint8_t*)base + offset);
    *out_d_ptr = r.users.back();
    g_ipc.push_back(r);
    return CSV_OK;
}

int csv_ipc_close(void* d_ptr) {
    for (size_t i = 0; i < g_ipc.size(); ++i) {
        std::vector<void*>& u = g_ipc[i].users;
        for (size_t k = 0; k < u.size(); ++k) {
            if (u[k] != d_ptr) continue;
            u.erase(u.begin() + (long)k);
            if (u.empty()) {
                void* base = g_ipc[i].base;
                const int owner = g_ipc[i].device;
                g_ipc.erase(g_ipc.begin() + (long)i);
                int cur = 0;
                CSV_CUDA_TRY(cudaGetDevice(&cur));
                if (cur != owner) CSV_CUDA_TRY(cudaSetDevice(owner));
                const cudaError_t ce = cudaIpcCloseMemHandle(base);
                if (cur != owner) CSV_CUDA_TRY(cudaSetDevice(cur));
                if (ce != cudaSuccess) return csv_set_cuda_error((int)ce);
            }
            return CSV_OK;
        }
    }
    return CSV_E_INVAL;
}

int csv_ipc_mapped_bytes(const void* d_ptr, size_t* out_bytes) {
    if (!d_ptr || !out_bytes) return CSV_E_INVAL;
    for (const ipc_region& r : g_ipc)
        for (void* u : r.users) {
            if (u != d_ptr) continue;
            cu_get_range_fn get_range = driver_get_range();
            if (!get_range) return csv_set_cuda_error((int)cudaErrorNotSupported);
            unsigned long long base = 0;
            size_t size = 0;
            if (get_range(&base, &size, (unsigned long long)(uintptr_t)r.base) != 0)
                return csv_set_cuda_error((int)cudaErrorInvalidValue);
            const uintptr_t end = (uintptr_t)base + size;
            *out_bytes = (uintptr_t)d_ptr < end ? (size_t)(end - (uintptr_t)d_ptr) : 0;   // an offset past the end leaves nothing
            return CSV_OK;
        }
    return CSV_E_INVAL;
}

int csv_ipc_copy(void* d_dst, const void* d_src, size_t bytes, void* stream) {
    if (!d_dst || !d_src) return CSV_E_INVAL;
    if (bytes == 0) return CSV_OK;
    CSV_CUDA_TRY(cudaMemcpyAsync(d_dst, d_src, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return CSV_OK;
}

// Points a host-built plan at its device workspace and enqueues the upload of its work lists.
static int plan_attach(csv_plan* p, void* d_workspace, size_t ws_bytes, void* stream) {
    if (!aligned(d_workspace, 128)) return CSV_E_INVAL;
    if (ws_bytes < p->lay.total) return CSV_E_NOMEM;
    p->d_ws = (uint8_t*)d_workspace;
    if (!p->h_image.empty()) {
        // pageable source: the runtime stages it before returning, so h_image may be reused freely
        cudaError_t e = cudaMemcpyAsync(d_workspace, p->h_image.data(), p->h_image.size(), cudaMemcpyHostToDevice,
                                        (cudaStream_t)stream);
        if (e != cudaSuccess) return csv_set_cuda_error((int)e);
    }
    return CSV_OK;
}

int csv_plan_create(const csv_attn_shape* shape, const int32_t* h_q_lens, const int32_t* h_kv_lens, int32_t batch,
                    int32_t max_partition_tokens, void* d_workspace, size_t ws_bytes, void* stream, csv_plan_t** out) {
    if (!out) return CSV_E_INVAL;
    int err;
    csv_plan* p = csv_plan_build_host(shape, h_q_lens, h_kv_lens, batch, max_partition_tokens, &err);
    if (!p) return err;
    if (d_workspace) {
        const int rc = plan_attach(p, d_workspace, ws_bytes, stream);
        if (rc != CSV_OK) {
            delete p;
            return rc;
        }
    }
    *out = p;
    return CSV_OK;
}

static int check_attn_args(const csv_plan_t* plan, const kv_pool_t* pool, int32_t layer, const void* d_q,
                           const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse) {
    if (!plan || !pool || !plan->d_ws) return CSV_E_INVAL;
    if (!same_shape(pool->desc, plan->shape)) return CSV_E_INVAL;
    if (layer < 0 || layer >= pool->desc.num_layers) return CSV_E_INVAL;
    if (!d_q || !d_block_tables || !d_out || !d_lse || !aligned(d_q, 16) || !aligned(d_out, 16) || !aligned(d_lse, 4))
        return CSV_E_INVAL;
    int64_t need = 0;
    for (int b = 0; b < plan->batch; ++b)
        if (plan->q_lens[(size_t)b] > 0) need = std::max<int64_t>(need, ((int64_t)plan->kv_lens[(size_t)b] + 15) / 16);
    if ((int64_t)max_blocks < need) return CSV_E_INVAL;
    return CSV_OK;
}

int paged_decode_attn(const csv_plan_t* plan, const kv_pool_t* pool, int32_t layer, const void* d_q,
                      const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse, void* stream) {
    const int rc = check_attn_args(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse);
    if (rc != CSV_OK) return rc;
    return launch_decode(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse, stream);
}

int paged_decode_step(const csv_plan_t* plan, kv_pool_t* pool, int32_t layer, const void* d_q, const void* d_k_new,
                      const void* d_v_new, const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse,
                      void* stream) {
    const int rc = check_attn_args(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse);
    if (rc != CSV_OK) return rc;
    if (!d_k_new || !d_v_new || !aligned(d_k_new, 16) || !aligned(d_v_new, 16)) return CSV_E_INVAL;
    return launch_decode(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse, stream, d_k_new, d_v_new);
}

int append_prefill_attn(const csv_plan_t* plan, const kv_pool_t* pool, int32_t layer, const void* d_q,
                        const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse, void* stream) {
    const int rc = check_attn_args(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse);
    if (rc != CSV_OK) return rc;
    return launch_append_attn(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse, stream);
}

int kv_append_tokens(kv_pool_t* dst, const csv_plan_t* plan, const void* d_k_new, const void* d_v_new,
                     const int32_t* d_block_tables, int32_t max_blocks, void* stream) {
    if (!dst || !plan || !plan->d_ws || !same_shape(dst->desc, plan->shape)) return CSV_E_INVAL;
    if (plan->total_q == 0) return CSV_OK;
    if (!d_k_new || !d_v_new || !d_block_tables || !aligned(d_k_new, 16) || !aligned(d_v_new, 16)) return CSV_E_INVAL;
    int64_t need = 0;
    for (int b = 0; b < plan->batch; ++b)
        if (plan->q_lens[(size_t)b] > 0) need = std::max<int64_t>(need, ((int64_t)plan->kv_lens[(size_t)b] + 15) / 16);
    if ((int64_t)max_blocks < need) return CSV_E_INVAL;
    return launch_append_tokens(dst, plan, d_k_new, d_v_new, d_block_tables, max_blocks, stream);
}

// The layer `layer` of a pool as a 1-layer pool (descriptor + base only; the allocator state is neither copied nor used).
static kv_pool layer_view_of(const kv_pool* pool, int layer) {
    kv_pool v;
    v.desc = pool->desc;
    v.desc.num_layers = 1;
    v.bytes = 0;
    v.used = 0;
    v.d_base = pool->d_base + (size_t)layer * pool->desc.num_blocks * 2 * pool->desc.num_kv_heads *
                                  csv_tile_bytes(pool->desc.head_dim);
    return v;
}

int csv_tail_step(const csv_plan_t* plan, kv_pool_t* pool, int32_t layer, const void* d_q, const void* d_k_new,
                  const void* d_v_new, const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse,
                  void* stream) {
    const int rc = check_attn_args(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse);
    if (rc != CSV_OK) return rc;
    const bool write_kv = d_k_new != nullptr || d_v_new != nullptr;   // both NULL: attention only (the rows are in the pool)
    if (write_kv && (!d_k_new || !d_v_new || !aligned(d_k_new, 16) || !aligned(d_v_new, 16))) return CSV_E_INVAL;
    if (plan->append_items.empty())   // decode rows only: the KV write rides in the decode launch
        return launch_decode(plan, pool, layer, d_q, d_block_tables, max_blocks, d_out, d_lse, stream, d_k_new, d_v_new);
    kv_pool view = layer_view_of(pool, layer);
    const bool fuse = plan->tail_n_dec > 0 && !plan->tail_two_kernels;   // tuning override recorded in the plan (csv_tuning_set)
    int r = CSV_OK;
    if (fuse && write_kv) r = launch_tail_zero_queue(plan, stream);
    if (r == CSV_OK && write_kv) r = launch_append_tokens(&view, plan, d_k_new, d_v_new, d_block_tables, max_blocks, stream);
    if (r != CSV_OK) return r;
    if (fuse) {
        // decode rows and appended chunks as work items of ONE persistent launch (tail_fused.cu)
        r = launch_tail_fused(plan, &view, 0, d_q, d_block_tables, max_blocks, d_out, d_lse, stream, write_kv);
        if (r == CSV_OK && !plan->zero_rows.empty()) r = launch_decode_zero_rows(plan, &view, d_out, d_lse, stream);
        return r;
    }
    r = launch_decode(plan, &view, 0, d_q, d_block_tables, max_blocks, d_out, d_lse, stream);
    if (r == CSV_OK) r = launch_append_attn(plan, &view, 0, d_q, d_block_tables, max_blocks, d_out, d_lse, stream);
    return r;
}

// ---- host-buffer tail step (bench.py "e2e") ---------------------------------------------------
struct TailLayout {
    size_t plan, q, k, v, tables, out, lse, total;
};
static TailLayout tail_layout(const csv_attn_shape* s, int64_t rows, int batch, int max_blocks, size_t plan_bytes) {
    TailLayout L;
    size_t off = 0;
    auto take = [&](size_t b) {
        const size_t at = off;
        off = (off + b + 127) / 128 * 128;
        return at;
    };
    L.q = take((size_t)rows * s->num_q_heads * s->head_dim * 2);
    L.k = take((size_t)rows * s->num_kv_heads * s->head_dim * 2);
    L.v = take((size_t)rows * s->num_kv_heads * s->head_dim * 2);
    L.tables = take((size_t)batch * max_blocks * 4);
    L.out = take((size_t)rows * s->num_q_heads * s->head_dim * 2);
    L.lse = take((size_t)rows * s->num_q_heads * 4);
    L.plan = take(plan_bytes);   // last: its size is only known once the plan is built
    L.total = off;
    return L;
}

static int64_t host_step_rows(const int32_t* h_q_lens, int32_t batch) {   // total_q of one layer; -1 = bad lengths
    if (!h_q_lens) return batch;
    int64_t t = 0;
    for (int b = 0; b < batch; ++b) {
        if (h_q_lens[b] < 0) return -1;
        t += h_q_lens[b];
    }
    return t;
}

size_t csv_tail_step_host_workspace_bytes(const csv_attn_shape* shape, const int32_t* h_q_lens, const int32_t* h_kv_lens,
                                          int32_t batch, int32_t max_blocks, int32_t n_layers, int32_t max_partition_tokens) {
    if (!shape || batch <= 0 || max_blocks <= 0 || n_layers <= 0 || !h_kv_lens) return 0;
    const int64_t rows = host_step_rows(h_q_lens, batch);
    if (rows <= 0) return 0;
    std::vector<int32_t> ones;
    if (!h_q_lens) ones.assign((size_t)batch, 1);
    const size_t pb = csv_plan_workspace_bytes(shape, h_q_lens ? h_q_lens : ones.data(), h_kv_lens, batch, max_partition_tokens);
    if (pb == 0) return 0;
    return tail_layout(shape, rows * n_layers, batch, max_blocks, pb).total;
}

int csv_tail_step_host(kv_pool_t* pool, int32_t layer_begin, int32_t n_layers, const csv_attn_shape* shape, int32_t batch,
                       const int32_t* h_q_lens, const int32_t* h_kv_lens, const void* h_q, const void* h_k_new,
                       const void* h_v_new, const int32_t* h_block_tables, int32_t max_blocks, int32_t max_partition_tokens,
                       void* d_workspace, size_t ws_bytes, void* h_out, float* h_lse, void* stream) {
    if (!pool || !shape || batch <= 0 || n_layers <= 0 || !h_kv_lens || !h_q || !h_k_new || !h_v_new || !h_block_tables ||
        !h_out || !h_lse || !d_workspace || !aligned(d_workspace, 128) || max_blocks <= 0)
        return CSV_E_INVAL;
    if (layer_begin < 0 || layer_begin + (int64_t)n_layers > pool->desc.num_layers || !same_shape(pool->desc, *shape))
        return CSV_E_INVAL;
    if (shape->num_q_heads <= 0 || shape->num_q_heads % shape->num_kv_heads != 0) return CSV_E_INVAL;
    const int64_t rows = host_step_rows(h_q_lens, batch);   // per layer
    if (rows <= 0 || rows * n_layers > INT32_MAX) return CSV_E_INVAL;
    // Everything csv_plan_build_host would refuse is refused HERE, before the first copy is enqueued: a CSV_E_INVAL must
    // not leave DMA from the caller's host buffers in flight (the plan itself is still built under the copies, below).
    {
        const int g = shape->num_q_heads / shape->num_kv_heads;
        if (g != 1 && g != 2 && g != 4 && g != 8) return CSV_E_INVAL;
        if (max_partition_tokens < 0 || max_partition_tokens % CSV_BLOCK_SIZE != 0) return CSV_E_INVAL;
        for (int b = 0; b < batch; ++b) {
            const int32_t q = h_q_lens ? h_q_lens[b] : 1, kv = h_kv_lens[b];
            if (kv < 0 || q < 0 || (q > kv && !(q == 1 && kv == 0))) return CSV_E_INVAL;
        }
    }
    // The plan's size is not known before it is built, so the fixed-size buffers sit in front of it: their copies
    // are enqueued first and fly while the host plans.
    const size_t q_layer = (size_t)rows * shape->num_q_heads * shape->head_dim * 2;
    const size_t k_layer = (size_t)rows * shape->num_kv_heads * shape->head_dim * 2;
    const size_t lse_layer = (size_t)rows * shape->num_q_heads * 4;
    const TailLayout L = tail_layout(shape, rows * n_layers, batch, max_blocks, 0);   // L.plan is the END region here
    if (ws_bytes < L.total) return CSV_E_NOMEM;
    uint8_t* ws = (uint8_t*)d_workspace;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(ws + L.q, h_q, q_layer * n_layers, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ws + L.k, h_k_new, k_layer * n_layers, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ws + L.v, h_v_new, k_layer * n_layers, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ws + L.tables, h_block_tables, (size_t)batch * max_blocks * 4, cudaMemcpyHostToDevice, st)) !=
            cudaSuccess) {
        (void)cudaStreamSynchronize(st);   // some copies may be in flight: the caller's buffers are free again on return
        return csv_set_cuda_error((int)e);
    }
    // One plan serves every layer of the step (lengths are per step, not per layer).  It is built here, while the copies
    // above are in flight: measured on configs[1], keeping the previous step's plan alive and extending it (no planning,
    // pinned plan image) did not shorten the call (0.289 against 0.282 ms): the host work is hidden under the DMA.
    std::vector<int32_t> ones;
    if (!h_q_lens) ones.assign((size_t)batch, 1);
    int err;
    csv_plan_t* plan = csv_plan_build_host(shape, h_q_lens ? h_q_lens : ones.data(), h_kv_lens, batch, max_partition_tokens, &err);
    if (!plan) {
        (void)cudaStreamSynchronize(st);   // (only CSV_E_NOMEM of the host heap can get here: lengths were checked above)
        return err;
    }
    int rc = ws_bytes - L.plan < plan->lay.total ? CSV_E_NOMEM : plan_attach(plan, ws + L.plan, ws_bytes - L.plan, stream);
    for (int l = 0; rc == CSV_OK && l < n_layers; ++l)   // KV write of every new row + decode rows + appended chunks
        rc = csv_tail_step(plan, pool, layer_begin + l, ws + L.q + l * q_layer, ws + L.k + l * k_layer, ws + L.v + l * k_layer,
                           (const int32_t*)(ws + L.tables), max_blocks, ws + L.out + l * q_layer,
                           (float*)(ws + L.lse + l * lse_layer), stream);
    if (rc == CSV_OK) {
        if ((e = cudaMemcpyAsync(h_out, ws + L.out, q_layer * n_layers, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
            (e = cudaMemcpyAsync(h_lse, ws + L.lse, lse_layer * n_layers, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
            (e = cudaStreamSynchronize(st)) != cudaSuccess)
            rc = csv_set_cuda_error((int)e);
    } else {
        // Workspace too small for the plan, or a launch failed part-way: the input copies (and perhaps some layers' work)
        // are enqueued.  Drain the stream so that nothing reads the caller's host buffers after the error is returned.
        (void)cudaStreamSynchronize(st);
    }
    csv_plan_destroy(plan);
    return rc;
}

}   // extern "C"
