// pool.cpp — host-only part of libconserve_kv.so: block-table allocator (a1), placement (a6),
// provisioning (§4.1).  No CUDA calls in this file.
#include <math.h>

#include <new>

#include "internal.h"

static bool shape_ok(const kv_pool_desc* s, bool need_blocks) {
    if (!s) return false;
    if (s->dtype != CSV_DTYPE_BF16 || s->block_size != CSV_BLOCK_SIZE) return false;
    if (s->head_dim != 64 && s->head_dim != 128) return false;
    if (s->num_kv_heads != 1 && s->num_kv_heads != 2 && s->num_kv_heads != 4 && s->num_kv_heads != 8) return false;
    if (s->num_layers < 1) return false;
    if (need_blocks && s->num_blocks < 1) return false;
    return true;
}
bool csv_shape_ok(const kv_pool_desc* s, bool need_blocks) { return shape_ok(s, need_blocks); }

extern "C" {

const char* csv_version(void) { return "conserve_kv 0.1.0 (sm_100a)"; }

size_t kv_pool_bytes(const kv_pool_desc* desc) {
    if (!shape_ok(desc, true)) return 0;
    return (size_t)desc->num_layers * (size_t)desc->num_blocks * 2u * (size_t)desc->num_kv_heads *
           csv_tile_bytes(desc->head_dim);
}

int kv_pool_create(const kv_pool_desc* desc, void* d_base, size_t bytes, kv_pool_t** out) {
    if (!out || !shape_ok(desc, true) || !d_base) return CSV_E_INVAL;
    if (((uintptr_t)d_base & 127u) != 0) return CSV_E_INVAL;
    if (bytes < kv_pool_bytes(desc)) return CSV_E_INVAL;
    kv_pool* p = new (std::nothrow) kv_pool();
    if (!p) return CSV_E_NOMEM;
    p->desc = *desc;
    p->d_base = (uint8_t*)d_base;
    p->bytes = bytes;
    p->in_use.assign((size_t)desc->num_blocks, 0);
    for (int32_t i = 0; i < desc->num_blocks; ++i) p->free_list.push_back(i);
    p->used = 0;
    *out = p;
    return CSV_OK;
}

int kv_pool_destroy(kv_pool_t* pool) {
    if (!pool) return CSV_E_INVAL;
    delete pool;
    return CSV_OK;
}

int kv_pool_set_free_order(kv_pool_t* pool, const int32_t* h_order, int32_t n) {
    if (!pool || n < 0 || (n > 0 && !h_order)) return CSV_E_INVAL;
    if ((size_t)n != pool->free_list.size()) return CSV_E_INVAL;
    std::vector<uint8_t> seen((size_t)pool->desc.num_blocks, 0);
    for (int32_t i = 0; i < n; ++i) {
        const int32_t id = h_order[i];
        if (id < 0 || id >= pool->desc.num_blocks || pool->in_use[(size_t)id] || seen[(size_t)id]) return CSV_E_INVAL;
        seen[(size_t)id] = 1;
    }
    pool->free_list.assign(h_order, h_order + n);
    return CSV_OK;
}

int kv_alloc_blocks(kv_pool_t* pool, int32_t n, int32_t* h_out_ids) {
    if (!pool || n < 0 || (n > 0 && !h_out_ids)) return CSV_E_INVAL;
    if ((size_t)n > pool->free_list.size()) return CSV_E_NOMEM;
    for (int32_t i = 0; i < n; ++i) {
        const int32_t id = pool->free_list.front();
        pool->free_list.pop_front();
        pool->in_use[(size_t)id] = 1;
        h_out_ids[i] = id;
    }
    pool->used += n;
    return CSV_OK;
}

int kv_free_blocks(kv_pool_t* pool, const int32_t* h_ids, int32_t n) {
    if (!pool || n < 0 || (n > 0 && !h_ids)) return CSV_E_INVAL;
    // validate everything first: a failed call changes nothing
    for (int32_t i = 0; i < n; ++i) {
        const int32_t id = h_ids[i];
        if (id < 0 || id >= pool->desc.num_blocks || pool->in_use[(size_t)id] != 1) {
            for (int32_t j = 0; j < i; ++j) pool->in_use[(size_t)h_ids[j]] = 1;   // undo the marks
            return CSV_E_INVAL;
        }
        pool->in_use[(size_t)id] = 2;   // mark: catches a duplicate inside h_ids
    }
    for (int32_t i = 0; i < n; ++i) {
        pool->in_use[(size_t)h_ids[i]] = 0;
        pool->free_list.push_back(h_ids[i]);
    }
    pool->used -= n;
    return CSV_OK;
}

int32_t kv_pool_used_blocks(const kv_pool_t* pool) { return pool ? pool->used : -1; }
int32_t kv_pool_num_blocks(const kv_pool_t* pool) { return pool ? pool->desc.num_blocks : -1; }
int32_t kv_pool_free_blocks(const kv_pool_t* pool) { return pool ? (int32_t)pool->free_list.size() : -1; }

int kv_pool_get_desc(const kv_pool_t* pool, kv_pool_desc* out) {
    if (!pool || !out) return CSV_E_INVAL;
    *out = pool->desc;
    return CSV_OK;
}

int csv_place(const kv_pool_t* const* pools, int32_t n_pools, int32_t need_blocks, int32_t* out_idx) {
    if (!pools || n_pools <= 0 || need_blocks < 0 || !out_idx) return CSV_E_INVAL;
    for (int32_t i = 0; i < n_pools; ++i)
        if (!pools[i]) return CSV_E_INVAL;
    int32_t best = -1;
    for (int32_t i = 0; i < n_pools; ++i) {
        const kv_pool* p = pools[i];
        if ((int64_t)p->free_list.size() < (int64_t)need_blocks) continue;   // saturated: route elsewhere
        if (best < 0) {
            best = i;
            continue;
        }
        const kv_pool* b = pools[best];
        // used_i / total_i < used_b / total_b, exactly
        if ((int64_t)p->used * b->desc.num_blocks < (int64_t)b->used * p->desc.num_blocks) best = i;
    }
    if (best < 0) return CSV_E_NOMEM;
    *out_idx = best;
    return CSV_OK;
}

int csv_provision(double T_p, double L_in, double T_d, double L_d, double B, double W, double* out_rate,
                  double* out_n_throughput, double* out_n_memory, int32_t* out_n) {
    if (!(T_p > 0.0) || !(L_in > 0.0) || !(T_d > 0.0) || !(L_d > 0.0) || !(B > 0.0) || !(W > 0.0)) return CSV_E_INVAL;
    const double rate = T_p / L_in;       // R*
    const double n_thr = rate * L_d / T_d;   // Eq. 1
    const double n_mem = rate * W / B;       // Eq. 2
    if (out_rate) *out_rate = rate;
    if (out_n_throughput) *out_n_throughput = n_thr;
    if (out_n_memory) *out_n_memory = n_mem;
    if (out_n) *out_n = (int32_t)ceil(n_thr > n_mem ? n_thr : n_mem);
    return CSV_OK;
}

}   // extern "C"
