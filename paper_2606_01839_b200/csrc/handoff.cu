// handoff.cu — kv_pack / kv_unpack / kv_handoff_direct / kv_append_tokens: the one-shot KV handoff (a2, a3;
// PAPER.md:150 §4 "transferred once", §3.1 cost linear in tokens) and the
// tail step's new-token KV write (§2.1 "appending one new entry").
//
// Pure 16-byte moves (bit-exact for any pattern).  Roofline: HBM, read + write bytes.
//  - pack:   one unit = (conversation, layer, message block, K|V): 16 token rows of
//            Hkv*d*2 bytes, contiguous in the source (32 KiB at the 8B shape), rewritten as
//            Hkv tiles in the pool's in-tile format (also 32 KiB contiguous).  Thread ->
//            consecutive 16-byte source chunks (fully coalesced reads); writes land as
//            whole 128-byte tile rows.
//  - unpack: one unit = (conversation, layer, message block): 2*Hkv tiles, contiguous in the
//            message AND in the pool (64 KiB at the 8B shape): a straight copy to the
//            block's address from the block table, masked by slot in the first / last block.
#include <stdlib.h>

#include "common.cuh"
#include "internal.h"

namespace {

constexpr int kMaxBatch = 32;        // conversations per launch (descriptors travel as kernel params)
constexpr int kThreads = 256;

struct PackEntry {
    const uint8_t* k;
    const uint8_t* v;
    uint8_t* staging;
    int32_t tokens, slot0, ntb, unit_begin;   // units of this entry: [unit_begin, next.unit_begin)
};
struct PackParams {
    PackEntry e[kMaxBatch];
    int32_t n, total_units, NL, Hkv;
};

struct UnpackEntry {
    const uint8_t* staging;
    const int32_t* ids;     // conversation's table, device
    int32_t tokens, slot0, ntb, blk0, unit_begin, pad;
};
struct UnpackParams {
    UnpackEntry e[kMaxBatch];
    int32_t n, total_units, NL, Hkv;
    int32_t num_blocks, pad;
    uint8_t* pool;
};

struct DirectEntry {
    const uint8_t* k;
    const uint8_t* v;
    const int32_t* ids;     // conversation's table, readable on the device that runs the kernel
    int32_t tokens, slot0, ntb, blk0, unit_begin, pad;
};
struct DirectParams {
    DirectEntry e[kMaxBatch];
    int32_t n, total_units, NL, Hkv;
    int32_t num_blocks, pad;
    uint8_t* pool;          // local or peer-mapped (NVLink) pool base
};

// Plain ld / st: measured faster here than .nc / L1::no_allocate / .cs hints (6.8 vs 6.2 TB/s).
__device__ __forceinline__ uint4 ld16(const void* p) { return *reinterpret_cast<const uint4*>(p); }
__device__ __forceinline__ void st16(void* p, const uint4& v) { *reinterpret_cast<uint4*>(p) = v; }
template <typename P>
__device__ __forceinline__ int find_entry(const P& p, int unit) {
    int lo = 0;
#pragma unroll 1
    for (int i = 1; i < p.n; ++i)
        if (p.e[i].unit_begin <= unit) lo = i;
    return lo;
}

// D = head_dim.  Chunks (16 B) per token row of one head: D/8.  U = 16-byte loads in flight per thread.
// Hkv is a power of two (1, 2, 4, 8): all index arithmetic is shifts and masks.
template <int D, int U>
__global__ void __launch_bounds__(kThreads, 4) pack_kernel(const __grid_constant__ PackParams p) {
    constexpr int CPR = D / 8;                  // chunks per (token, head) row
    constexpr int LCPR = D == 128 ? 4 : 3;
    constexpr int TB = 16 * D * 2;              // tile bytes
    const int lh = 31 - __clz(p.Hkv);           // log2(Hkv)
    const int chunks_per_unit = 16 * p.Hkv * CPR;   // one (layer, tb, kv): 16 slots x Hkv heads x CPR
    const size_t row_bytes = (size_t)p.Hkv * D * 2;
    for (int unit = blockIdx.x; unit < p.total_units; unit += gridDim.x) {
        const int ei = find_entry(p, unit);
        const PackEntry& e = p.e[ei];
        const int u = unit - e.unit_begin;      // ((layer * ntb) + tb) * 2 + kv
        const int kv = u & 1;
        const int layer = (u >> 1) / e.ntb;
        const int tb = (u >> 1) - layer * e.ntb;
        const uint8_t* src_layer = (kv ? e.v : e.k) + (size_t)layer * e.tokens * row_bytes;
        uint8_t* dst_unit = e.staging + ((size_t)(layer * e.ntb + tb) * 2 + kv) * p.Hkv * TB;
        const int tok_base = tb * 16 - e.slot0;   // message token of slot 0 of this block
        // the 16 token rows of a block are contiguous in the source: chunk c of the unit is at src_row0 + 16 c
        const uint8_t* src_row0 = src_layer + (ptrdiff_t)tok_base * (ptrdiff_t)row_bytes;
        for (int c0 = threadIdx.x; c0 < chunks_per_unit; c0 += kThreads * U) {
            uint4 val[U];
#pragma unroll
            for (int j = 0; j < U; ++j) {
                const int c = c0 + j * kThreads;
                const int tok = tok_base + (c >> (LCPR + lh));
                val[j] = make_uint4(0, 0, 0, 0);
                if (c < chunks_per_unit && tok >= 0 && tok < e.tokens) val[j] = ld16(src_row0 + (size_t)c * 16);
            }
#pragma unroll
            for (int j = 0; j < U; ++j) {
                const int c = c0 + j * kThreads;
                if (c < chunks_per_unit) {
                    const int chunk = c & (CPR - 1);
                    const int head = (c >> LCPR) & (p.Hkv - 1);
                    const int slot = c >> (LCPR + lh);
                    st16(dst_unit + head * TB + (chunk >> 3) * 2048 + slot * 128 + (((chunk & 7) ^ (slot & 7)) << 4), val[j]);
                }
            }
        }
    }
}

template <int D, int U>
__global__ void __launch_bounds__(kThreads, 4) unpack_kernel(const __grid_constant__ UnpackParams p) {
    constexpr int TB = 16 * D * 2;
    constexpr int CPT = TB / 16;                       // chunks per tile
    const int chunks_per_unit = 2 * p.Hkv * CPT;       // one (layer, tb): K and V tiles of all heads
    for (int unit = blockIdx.x; unit < p.total_units; unit += gridDim.x) {
        const int ei = find_entry(p, unit);
        const UnpackEntry& e = p.e[ei];
        const int u = unit - e.unit_begin;             // layer * ntb + tb
        const int layer = u / e.ntb;
        const int tb = u - layer * e.ntb;
        const int block = __ldg(e.ids + e.blk0 + tb);
        const int lo = tb == 0 ? e.slot0 : 0;
        const int hi = tb == e.ntb - 1 ? ((e.slot0 + e.tokens - 1) & 15) + 1 : 16;
        const uint8_t* src = e.staging + (size_t)u * chunks_per_unit * 16;
        uint8_t* dst = p.pool + ((size_t)layer * p.num_blocks + block) * chunks_per_unit * 16;
        const bool full = lo == 0 && hi == 16;
        for (int c0 = threadIdx.x; c0 < chunks_per_unit; c0 += kThreads * U) {
            uint4 val[U];
            bool ok[U];
#pragma unroll
            for (int j = 0; j < U; ++j) {
                const int c = c0 + j * kThreads;
                ok[j] = c < chunks_per_unit;
                if (ok[j] && !full) {
                    const int slot = ((c & (CPT - 1)) & 127) >> 3;
                    ok[j] = slot >= lo && slot < hi;
                }
                if (ok[j]) val[j] = ld16(src + (size_t)c * 16);
            }
#pragma unroll
            for (int j = 0; j < U; ++j)
                if (ok[j]) st16(dst + (size_t)(c0 + j * kThreads) * 16, val[j]);
        }
    }
}

// kv_handoff_direct: pack and unpack composed, no staging message ("transferred once to
// the bound decoder").  Unit = (conversation, layer, block, K|V): 16 contiguous source token rows (32 KiB at the 8B
// shape) -> the Hkv tiles of (layer, table[block], K|V), also 32 KiB contiguous in the destination pool.  The kernel runs
// where the source lives and PUSHES: loads are local and coalesced, stores are whole 128-byte tile rows and may cross
// NVLink (posted writes; nothing is ever loaded from the peer).  Slots outside the message are not written.
template <int D, int U>
__global__ void __launch_bounds__(kThreads, 4) direct_kernel(const __grid_constant__ DirectParams p) {
    constexpr int CPR = D / 8;
    constexpr int LCPR = D == 128 ? 4 : 3;
    constexpr int TB = 16 * D * 2;
    const int lh = 31 - __clz(p.Hkv);
    const int chunks_per_unit = 16 * p.Hkv * CPR;
    const size_t row_bytes = (size_t)p.Hkv * D * 2;
    for (int unit = blockIdx.x; unit < p.total_units; unit += gridDim.x) {
        const int ei = find_entry(p, unit);
        const DirectEntry& e = p.e[ei];
        const int u = unit - e.unit_begin;      // ((layer * ntb) + tb) * 2 + kv
        const int kv = u & 1;
        const int layer = (u >> 1) / e.ntb;
        const int tb = (u >> 1) - layer * e.ntb;
        const int block = __ldg(e.ids + e.blk0 + tb);
        const uint8_t* src_layer = (kv ? e.v : e.k) + (size_t)layer * e.tokens * row_bytes;
        uint8_t* dst_unit = p.pool + (((size_t)layer * p.num_blocks + block) * 2 + kv) * p.Hkv * TB;
        const int tok_base = tb * 16 - e.slot0;
        const uint8_t* src_row0 = src_layer + (ptrdiff_t)tok_base * (ptrdiff_t)row_bytes;
        for (int c0 = threadIdx.x; c0 < chunks_per_unit; c0 += kThreads * U) {
            uint4 val[U];
            bool ok[U];
#pragma unroll
            for (int j = 0; j < U; ++j) {
                const int c = c0 + j * kThreads;
                const int tok = tok_base + (c >> (LCPR + lh));
                ok[j] = c < chunks_per_unit && tok >= 0 && tok < e.tokens;
                if (ok[j]) val[j] = ld16(src_row0 + (size_t)c * 16);
            }
#pragma unroll
            for (int j = 0; j < U; ++j) {
                if (ok[j]) {
                    const int c = c0 + j * kThreads;
                    const int chunk = c & (CPR - 1);
                    const int head = (c >> LCPR) & (p.Hkv - 1);
                    const int slot = c >> (LCPR + lh);
                    st16(dst_unit + head * TB + (chunk >> 3) * 2048 + slot * 128 + (((chunk & 7) ^ (slot & 7)) << 4), val[j]);
                }
            }
        }
    }
}

// New-token KV of a whole batch, token-major [NL][total_q][Hkv][D] -> pool.
// meta: [q_start[batch+1] | kv_len[batch] | q_len[batch]] on the device.
template <int D>
__global__ void __launch_bounds__(kThreads) append_tokens_kernel(uint8_t* pool, int num_blocks, int NL, int Hkv,
                                                                 const uint8_t* k_new, const uint8_t* v_new,
                                                                 const int32_t* meta, int batch, int total_q,
                                                                 const int32_t* tables, int max_blocks) {
    constexpr int CPR = D / 8;
    constexpr int TB = 16 * D * 2;
    pdl_trigger();   // a PDL-launched paged_decode_attn may start its prologue; it waits for this grid
    const int32_t* q_start = meta;
    const int32_t* kv_len = meta + batch + 1;
    const int32_t* q_len = kv_len + batch;
    const long long total = (long long)NL * total_q * 2 * Hkv * CPR;
    for (long long idx = (long long)blockIdx.x * kThreads + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * kThreads) {
        const int chunk = (int)(idx % CPR);
        long long r = idx / CPR;
        const int head = (int)(r % Hkv);
        r /= Hkv;
        const int kv = (int)(r & 1);
        r >>= 1;
        const int row = (int)(r % total_q);
        const int layer = (int)(r / total_q);
        int lo = 0, hi = batch;   // find conv with q_start[conv] <= row < q_start[conv+1]
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (q_start[mid] <= row) lo = mid; else hi = mid;
        }
        const int pos = kv_len[lo] - q_len[lo] + (row - q_start[lo]);
        if (pos < 0) continue;   // decode row on an empty cache (q_len 1, kv_len 0): it has no position to write
        const int block = __ldg(tables + (size_t)lo * max_blocks + (pos >> 4));
        const int slot = pos & 15;
        const uint8_t* src = (kv ? v_new : k_new) + (((size_t)layer * total_q + row) * Hkv + head) * D * 2 + chunk * 16;
        uint8_t* dst = pool + ((((size_t)layer * num_blocks + block) * 2 + kv) * Hkv + head) * TB + (chunk >> 3) * 2048 +
                       slot * 128 + (((chunk & 7) ^ (slot & 7)) << 4);
        st_stream(dst, ld_stream(src));
    }
}

}   // namespace

// One CTA per unit, NOT a persistent grid-stride loop: the chip then sweeps source and destination
// linearly.  Measured on config 4 shapes: grid = 8 CTAs/SM grid-striding 5.9 TB/s, one CTA per unit 6.8 TB/s.
static int grid_for(int total_units) { return total_units > 0 ? total_units : 1; }

int launch_pack(const kv_pool_desc& shape, int n, const void* const* k, const void* const* v, const int32_t* tokens,
                const int32_t* offs, void* const* staging, void* stream) {
    int i = 0;
    while (i < n) {
        PackParams p;
        p.n = 0;
        p.NL = shape.num_layers;
        p.Hkv = shape.num_kv_heads;
        long long units = 0;
        while (i < n && p.n < kMaxBatch) {
            if (tokens[i] > 0) {
                PackEntry& e = p.e[p.n];
                e.k = (const uint8_t*)k[i];
                e.v = (const uint8_t*)v[i];
                e.staging = (uint8_t*)staging[i];
                e.tokens = tokens[i];
                e.slot0 = offs[i] & 15;
                e.ntb = (e.slot0 + e.tokens + 15) / 16;
                const long long nu = (long long)shape.num_layers * e.ntb * 2;
                if (units + nu > INT32_MAX) break;
                e.unit_begin = (int32_t)units;
                units += nu;
                ++p.n;
            }
            ++i;
        }
        if (p.n == 0) {
            if (i < n && tokens[i] > 0) return CSV_E_INVAL;   // a single entry too large for one launch
            continue;
        }
        p.total_units = (int32_t)units;
        const int grid = grid_for(p.total_units);
        if (shape.head_dim == 128) {
            pack_kernel<128, 4><<<grid, kThreads, 0, (cudaStream_t)stream>>>(p);
        } else {
            pack_kernel<64, 4><<<grid, kThreads, 0, (cudaStream_t)stream>>>(p);
        }
        CSV_CUDA_TRY(cudaGetLastError());
    }
    return CSV_OK;
}

int launch_unpack(kv_pool* dst, int n, const void* const* staging, const int32_t* tokens, const int32_t* offs,
                  const int32_t* const* block_ids, void* stream) {
    const kv_pool_desc& shape = dst->desc;
    int i = 0;
    while (i < n) {
        UnpackParams p;
        p.n = 0;
        p.NL = shape.num_layers;
        p.Hkv = shape.num_kv_heads;
        p.num_blocks = shape.num_blocks;
        p.pool = dst->d_base;
        long long units = 0;
        while (i < n && p.n < kMaxBatch) {
            if (tokens[i] > 0) {
                UnpackEntry& e = p.e[p.n];
                e.staging = (const uint8_t*)staging[i];
                e.ids = block_ids[i];
                e.tokens = tokens[i];
                e.slot0 = offs[i] & 15;
                e.ntb = (e.slot0 + e.tokens + 15) / 16;
                e.blk0 = offs[i] >> 4;
                const long long nu = (long long)shape.num_layers * e.ntb;
                if (units + nu > INT32_MAX) break;
                e.unit_begin = (int32_t)units;
                units += nu;
                ++p.n;
            }
            ++i;
        }
        if (p.n == 0) {
            if (i < n && tokens[i] > 0) return CSV_E_INVAL;
            continue;
        }
        p.total_units = (int32_t)units;
        const int grid = grid_for(p.total_units);
        if (shape.head_dim == 128) {
            unpack_kernel<128, 8><<<grid, kThreads, 0, (cudaStream_t)stream>>>(p);
        } else {
            unpack_kernel<64, 4><<<grid, kThreads, 0, (cudaStream_t)stream>>>(p);
        }
        CSV_CUDA_TRY(cudaGetLastError());
    }
    return CSV_OK;
}

int launch_handoff_direct(kv_pool* dst, int n, const void* const* k, const void* const* v, const int32_t* tokens,
                          const int32_t* offs, const int32_t* const* block_ids, void* stream) {
    const kv_pool_desc& shape = dst->desc;
    int i = 0;
    while (i < n) {
        DirectParams p;
        p.n = 0;
        p.NL = shape.num_layers;
        p.Hkv = shape.num_kv_heads;
        p.num_blocks = shape.num_blocks;
        p.pool = dst->d_base;
        long long units = 0;
        while (i < n && p.n < kMaxBatch) {
            if (tokens[i] > 0) {
                DirectEntry& e = p.e[p.n];
                e.k = (const uint8_t*)k[i];
                e.v = (const uint8_t*)v[i];
                e.ids = block_ids[i];
                e.tokens = tokens[i];
                e.slot0 = offs[i] & 15;
                e.ntb = (e.slot0 + e.tokens + 15) / 16;
                e.blk0 = offs[i] >> 4;
                const long long nu = (long long)shape.num_layers * e.ntb * 2;
                if (units + nu > INT32_MAX) break;
                e.unit_begin = (int32_t)units;
                units += nu;
                ++p.n;
            }
            ++i;
        }
        if (p.n == 0) {
            if (i < n && tokens[i] > 0) return CSV_E_INVAL;
            continue;
        }
        p.total_units = (int32_t)units;
        const int grid = grid_for(p.total_units);
        if (shape.head_dim == 128) {
            direct_kernel<128, 4><<<grid, kThreads, 0, (cudaStream_t)stream>>>(p);
        } else {
            direct_kernel<64, 4><<<grid, kThreads, 0, (cudaStream_t)stream>>>(p);
        }
        CSV_CUDA_TRY(cudaGetLastError());
    }
    return CSV_OK;
}

int launch_append_tokens(kv_pool* dst, const csv_plan* plan, const void* k_new, const void* v_new,
                         const int32_t* tables, int max_blocks, void* stream) {
    const kv_pool_desc& s = dst->desc;
    if (plan->total_q == 0) return CSV_OK;
    const long long total = (long long)s.num_layers * plan->total_q * 2 * s.num_kv_heads * (s.head_dim / 8);
    long long blocks = (total + kThreads - 1) / kThreads;
    const int cap = csv_query_num_sms() * 8;
    const int grid = (int)(blocks < cap ? blocks : cap);
    const int32_t* meta = (const int32_t*)(plan->d_ws + plan->lay.conv_meta);
    if (s.head_dim == 128)
        append_tokens_kernel<128><<<grid, kThreads, 0, (cudaStream_t)stream>>>(
            dst->d_base, s.num_blocks, s.num_layers, s.num_kv_heads, (const uint8_t*)k_new, (const uint8_t*)v_new, meta,
            plan->batch, plan->total_q, tables, max_blocks);
    else
        append_tokens_kernel<64><<<grid, kThreads, 0, (cudaStream_t)stream>>>(
            dst->d_base, s.num_blocks, s.num_layers, s.num_kv_heads, (const uint8_t*)k_new, (const uint8_t*)v_new, meta,
            plan->batch, plan->total_q, tables, max_blocks);
    CSV_CUDA_TRY(cudaGetLastError());
    return CSV_OK;
}
