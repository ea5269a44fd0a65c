// internal.h — structures shared by the host side (pool.cpp, plan.cpp, api.cpp) and the
// kernels (*.cu) of libconserve_kv.so.  Nothing here is visible across the C ABI.
#pragma once
#include <stddef.h>
#include <stdint.h>
#include <string.h>

#include <deque>
#include <vector>

#include "../../include/conserve_kv.h"

// ---- pool -----------------------------------------------------------------------------
struct kv_pool {
    kv_pool_desc desc;
    uint8_t* d_base;
    size_t bytes;
    std::deque<int32_t> free_list;   // hand-out order: front first; frees go to the back
    std::vector<uint8_t> in_use;     // 1 = handed out
    int32_t used;
};

static inline size_t csv_tile_bytes(int d) { return (size_t)CSV_BLOCK_SIZE * d * 2; }

// ---- work lists (device-visible, 16-byte-aligned records) ---------------------------------------
// One decode partition: blocks [blk_begin, blk_end) of conversation `conv`, KV head `head`.
struct DecodeItem {
    int32_t conv;
    int32_t head;
    int32_t blk_begin;
    int32_t blk_end;
    int32_t kv_len;
    int32_t partial;   // index into the decode partial arrays
    int32_t direct;    // 1 = the only partition of its (conv, head): write O / LSE directly
    int32_t q_row;     // row of this conversation in d_q / d_out / d_lse (= sum of earlier q_lens)
    int32_t group;        // index of the (conv, head) merge group, -1 if direct
    int32_t group_first;  // first partial of the group
    int32_t group_count;  // partials in the group
    int32_t pad;
};

// One append work item: a tile of stacked rows (token-major: row r = i * G + hh) of one
// chunk and one KV head, against blocks [blk_begin, blk_end) of the conversation.
struct AppendItem {
    int32_t conv;
    int32_t head;
    int32_t row_begin;   // first stacked row of the tile (multiple of the tile height)
    int32_t q_start;     // first row of this conversation in d_q / d_out
    int32_t m;           // chunk length (q_len)
    int32_t kv_len;      // P + m
    int32_t blk_begin;
    int32_t blk_end;
    int32_t partial;     // index into the append partial arrays (units of tiles)
    int32_t direct;      // 1 = single KV partition: write O / LSE directly
    int32_t pad0, pad1;
};

// Merge group: partials [first, first + count) belong to one output tile.
struct MergeGroup {
    int32_t first;
    int32_t count;
    int32_t conv;       // decode: conversation (row of d_q); append: conversation
    int32_t head;       // KV head
    int32_t row_begin;  // append only
    int32_t q_start;    // append only
    int32_t m;          // append only
    int32_t pad;
};

constexpr int kDecodeWarps = 8;      // independent warp-workers per decode CTA (d = 64)
constexpr int kDecodeWarps128 = 7;   // ... at d = 128, with 2-stage rings
constexpr int kAppendTileRows = 64;  // stacked rows per append work item of the mma.sync kernel (4 warps x 16)
constexpr int kAppendTileRowsTc2 = 256;  // ... of the two-tile tcgen05 kernel (two UMMA M = 128 tiles sharing K/V)
constexpr int kAppendKvSplit = 8192; // default KV tokens per append partition

struct PlanLayout {   // byte offsets into the caller's workspace (all 128-byte aligned)
    size_t decode_items, worker_begin, decode_groups, decode_po, decode_pml;
    size_t append_items, append_groups, append_po, append_pml;
    size_t tail_items, tail_worker_begin, tail_groups;   // the decode share list of tail_kernel's decode-role CTAs (mixed steps)
    size_t zero_rows;   // int32 rows of d_out / d_lse whose conversation has q_len = 1 and an empty cache
    size_t conv_meta;   // int32 [q_start[batch+1] | kv_len[batch] | q_len[batch]]
    size_t append_sched;   // uint32 [0] next append item, [1] CTAs done, [2] next decode share (tail_kernel): zeroed by a cudaMemsetAsync before every launch
    size_t total;
};

struct csv_plan {
    csv_attn_shape shape;
    int32_t batch;
    int32_t max_partition_tokens;        // decode partition cap in force (1 << 30 when the caller passed 0: share cuts only)
    int32_t max_partition_tokens_user;   // what the caller passed (0 = defaults)
    int32_t num_sms;
    std::vector<int32_t> q_lens, kv_lens, q_start;
    int32_t total_q;
    // decode
    std::vector<DecodeItem> decode_items;
    std::vector<int32_t> worker_begin;       // [workers + 1] into decode_items
    std::vector<MergeGroup> decode_groups;   // groups with count > 1 only
    int32_t n_decode_rows;
    int32_t decode_grid;                     // CTAs
    int32_t decode_warps;                    // warp-workers per CTA (7 at d = 128, 8 at d = 64; others: experiment knobs)
    int32_t n_decode_partials;               // partial slots (non-direct items)
    std::vector<int32_t> zero_rows;          // q rows of decode conversations with kv_len = 0 (O = 0, LSE = -inf)
    // mixed step in one launch (tail_kernel): the decode rows cut again for tail_n_dec CTAs x 8 warp-workers
    int32_t tail_n_dec;                      // SMs that start in the decode role (0 = no fused launch for this plan)
    int32_t tail_n_shares;                   // decode shares of 8 warp-workers each (a queue: any CTA may take one)
    int32_t tail_two_kernels;                // CSV_TUNE_TAIL_TWO_KERNELS in force when the plan was built: csv_tail_step keeps decode + append apart
    std::vector<DecodeItem> tail_items;
    std::vector<int32_t> tail_worker_begin;
    std::vector<MergeGroup> tail_groups;
    int32_t tail_n_partials;
    // append
    std::vector<AppendItem> append_items;
    std::vector<MergeGroup> append_groups;   // groups with count > 1 only
    int32_t n_append_chunks, n_append_rows;
    int32_t append_tile_rows;                // stacked rows per append item: 256 (tcgen05, d = 128: two UMMA tiles) or 64 (mma.sync, d = 64)
    int32_t n_append_partials;               // partial tiles (non-direct items)
    // device
    PlanLayout lay;
    uint8_t* d_ws;                           // NULL = host-only plan
    std::vector<uint8_t> h_image;            // host image of the list part of the workspace
};

// ---- launchers implemented in the .cu files ---------------------------------------------
int csv_set_cuda_error(int err);   // records err, returns CSV_E_CUDA
int launch_pack(const kv_pool_desc& shape, int n, const void* const* k, const void* const* v, const int32_t* tokens,
                const int32_t* offs, void* const* staging, void* stream);
int launch_handoff_direct(kv_pool* dst, int n, const void* const* k, const void* const* v, const int32_t* tokens,
                          const int32_t* offs, const int32_t* const* block_ids, void* stream);
int launch_unpack(kv_pool* dst, int n, const void* const* staging, const int32_t* tokens, const int32_t* offs,
                  const int32_t* const* block_ids, void* stream);
int launch_append_tokens(kv_pool* dst, const csv_plan* plan, const void* k_new, const void* v_new,
                         const int32_t* tables, int max_blocks, void* stream);
int launch_decode(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                  int max_blocks, void* out, float* lse, void* stream, const void* k_new = nullptr,
                  const void* v_new = nullptr);
int launch_append_attn(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                       int max_blocks, void* out, float* lse, void* stream);
int launch_decode_zero_rows(const csv_plan* plan, const kv_pool* pool, void* out, float* lse, void* stream);
int launch_decode_merge_128(const csv_plan* plan, size_t groups_off, int ng, void* out, float* lse, void* stream);
int launch_append_merge_128(const csv_plan* plan, void* out, float* lse, void* stream);   // append partials -> O / LSE
int launch_tail_zero_queue(const csv_plan* plan, void* stream);   // before the kernel that launch_tail_fused(pdl) is chained to
int launch_tail_fused(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                      int max_blocks, void* out, float* lse, void* stream, bool pdl);
int launch_append_attn_tc2(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                           int max_blocks, void* out, float* lse, void* stream);
// Tuning knobs (conserve_kv.h csv_tuning_set): one process-wide table, initialised once from the environment; every plan
// records what it was built with, so a plan and its workspace size cannot disagree unless the caller changes a knob between.
struct CsvTuning {
    int32_t v[CSV_TUNE_COUNT];   // indexed by CSV_TUNE_*; 0 = library default
};
CsvTuning& csv_tuning();
int csv_query_num_sms();   // SM count of the current device, 148 if none is usable
csv_plan* csv_plan_build_host(const csv_attn_shape* shape, const int32_t* h_q_lens, const int32_t* h_kv_lens,
                              int32_t batch, int32_t max_partition_tokens, int* err);
bool csv_shape_ok(const kv_pool_desc* s, bool need_blocks);   // supported (Hkv, d, bs, dtype); need_blocks: num_blocks > 0 too
