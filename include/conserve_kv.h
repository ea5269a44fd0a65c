/*
 * conserve_kv.h — C ABI of libconserve_kv.so
 *
 * The data-parallel hot path under ConServe's conversation-level
 * disaggregation (arxiv/paper_2606_01839): the memory-bound conversation tail
 * that is pinned to one decoder, plus the one-shot KV handoff that brings a
 * conversation's turn-1 prefill KV into that decoder's paged pool.
 *
 * Citations are "PAPER.md:N" = line N of the paper text, with the section.
 * The paper describes no kernel and no layout (it names vLLM + LMCache,
 * PAPER.md:213 §5.1); every layout below is this library's own and is
 * restated, independently, by the CPU oracle under oracle/.
 *
 * Conventions
 *  - Plain C ABI. Every call that can fail returns int: CSV_OK (0) or a
 *    negative CSV_E_* code. A failed call changes nothing (no partial
 *    allocation, no launch).
 *  - The library NEVER allocates device memory. "d_" arguments are device
 *    pointers owned by the caller (e.g. torch tensors' data_ptr()); "h_"
 *    arguments are host pointers. `stream` is a cudaStream_t passed as void*.
 *    (The one piece of device memory that is the library's own is the fixed
 *    CSV_STATIC_SCRATCH_BYTES array behind paged_decode_attn_static: part of
 *    the loaded image, not an allocation; see that call for what it costs.)
 *  - Kernel-launching calls enqueue on `stream` and return without
 *    synchronising. Host-side calls (allocator, plan, place) are synchronous,
 *    thread-compatible, not thread-safe.
 *  - Supported shapes (anything else -> CSV_E_INVAL): bf16 (dtype 0),
 *    block_size 16, head_dim in {64, 128}, num_kv_heads in {1, 2, 4, 8},
 *    GQA group G = Hq / Hkv in {1, 2, 4, 8}.
 *  - There is no CPU fallback: if no CUDA device / kernel image is usable the
 *    launching calls return CSV_E_CUDA.
 *  - Devices.  Every call works on the CURRENT device (cudaSetDevice) of the
 *    calling thread: a pool, a plan and its workspace, and the stream passed
 *    with them must all belong to the device that is current at the call.  The
 *    usual deployment is one process per GPU (§5.1 "each served
 *    model replica occupies one GPU").  A process that drives several GPUs may
 *    do so, one device current at a time: the library keeps its per-device
 *    state (kernel attributes, SM count, IPC mappings) per device ordinal.  A
 *    plan is sized for the SM count of the device current at csv_plan_create.
 *    The only cross-device access is the STORE side of kv_handoff_direct into a
 *    peer-mapped pool.
 *  - Block ids handed to kernels (d_block_ids, d_block_tables) are NOT
 *    range-checked on the device: an id outside [0, num_blocks) among the
 *    entries a call addresses is undefined behaviour (an out-of-bounds access).
 *    Entries a call does not address (past ceil(kv_len / 16)) are never read.
 *    Ids that crossed a process boundary must be validated by the receiver
 *    before the launch (replicas.PeerPools.push does).
 *
 * Pool layout (one pool = one decoder's, or the prefiller's, KV memory)
 *
 *   A pool is an array of TILES.  tile(layer, block, kv, head) has index
 *       ((layer * num_blocks + block) * 2 + kv) * Hkv + head        kv: 0 = K, 1 = V
 *   and holds block_size * head_dim bf16 = the K (or V) rows of one KV head
 *   for the 16 token slots of one block: 4 KiB at head_dim 128, 2 KiB at 64.
 *   All tiles of one (layer, block) are contiguous (2 * Hkv tiles = 64 KiB at
 *   the 8B / 70B shapes).
 *
 *   Inside a tile, element (slot, c), slot in [0,16), c in [0,head_dim):
 *       half  = c / 64            (head_dim 64 has one half)
 *       chunk = (c % 64) / 8      (a chunk = 8 bf16 = 16 bytes)
 *       e     = c % 8
 *       off   = half * (16 * 64) + slot * 64 + ((chunk ^ (slot & 7)) * 8) + e     [bf16 units]
 *   i.e. each half is 16 rows of 128 bytes whose 16-byte chunks are XOR-ed
 *   with the row index mod 8.  This is the image a TMA load with
 *   SWIZZLE_128B would leave in shared memory; storing it in HBM means a
 *   plain 1-D bulk copy (cp.async.bulk) of a tile lands ready for
 *   bank-conflict-free ldmatrix / tensor-core use. The handoff writes it once
 *   (§4 "transferred once"), every tail step reads it
 *   (§2.1 "reading the full KV cache").
 *
 *   Token t of a conversation lives in block table[t / 16], slot t % 16; one
 *   block table per conversation serves all layers.
 *
 * Staging message layout (the unit that crosses from prefiller to decoder)
 *
 *   For `tokens` tokens that will occupy conversation positions
 *   [token_offset, token_offset + tokens): slot0 = token_offset % 16,
 *   ntile_blocks = ceil((slot0 + tokens) / 16).  The message is the run of
 *   tiles  [layer][tb][kv][head],  tb in [0, ntile_blocks), each in the pool's
 *   intra-tile format; message token i sits in tb = (slot0 + i) / 16 at slot
 *   (slot0 + i) % 16.  Slots of the message that carry no token are written
 *   as zero by kv_pack and ignored by kv_unpack.
 */
#ifndef CONSERVE_KV_H_
#define CONSERVE_KV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CSV_OK        0
#define CSV_E_INVAL  (-1)   /* bad argument, unsupported shape, misaligned pointer */
#define CSV_E_NOMEM  (-2)   /* pool exhausted / workspace too small */
#define CSV_E_CUDA   (-3)   /* a CUDA runtime call failed; see csv_last_cuda_error() */

#define CSV_DTYPE_BF16 0
#define CSV_BLOCK_SIZE 16

typedef struct kv_pool  kv_pool_t;   /* host object; owns no device memory */
typedef struct csv_plan csv_plan_t;  /* host object + pointers into caller workspace */

/* Shape of a pool / of a conversation's KV. */
typedef struct {
    int32_t num_layers;    /* NL */
    int32_t num_blocks;    /* blocks in the pool (ignored by kv_pack / kv_staging_bytes) */
    int32_t block_size;    /* must be 16 */
    int32_t num_kv_heads;  /* Hkv */
    int32_t head_dim;      /* d: 64 or 128 */
    int32_t dtype;         /* CSV_DTYPE_BF16 */
} kv_pool_desc;

/* Shape of an attention call. */
typedef struct {
    int32_t num_q_heads;   /* Hq, a multiple of Hkv */
    int32_t num_kv_heads;  /* Hkv */
    int32_t head_dim;      /* d */
    int32_t block_size;    /* 16 */
} csv_attn_shape;

/* cudaError_t of the last failing CUDA call made by this library (0 if none). */
int csv_last_cuda_error(void);
/* Library version string, static storage. */
const char* csv_version(void);

/* ------------------------------------------------------------------------
 * a1. Block-table allocator (host only).  PAPER.md:11 §1 "a KV cache that only
 * grows"; §4.2: per-decoder *active* KV occupancy, decremented on
 * conversation termination; §5.1: a decoder holds ~300k tokens.
 * ---------------------------------------------------------------------- */

/* Bytes a pool of this shape occupies: NL * num_blocks * 2 * Hkv * 16 * d * 2. */
size_t kv_pool_bytes(const kv_pool_desc* desc);

/* Wrap caller memory as a pool.  d_base: device pointer, 128-byte aligned,
 * `bytes` >= kv_pool_bytes(desc).  The free list starts as 0,1,...,num_blocks-1.
 * The pool contents are not touched.  *out receives the handle. */
int kv_pool_create(const kv_pool_desc* desc, void* d_base, size_t bytes, kv_pool_t** out);
/* Frees the host object only. */
int kv_pool_destroy(kv_pool_t* pool);
/* Install a caller-chosen order of the currently free blocks: `order` must be
 * a permutation of exactly the free ids (n = number free).  Blocks are then
 * handed out order[0], order[1], ...  (how the harness gets "a shuffled
 * free-block list"). */
int kv_pool_set_free_order(kv_pool_t* pool, const int32_t* h_order, int32_t n);
/* Pop n ids in free-list order into h_out_ids.  All-or-nothing: CSV_E_NOMEM
 * and no change if fewer than n are free.  n = 0 is OK.  Growing a
 * conversation = another call, appended to the caller's table. */
int kv_alloc_blocks(kv_pool_t* pool, int32_t n, int32_t* h_out_ids);
/* Conversation termination.  Ids are pushed back at the tail of
 * the free list in the order given.  Out-of-range id, double free, or a
 * duplicate inside `h_ids` -> CSV_E_INVAL and no change. */
int kv_free_blocks(kv_pool_t* pool, const int32_t* h_ids, int32_t n);
/* Active occupancy in blocks / pool size / free count (negative on NULL). */
int32_t kv_pool_used_blocks(const kv_pool_t* pool);
int32_t kv_pool_num_blocks(const kv_pool_t* pool);
int32_t kv_pool_free_blocks(const kv_pool_t* pool);
/* Copy the pool's shape into *out. */
int kv_pool_get_desc(const kv_pool_t* pool, kv_pool_desc* out);

/* ------------------------------------------------------------------------
 * a6. Placement (host only).  PAPER.md:178 §4.2: "binds the conversation to
 * the decoder replica with the lowest current KV cache occupancy. The binding
 * is persistent"; §1: a saturated decoder is skipped ("routes the
 * next conversation elsewhere rather than migrating one already placed").
 * Occupancy = used / total blocks (compared exactly, as cross-multiplied
 * integers); ties -> lowest index; pools with fewer than need_blocks free are
 * skipped; none fits -> CSV_E_NOMEM.  Never moves anything.
 * ---------------------------------------------------------------------- */
int csv_place(const kv_pool_t* const* pools, int32_t n_pools, int32_t need_blocks, int32_t* out_idx);

/* Provisioning, §4.1: R* = T_p / L_in; Eq. 1  N*T_d >= R*L_d;
 * Eq. 2  N*B >= R*W.  Writes R*, the two real-valued lower bounds on N at
 * R = R*, and the smallest integer N satisfying both.  Any non-positive
 * input -> CSV_E_INVAL.  Worked example PAPER.md:209: 25k, 15k, 1k, 1k -> 1.67. */
int csv_provision(double T_p, double L_in, double T_d, double L_d, double B, double W,
                  double* out_rate, double* out_n_throughput, double* out_n_memory, int32_t* out_n);

/* ------------------------------------------------------------------------
 * a2 / a3. One-shot KV handoff.  PAPER.md:150 §4: "the resulting KV cache is
 * transferred once to the bound decoder"; §3.1 / Fig. 3: cost
 * linear in tokens.  Pure 16-byte moves: bit-exact for any bit pattern.
 * ---------------------------------------------------------------------- */

/* Bytes of the staging message for `tokens` tokens landing at token_offset
 * (see layout above).  0 if tokens <= 0 or the shape is unsupported. */
size_t kv_staging_bytes(const kv_pool_desc* shape, int32_t tokens, int32_t token_offset);

/* One conversation's handoff.  Source is contiguous and token-major, as a
 * prefiller holds it: d_k, d_v each [NL][tokens][Hkv][d] bf16, 16-byte
 * aligned.  d_staging: >= kv_staging_bytes(...), 128-byte aligned; every byte
 * of the message is written (unused slots as zero). */
int kv_pack(const kv_pool_desc* shape, const void* d_k, const void* d_v, int32_t tokens,
            int32_t token_offset, void* d_staging, void* stream);

/* Scatter a message into `dst` through the conversation's block table.
 * Writes conversation positions [token_offset, token_offset + tokens);
 * token_offset = 0 for the handoff, = P for a tail append.  d_block_ids: the
 * conversation's whole table on the device (n_ids entries, n_ids >=
 * ceil((token_offset + tokens) / 16), else CSV_E_INVAL before any launch).
 * Slots not addressed are NOT written.  Destination blocks must be exclusive
 * to this conversation.  The pool's shape must equal the message's. */
int kv_unpack(kv_pool_t* dst, const void* d_staging, int32_t tokens, int32_t token_offset,
              const int32_t* d_block_ids, int32_t n_ids, void* stream);

/* Batched forms: n conversations in as few launches as possible (arrays are
 * host arrays of length n; device pointers inside).  Entries with tokens = 0
 * are skipped.  Semantics per entry identical to the single calls. */
int kv_pack_batch(const kv_pool_desc* shape, int32_t n, const void* const* h_d_k,
                  const void* const* h_d_v, const int32_t* h_tokens, const int32_t* h_token_offsets,
                  void* const* h_d_staging, void* stream);
int kv_unpack_batch(kv_pool_t* dst, int32_t n, const void* const* h_d_staging,
                    const int32_t* h_tokens, const int32_t* h_token_offsets,
                    const int32_t* const* h_d_block_ids, const int32_t* h_n_ids, void* stream);

/* Direct one-shot handoff: the composition
 * kv_unpack(kv_pack(.)) in ONE kernel with no staging message.
 * §4: "the resulting KV cache is transferred once to the bound decoder";
 * PAPER.md:96 §3.1 / Fig. 3: the transfer is the cost the handoff adds.  The
 * kernel runs on the CURRENT device, which must be the one holding d_k / d_v
 * (the prefiller), and pushes 16-byte stores into `dst`'s memory; dst's
 * d_base may be local (two pools on one GPU) or a PEER mapping of the
 * decoder's pool (csv_ipc_open below, or cudaDeviceEnablePeerAccess inside
 * one process): the stores then cross NVLink and nothing is loaded from the
 * peer.  d_k, d_v: [NL][tokens][Hkv][d] bf16, 16-byte aligned, as kv_pack.
 * d_block_ids: the conversation's table as kv_unpack, readable on the current
 * device (the router sends the ids with the binding: a few KB).  Result in the
 * pool: bit-identical to kv_unpack(kv_pack(.)); slots not addressed are NOT
 * written.  Ordering across GPUs is the caller's: the decoder may read the
 * blocks after the prefiller's stream has passed this call (event / message). */
int kv_handoff_direct(kv_pool_t* dst, const void* d_k, const void* d_v, int32_t tokens, int32_t token_offset,
                      const int32_t* d_block_ids, int32_t n_ids, void* stream);
int kv_handoff_direct_batch(kv_pool_t* dst, int32_t n, const void* const* h_d_k, const void* const* h_d_v,
                            const int32_t* h_tokens, const int32_t* h_token_offsets,
                            const int32_t* const* h_d_block_ids, const int32_t* h_n_ids, void* stream);

/* Peer mapping for one process per GPU (CUDA IPC), so that a prefiller
 * process can wrap a decoder process's pool memory in its own kv_pool_t
 * (kv_pool_create over the opened pointer; the ALLOCATOR state stays with the
 * decoder, which allocates the blocks and sends their ids).
 * csv_ipc_export: d_ptr is any device pointer inside a cudaMalloc allocation
 *   of the calling process; writes the CSV_IPC_HANDLE_BYTES-byte handle of the
 *   allocation and d_ptr's byte offset inside it.  Host bytes, sendable over
 *   any channel (torch.distributed object collectives in the tests).
 * csv_ipc_open: in another process, maps the allocation (peer access enabled
 *   lazily when it lives on another GPU) and returns base + offset.
 *   Opens of the same allocation are counted (several exported pointers may
 *   share one allocation); the mapping goes away with the last close.
 * csv_ipc_mapped_bytes: d_ptr is what csv_ipc_open returned; writes how many bytes of the mapped allocation lie
 *   at and after d_ptr (0 if the sender's offset points past its end).  The opener uses it to refuse a pool
 *   descriptor that claims more memory than the sender really shared, before wrapping the pointer in a kv_pool_t:
 *   shape and offset arrive in the same untrusted message as the handle.
 * csv_ipc_close: d_ptr is what csv_ipc_open returned (one close per open).
 * csv_ipc_copy: copy-engine transfer (cudaMemcpyAsync, device to device) of
 *   `bytes` bytes between two device pointers of which either may be a
 *   csv_ipc_open mapping: the staged route's "send the message" step
 *   (kv_pack locally, copy the staging message to the decoder, kv_unpack there),
 *   kept as the comparison arm of kv_handoff_direct.  Enqueued
 *   on `stream`, never synchronises.
 * Errors: CSV_E_INVAL bad argument / unknown pointer, CSV_E_CUDA otherwise. */
#define CSV_IPC_HANDLE_BYTES 64
int csv_ipc_export(const void* d_ptr, void* out_handle, uint64_t* out_offset);
int csv_ipc_open(const void* handle, uint64_t offset, void** out_d_ptr);
int csv_ipc_mapped_bytes(const void* d_ptr, size_t* out_bytes);
int csv_ipc_close(void* d_ptr);
int csv_ipc_copy(void* d_dst, const void* d_src, size_t bytes, void* stream);

/* Tail-step KV append ("appending one new entry"; PAPER.md:94
 * "only calculating new KV cache entries for the appended tokens"): writes the
 * new tokens' K/V of a whole batch straight from token-major projections into
 * the pool — the composition kv_unpack(kv_pack(.)) without the staging round
 * trip.  d_k_new, d_v_new: [NL][total_q][Hkv][d] bf16 where total_q = sum of
 * the plan's q_lens; conversation b's rows start at sum_{b'<b} q_len[b'] and go
 * to positions [kv_len[b] - q_len[b], kv_len[b]).  d_block_tables:
 * [batch][max_blocks] int32. */
int kv_append_tokens(kv_pool_t* dst, const csv_plan_t* plan, const void* d_k_new, const void* d_v_new,
                     const int32_t* d_block_tables, int32_t max_blocks, void* stream);

/* ------------------------------------------------------------------------
 * Step plan (host).  Lengths are per step, not per layer: one plan serves all
 * layers of a step and both attention calls.  Conversation b has q_len[b] new
 * query rows and kv_len[b] tokens in the cache INCLUDING those rows' own K/V
 * (the caller writes them first; a token attends to itself).  q_len 1 =
 * decode row, q_len m > 1 = appended chunk with prefix P = kv_len - m.
 *
 * Split-K: the flattened (conversation, block) stream of the q_len = 1 rows is
 * cut into one contiguous share per warp-worker (7 per CTA at head_dim 128, 8 at 64), and each share into
 * partitions that never cross a (conversation, KV head) boundary and, if
 * max_partition_tokens > 0 (a multiple of 16), hold at most that many tokens
 * (0 = no extra cut).  The schedule depends only on the lengths, so
 * results are bit-identical under any block permutation and from run to run.
 * ---------------------------------------------------------------------- */

/* Tuning overrides (measurement aids; the defaults are what the bench times).  One process-wide table, read when a
 * plan is BUILT (csv_plan_workspace_bytes, csv_plan_create, the *_host calls) and recorded in it: later changes do not
 * affect existing plans, and a workspace size always matches a plan built under the same settings.  value 0 = default.
 *   CSV_TUNE_DECODE_GRID        cap on the CTAs of the decode launch (default: one per SM)
 *   CSV_TUNE_TAIL_DECODE_CTAS   decode-role CTAs of a mixed step's one launch, also where the planner would have kept
 *                               the two kernels (default: chosen from the two roles' work, conserve_kv.h csv_tail_step)
 *   CSV_TUNE_TAIL_TWO_KERNELS   non-zero: csv_tail_step never uses the one-launch route for plans built from now on
 *   CSV_TUNE_SM_DECODE_GBS      GB/s ONE SM pulls in the decode role (default 75) and
 *   CSV_TUNE_SM_APPEND_GFLOPS   GFLOP/s one SM sustains in the append role (default 7400): the two rates from which a
 *                               mixed step's split is computed; a caller that calibrated its own device sets both
 * At first use each knob is initialised from the environment variable of the same name without "TUNE_"
 * (CSV_DECODE_GRID, CSV_TAIL_DECODE_CTAS, CSV_SM_DECODE_GBS, CSV_SM_APPEND_GFLOPS: a positive decimal integer, anything
 * else is ignored; CSV_TAIL_TWO_KERNELS: any value other than 0).  Not thread-safe against concurrent plan builds.  csv_tuning_get returns -1 for a bad knob. */
#define CSV_TUNE_DECODE_GRID       0
#define CSV_TUNE_TAIL_DECODE_CTAS  1
#define CSV_TUNE_TAIL_TWO_KERNELS  2
#define CSV_TUNE_SM_DECODE_GBS     3
#define CSV_TUNE_SM_APPEND_GFLOPS  4
#define CSV_TUNE_COUNT             5
int csv_tuning_set(int32_t knob, int32_t value);
int32_t csv_tuning_get(int32_t knob);

/* Device workspace the plan needs (partials, work lists), for these lengths. */
size_t csv_plan_workspace_bytes(const csv_attn_shape* shape, const int32_t* h_q_lens,
                                const int32_t* h_kv_lens, int32_t batch, int32_t max_partition_tokens);
/* Builds the plan and enqueues the copy of its work lists into d_workspace
 * (128-byte aligned) on `stream`.  q_len[b] must be in [0, kv_len[b]]
 * (a row's own K/V is already counted in kv_len), with one exception: a decode
 * row on an EMPTY cache, q_len = 1 and kv_len = 0, is accepted and gives
 * O = 0, LSE = -inf (kv_append_tokens / the fused steps write nothing for it).
 * Any other q_len > kv_len -> CSV_E_INVAL.  q_len = 0 rows are inert.  The plan may be used on that stream (or after
 * synchronising with it) until destroyed; the workspace must outlive it.
 * Launches of the SAME call on one plan share workspace (the decode partials;
 * the append partials and the append kernel's work queue): they must be
 * ordered on the device (same stream, or events), never concurrent.  A decode
 * call and an append call of one plan use disjoint regions and may overlap.
 * One plan serves all the layers of a step in turn.
 * d_workspace = NULL builds a host-only plan (no device memory is touched; the
 * only CUDA runtime call is the SM-count query of the current device, 148 being
 * assumed when there is none): good for csv_plan_info / csv_plan_*_items,
 * refused (CSV_E_INVAL) by the attention calls.
 * ws_bytes too small -> CSV_E_NOMEM. */
int csv_plan_create(const csv_attn_shape* shape, const int32_t* h_q_lens, const int32_t* h_kv_lens,
                    int32_t batch, int32_t max_partition_tokens, void* d_workspace, size_t ws_bytes,
                    void* stream, csv_plan_t** out);
int csv_plan_destroy(csv_plan_t* plan);
/* Introspection for tests / bench: number of decode work items (partitions),
 * number of decode rows, of append chunks, sum of append q rows, CTAs used. */
int csv_plan_info(const csv_plan_t* plan, int32_t* n_decode_items, int32_t* n_decode_rows,
                  int32_t* n_append_chunks, int32_t* n_append_rows, int32_t* decode_grid);
/* Warp-workers of the decode launch = rows of h_worker_begin minus one (CTAs x workers per CTA: 7 at head_dim 128, 8 at 64). */
int32_t csv_plan_decode_workers(const csv_plan_t* plan);

/* The mixed-step split of a plan (csv_tail_step at head_dim 128 with decode rows AND chunks): how many CTAs of the one
 * launch start in the decode role and into how many shares their work is cut; 0, 0 when the plan has no fused launch. */
int csv_plan_tail_split(const csv_plan_t* plan, int32_t* n_decode_ctas, int32_t* n_decode_shares);
/* Sum of the plan's q_lens (rows of d_q / d_out for append_prefill_attn); -1 on NULL. */
int32_t csv_plan_total_q(const csv_plan_t* plan);
/* Copies the decode work list for inspection (host tests): item i is 8 int32
 * {conv, kv_head, blk_begin, blk_end, kv_len, partial, direct, q_row} at h_out[8*i];
 * h_worker_begin[w] .. h_worker_begin[w+1] are the items of warp-worker w
 * (csv_plan_decode_workers(plan) of them).  Either output may be NULL.  Returns the item count. */
int32_t csv_plan_decode_items(const csv_plan_t* plan, int32_t* h_out, int32_t max_items,
                              int32_t* h_worker_begin, int32_t max_workers_plus_1);
/* Same for the append work list: item i is 12 int32 {conv, kv_head, row_begin,
 * q_start, m, kv_len, blk_begin, blk_end, partial, direct, 0, 0}; rows are the
 * m * G query rows of a chunk stacked token-major (row = token * G + head_in_group),
 * in tiles of 256 rows
 * (head_dim 128) or 64 rows (head_dim 64).  Returns the item count. */
int32_t csv_plan_append_items(const csv_plan_t* plan, int32_t* h_out, int32_t max_items);

/* ------------------------------------------------------------------------
 * a4. paged_decode_attn.  PAPER.md:50 §2.1: decode "generates each subsequent
 * token by reading the full KV cache"; §3.2 / Fig. 4: the
 * tail is bandwidth-bound.  For every conversation b of the plan with
 * q_len[b] = 1 and every query head h (KV head h / G):
 *     s_j = q . K_j / sqrt(d),  j in [0, kv_len[b])
 *     O   = sum_j softmax(s)_j V_j          (bf16, round-to-nearest-even)
 *     LSE = ln sum_j exp(s_j)               (fp32, natural log)
 * kv_len = 0 (empty cache) -> O = 0 (all bits zero), LSE = -inf.  bf16 inputs, fp32 scores / softmax /
 * accumulation; softmax weights are rounded to bf16 for the PV product.
 *
 * d_q:   [total_q][Hq][d] bf16, 16-byte aligned, total_q = sum of ALL q_lens of the plan in
 *        batch order (= [batch][Hq][d] when every q_len is 1); conversation b's row is
 *        sum_{b'<b} q_len[b'] and is read only if q_len[b] = 1.
 * d_block_tables: [batch][max_blocks] int32; entries past ceil(kv_len/16) are never read.
 * d_out: [total_q][Hq][d] bf16;  d_lse: [total_q][Hq] fp32.  Rows with q_len != 1 are untouched.
 * Pool slots past kv_len in the last block may hold anything (NaN patterns included).
 * ---------------------------------------------------------------------- */
int paged_decode_attn(const csv_plan_t* plan, const kv_pool_t* pool, int32_t layer, const void* d_q,
                      const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse,
                      void* stream);

/* paged_decode_attn for callers that cannot allocate device memory and have no workspace to pass.
 *
 * Two kinds of caller are meant.  (1) A decoder that gave all of its HBM to the KV pool at start-up
 * (§5.1: a decoder's memory is its ~300k-token KV budget): later cudaMalloc calls may simply fail.
 * (2) A step that runs inside an engine which owns the device allocator, where cudaMalloc / cudaFree are off
 * limits because they can fail mid-request and stall every stream of the device while they run.
 * Every other attention call here needs a caller-owned plan workspace; this one needs only inputs and outputs.
 *
 * It builds the step's split-K plan on the host (host heap only), puts the work lists and the fp32 partials in
 * a fixed CSV_STATIC_SCRATCH_BYTES array that is part of the library's device image, and runs the same kernels
 * as paged_decode_attn: every conversation b in [0, batch) is one decode row (q_len 1) over h_kv_lens[b] cached
 * tokens, with d_q / d_out [batch][Hq][d] bf16, d_lse [batch][Hq] fp32, d_block_tables [batch][max_blocks];
 * results, kv_len = 0 behaviour and precision are those of paged_decode_attn on the same lengths and
 * max_partition_tokens (bit-identical: same plan, same kernels).  No cudaMalloc, cudaFree, pinned-host or other
 * allocating CUDA call is made; the call enqueues on `stream` and returns without synchronising.
 *
 * Limits and sharing, all of which the caller has to know:
 *  - The array costs CSV_STATIC_SCRATCH_BYTES (8 MiB) on EVERY GPU on which this library's code is loaded, for
 *    the life of the process, used or not.
 *  - A step whose plan needs more than that returns CSV_E_NOMEM and launches nothing (csv_plan_workspace_bytes
 *    with q_lens all 1 tells the need in advance; BASELINE.json's five configs need 0.03 - 4.9 MB).
 *  - One array per GPU, shared by every call: a call overwrites what the previous one left (it re-uploads its
 *    lists, queue words included, and only reads partial slots it has written itself, so nothing stale is ever
 *    consumed), and calls that overlap on one GPU (two streams, two threads) corrupt each other.  Keep them on
 *    one stream or order them with events.
 *  - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *    current).  Make that first call before starting any stream capture on the device.
 * Errors: CSV_E_INVAL (bad pointer / alignment / shape / layer, negative length, max_blocks too small),
 * CSV_E_NOMEM (over the limit above), CSV_E_CUDA. */
#define CSV_STATIC_SCRATCH_BYTES (8u << 20)
int paged_decode_attn_static(const kv_pool_t* pool, int32_t layer, const csv_attn_shape* shape, int32_t batch,
                             const int32_t* h_kv_lens, int32_t max_partition_tokens, const void* d_q,
                             const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse,
                             void* stream);

/* Fused decode tail step (§2.1: decode "generates each subsequent token by reading the
 * full KV cache and appending one new entry"): kv_append_tokens for the q_len = 1 rows of ONE layer
 * and paged_decode_attn in a single launch.  d_k_new, d_v_new: this layer's new-token K / V,
 * [total_q][Hkv][d] bf16 (rows of conversations with q_len != 1 are ignored: use kv_append_tokens
 * for appended chunks).  The warp that streams a conversation's last block patches the new token's
 * rows into the landed tiles and writes them to the pool at position kv_len - 1; results and all
 * other arguments are exactly those of kv_append_tokens followed by paged_decode_attn. */
int paged_decode_step(const csv_plan_t* plan, kv_pool_t* pool, int32_t layer, const void* d_q,
                      const void* d_k_new, const void* d_v_new, const int32_t* d_block_tables,
                      int32_t max_blocks, void* d_out, float* d_lse, void* stream);

/* ------------------------------------------------------------------------
 * a5. append_prefill_attn.  PAPER.md:94 §3.1: "relatively small prompts are
 * appended to the whole history context ... only calculating new KV cache
 * entries for the appended tokens"; §2.2: appends run on the
 * decoder holding the cached prefix.  For every conversation b with
 * q_len[b] = m > 1: query row i (position P + i, P = kv_len - m) attends to
 * keys 0 .. P + i (prefix fully visible, causal inside the chunk, diagonal
 * included).  Same softmax, outputs and precision as paged_decode_attn.
 *
 * d_q / d_out / d_lse: the same [total_q] buffers as paged_decode_attn (decode
 * rows are skipped here), so one step's two calls fill one output.
 * ---------------------------------------------------------------------- */
int append_prefill_attn(const csv_plan_t* plan, const kv_pool_t* pool, int32_t layer, const void* d_q,
                        const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse,
                        void* stream);

/* One tail step of a MIXED batch on one layer (PAPER.md:112 /
 * Fig. 5: decode rows and appended chunks run in the same iteration on the
 * decoder that holds their prefixes): writes every new row's K/V into the
 * pool, then attends.  Same results as kv_append_tokens (on this layer) +
 * paged_decode_attn + append_prefill_attn.  With decode rows AND chunks in the
 * plan (head_dim 128) the attention is ONE persistent launch whose work items
 * are both kinds: some CTAs stream the decode rows' KV (HBM-bound), the others
 * run the chunks on the tensor cores, and a CTA that finishes its decode share
 * takes chunk items (tail_fused.cu); the KV write precedes it as its own
 * kernel, chained by programmatic dependent launch.  With no appended chunk in
 * the plan it is paged_decode_step (KV write inside the decode launch).
 * d_q, d_out: [total_q][Hq][d]; d_k_new, d_v_new: [total_q][Hkv][d] bf16 of
 * THIS layer; rows ordered as in the plan.  d_k_new = d_v_new = NULL: the rows
 * are already in the pool, attention only.  Results are bit-identical from
 * run to run for a fixed plan.  Capturable in a CUDA graph (the bench does so).
 * Errors as the calls above. */
int csv_tail_step(const csv_plan_t* plan, kv_pool_t* pool, int32_t layer, const void* d_q, const void* d_k_new,
                  const void* d_v_new, const int32_t* d_block_tables, int32_t max_blocks, void* d_out, float* d_lse,
                  void* stream);

/* ------------------------------------------------------------------------
 * End-to-end convenience with HOST buffers (what bench.py's "e2e" times): one
 * tail step (decode rows and appended chunks in one iteration)
 * over layers [layer_begin, layer_begin + n_layers) of the pool.
 * h_q_lens[batch]: 1 = decode row, > 1 = appended chunk, 0 = inert; NULL = all 1.
 * h_kv_lens[batch]: cached tokens INCLUDING the new rows.  Per layer the rows
 * are ordered as in a plan (total_q = sum of q_lens):
 *   h_q, h_out:         [n_layers][total_q][Hq][d]  bf16
 *   h_k_new, h_v_new:   [n_layers][total_q][Hkv][d] bf16
 *   h_lse:              [n_layers][total_q][Hq]     fp32
 *   h_block_tables:     [batch][max_blocks] (one table serves all layers)
 * The call enqueues the host->device copies, builds ONE plan for the step while
 * they fly (lengths are per step, not per layer), runs csv_tail_step on every
 * layer, copies O and LSE back and synchronises `stream`.  Host buffers should
 * be pinned.  d_workspace: >= csv_tail_step_host_workspace_bytes(...), 128-byte
 * aligned.  Errors as csv_plan_create / csv_tail_step.  Every CSV_E_INVAL case
 * (pointers, shape, lengths, partition size) and a workspace smaller than the
 * buffers is refused before anything is enqueued.  A workspace that holds the
 * buffers but not the plan (CSV_E_NOMEM) or a CUDA failure part-way is only found
 * after the input copies were enqueued: the call then synchronises `stream`
 * before returning the error, so no DMA from the host buffers is left in flight
 * (the pool may hold some layers' new rows; outputs are unspecified).
 * ---------------------------------------------------------------------- */
size_t csv_tail_step_host_workspace_bytes(const csv_attn_shape* shape, const int32_t* h_q_lens, const int32_t* h_kv_lens,
                                          int32_t batch, int32_t max_blocks, int32_t n_layers,
                                          int32_t max_partition_tokens);
int csv_tail_step_host(kv_pool_t* pool, int32_t layer_begin, int32_t n_layers, const csv_attn_shape* shape, int32_t batch,
                       const int32_t* h_q_lens, const int32_t* h_kv_lens, const void* h_q, const void* h_k_new,
                       const void* h_v_new, const int32_t* h_block_tables, int32_t max_blocks, int32_t max_partition_tokens,
                       void* d_workspace, size_t ws_bytes, void* h_out, float* h_lse, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CONSERVE_KV_H_ */
