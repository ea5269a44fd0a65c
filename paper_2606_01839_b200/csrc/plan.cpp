// plan.cpp — host-side step planner: split-K work lists for paged_decode_attn and
// append_prefill_attn.  Pure host arithmetic on the lengths; the only CUDA call is the
// asynchronous copy of the finished lists into the caller's workspace (in api.cpp).
//
// Decode (SURVEY §7 hard part 4, BASELINE.json config 5 "split-K across >= 64 partitions"):
// the (conversation, KV head, block) stream of all q_len = 1 rows is flattened in that order
// and cut into one contiguous share per WARP-worker (decode_grid CTAs x kDecodeWarps warps),
// so every worker streams the same number of 8 KiB (K tile + V tile) units whatever the
// length mix.  A share is cut further at (conversation, head) boundaries and, if the caller asks for
// it, every max_partition_tokens tokens (the default adds no cut: equal shares already balance the
// load, and every extra partition is one more partial to merge).  Each piece is one DecodeItem = one
// partial (o, m, l).  Config 5 (16 x 131072 tokens) still gets >= 64 partitions per sequence: each of
// its 8 KV heads spans ~9.25 shares.
// The schedule depends only on the lengths: results are bit-identical under any block
// permutation and from run to run.
#include <stdlib.h>

#include <algorithm>
#include <new>

#include "internal.h"

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// A knob from the environment: a positive decimal integer, or (two-kernel switch only) any non-empty value = 1.
// Anything else is ignored rather than guessed at (atoi of garbage used to give a one-CTA grid).
static int32_t env_knob(const char* name, bool flag) {
    const char* e = getenv(name);
    if (!e || !*e) return 0;
    char* end = nullptr;
    const long v = strtol(e, &end, 10);
    if (end != e && *end == 0 && v > 0 && v <= (1 << 20)) return (int32_t)v;
    return (flag && !(end != e && *end == 0)) ? 1 : 0;   // flag: "yes", "on", ... count as set; "0" does not
}

CsvTuning& csv_tuning() {
    static CsvTuning t = {{env_knob("CSV_DECODE_GRID", false), env_knob("CSV_TAIL_DECODE_CTAS", false),
                           env_knob("CSV_TAIL_TWO_KERNELS", true), env_knob("CSV_SM_DECODE_GBS", false),
                           env_knob("CSV_SM_APPEND_GFLOPS", false)}};
    return t;
}

static bool attn_shape_ok(const csv_attn_shape* s) {
    if (!s) return false;
    if (s->block_size != CSV_BLOCK_SIZE) return false;
    if (s->head_dim != 64 && s->head_dim != 128) return false;
    const int hk = s->num_kv_heads;
    if (hk != 1 && hk != 2 && hk != 4 && hk != 8) return false;
    if (s->num_q_heads < hk || s->num_q_heads % hk != 0) return false;
    const int g = s->num_q_heads / hk;
    if (g != 1 && g != 2 && g != 4 && g != 8) return false;
    return true;
}

// Cuts the flattened (conversation, KV head, block) stream of the q_len = 1 rows into one contiguous share per worker
// (W workers) and each share into items at (conversation, head) boundaries (+ every part_blocks blocks).
static void build_decode_list(const csv_plan* p, int64_t units, int64_t W, int part_blocks, std::vector<DecodeItem>& items,
                              std::vector<int32_t>& worker_begin, std::vector<MergeGroup>& groups, int32_t& n_partials) {
    const int Hkv = p->shape.num_kv_heads;
    worker_begin.assign((size_t)W + 1, 0);
    items.clear();
    items.reserve((size_t)W + (size_t)p->n_decode_rows * Hkv + 16);
    groups.clear();
    n_partials = 0;
    if (units == 0) return;

    int64_t base = 0;   // first unit of the current (conv, head) segment
    int64_t w = 0;      // worker whose share contains `pos`
    // share k starts at floor(k * units / W) = k * sq + floor(k * sr / W): stepped without a division per item
    // (this loop is on the host path of every tail step)
    const int64_t sq = units / W, sr = units % W;
    int64_t next_start = sq, next_rem = sr;   // start of share w + 1, and (w + 1) * sr mod W
    if (next_rem >= W) {
        next_rem -= W;
        ++next_start;
    }
    for (int b = 0; b < p->batch; ++b) {
        if (p->q_lens[b] != 1 || p->kv_lens[b] == 0) continue;
        const int nblk = (p->kv_lens[b] + CSV_BLOCK_SIZE - 1) / CSV_BLOCK_SIZE;
        for (int g = 0; g < Hkv; ++g) {
            const size_t first_item = items.size();
            int blk = 0;
            while (blk < nblk) {
                const int64_t pos = base + blk;
                while (w + 1 < W && next_start <= pos) {   // advance to the worker owning pos
                    ++w;
                    worker_begin[(size_t)w] = (int32_t)items.size();
                    next_start += sq;
                    next_rem += sr;
                    if (next_rem >= W) {
                        next_rem -= W;
                        ++next_start;
                    }
                }
                const int64_t share_end = w + 1 < W ? next_start : units;   // start of share w + 1
                int end = (int)std::min<int64_t>(nblk, share_end - base);
                end = std::min(end, blk + part_blocks);
                DecodeItem it{};
                it.conv = b;
                it.head = g;
                it.blk_begin = blk;
                it.blk_end = end;
                it.kv_len = p->kv_lens[b];
                it.partial = -1;
                it.direct = 0;
                it.group = -1;
                it.q_row = p->q_start[(size_t)b];
                items.push_back(it);
                blk = end;
            }
            const size_t n = items.size() - first_item;
            if (n == 1) {
                items[first_item].direct = 1;
            } else {
                MergeGroup mg{};
                mg.first = n_partials;
                mg.count = (int32_t)n;
                mg.conv = b;
                mg.head = g;
                mg.q_start = p->q_start[(size_t)b];
                for (size_t i = 0; i < n; ++i) {
                    DecodeItem& di = items[first_item + i];
                    di.partial = n_partials++;
                    di.group = (int32_t)groups.size();
                    di.group_first = mg.first;
                    di.group_count = mg.count;
                }
                groups.push_back(mg);
            }
            base += nblk;
        }
    }
    for (int64_t k = w + 1; k <= W; ++k) worker_begin[(size_t)k] = (int32_t)items.size();
}

static int64_t decode_units(csv_plan* p) {
    const int Hkv = p->shape.num_kv_heads;
    int64_t units = 0;
    p->n_decode_rows = 0;
    p->zero_rows.clear();
    for (int b = 0; b < p->batch; ++b)
        if (p->q_lens[b] == 1) {
            units += (int64_t)((p->kv_lens[b] + CSV_BLOCK_SIZE - 1) / CSV_BLOCK_SIZE) * Hkv;
            ++p->n_decode_rows;
            if (p->kv_lens[b] == 0) p->zero_rows.push_back(p->q_start[(size_t)b]);   // empty cache: O = 0, LSE = -inf
        }
    return units;
}

static void plan_decode(csv_plan* p) {
    const int part_blocks = std::max(1, p->max_partition_tokens / CSV_BLOCK_SIZE);
    const int64_t units = decode_units(p);
    // CTAs: one per SM, fewer when there is under 4 blocks of work per warp
    const int WPC = p->decode_warps;   // warp-workers per CTA
    int64_t want = (units + (int64_t)WPC * 4 - 1) / ((int64_t)WPC * 4);
    p->decode_grid = (int)std::max<int64_t>(1, std::min<int64_t>(p->num_sms, want));
    if (const int32_t cap = csv_tuning().v[CSV_TUNE_DECODE_GRID]) p->decode_grid = std::max(1, std::min(p->decode_grid, cap));   // tuning override
    build_decode_list(p, units, (int64_t)p->decode_grid * WPC, part_blocks, p->decode_items, p->worker_begin, p->decode_groups,
                      p->n_decode_partials);
}

// Mixed step (decode rows AND appended chunks, d = 128): tail_kernel gives `tail_n_dec` CTAs the decode role (8 warp-workers
// each, a second share list cut for that many workers) and the others the append role; decode CTAs join the append queue
// when their share is done.  The split equalises the two predicted times: decode bytes / (CTAs x bandwidth one SM pulls)
// against append flops / (CTAs x tensor rate of one SM), both measured (kernels).
static void plan_tail(csv_plan* p) {
    p->tail_n_dec = 0;
    p->tail_n_shares = 0;
    p->tail_items.clear();
    p->tail_worker_begin.clear();
    p->tail_groups.clear();
    p->tail_n_partials = 0;
    if (p->shape.head_dim != 128 || p->append_items.empty() || p->decode_items.empty() || p->num_sms < 4) return;
    const int Hkv = p->shape.num_kv_heads, Hq = p->shape.num_q_heads, d = p->shape.head_dim;
    int64_t units = 0;
    double flops = 0.0;
    for (int b = 0; b < p->batch; ++b) {
        const int m = p->q_lens[b];
        if (m == 1) units += (int64_t)((p->kv_lens[b] + CSV_BLOCK_SIZE - 1) / CSV_BLOCK_SIZE) * Hkv;
        if (m > 1) flops += 4.0 * d * Hq * m * ((double)(p->kv_lens[b] - m) + (m + 1) / 2.0);
    }
    const double bytes = (double)units * 2.0 * csv_tile_bytes(d);
    // one SM: the decode role pulls ~75 GB/s, the append role sustains 7.0-7.8 TFLOP/s (one B200 pool's numbers, DESIGN.md
    // section 5: the best split moved between boxes).  A caller that has calibrated its own device passes its rates through
    // csv_tuning_set; only their ratio matters here.
    const CsvTuning& tune = csv_tuning();
    const double sm_gbs = tune.v[CSV_TUNE_SM_DECODE_GBS] ? (double)tune.v[CSV_TUNE_SM_DECODE_GBS] : 75.0;
    const double sm_tflops = tune.v[CSV_TUNE_SM_APPEND_GFLOPS] ? tune.v[CSV_TUNE_SM_APPEND_GFLOPS] / 1000.0 : 7.4;
    const double td = bytes / (sm_gbs * 1e9), ta = flops / (sm_tflops * 1e12);   // SM-seconds of each role
    // The one launch pays when the decode rows are a sizeable part of the step (configs[2]: td / (td + ta) = 0.34, one call
    // 4.53 ms against 4.73 for the two kernels back to back); with little decode work beside long chunks (configs[4]: 0.16)
    // giving SMs to the decode role for the whole launch costs more than it hides (8-layer step 46.1 against 44.4 ms), and
    // csv_tail_step keeps the two kernels.
    const int32_t force = csv_tuning().v[CSV_TUNE_TAIL_DECODE_CTAS];   // tuning override: the decode-role CTAs of the one launch
    if (td < 0.25 * (td + ta) && !force) return;
    // A decode side that is too small costs more than one that is too large (SMs that finish their decode share take chunk
    // items, while a chunk-role SM can only take over a whole share), so the split leans 8 % towards decode.
    int k = (int)(1.08 * p->num_sms * td / (td + ta) + 0.5);
    // HBM saturates near 3/4 of the SMs: more decode CTAs than that only take tensor pipes away from the chunks
    k = std::max(1, std::min(k, std::min(p->num_sms - 1, (p->num_sms * 3) / 4)));
    const int64_t want = (units + 8 * 4 - 1) / (8 * 4);
    k = (int)std::min<int64_t>(k, std::max<int64_t>(1, want));
    if (force) k = std::max(1, std::min(p->num_sms - 1, force));
    p->tail_n_dec = k;
    // shares per decode-role SM (measured on configs[2] / [4]: 1 share 4.64 / 5.07 ms, 4 shares 4.98 / 5.26 ms: every share
    // ends with a CTA-wide barrier and restarts the rings)
    const int shares = 1;
    p->tail_n_shares = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)k * shares, want));
    const int part_blocks = std::max(1, p->max_partition_tokens / CSV_BLOCK_SIZE);
    build_decode_list(p, units, (int64_t)p->tail_n_shares * 8, part_blocks, p->tail_items, p->tail_worker_begin, p->tail_groups,
                      p->tail_n_partials);
}

static void plan_append(csv_plan* p) {
    const int Hkv = p->shape.num_kv_heads;
    const int G = p->shape.num_q_heads / Hkv;
    const int TR = p->append_tile_rows = p->shape.head_dim == 128 ? kAppendTileRowsTc2 : kAppendTileRows;
    p->n_append_chunks = 0;
    p->n_append_rows = 0;
    p->append_items.clear();
    p->append_groups.clear();
    p->n_append_partials = 0;
    for (int b = 0; b < p->batch; ++b)
        if (p->q_lens[b] > 1) {
            ++p->n_append_chunks;
            p->n_append_rows += p->q_lens[b];
        }
    if (p->n_append_chunks == 0) return;

    auto count_items = [&](int split_blocks) {
        int64_t n = 0;
        for (int b = 0; b < p->batch; ++b) {
            const int m = p->q_lens[b];
            if (m <= 1) continue;
            const int P = p->kv_lens[b] - m;
            const int rows = m * G;
            for (int r0 = 0; r0 < rows; r0 += TR) {
                const int i_max = std::min(m - 1, (std::min(rows, r0 + TR) - 1) / G);
                const int nblk = (P + i_max + 1 + CSV_BLOCK_SIZE - 1) / CSV_BLOCK_SIZE;
                n += (int64_t)Hkv * ((nblk + split_blocks - 1) / split_blocks);
            }
        }
        return n;
    };
    int split_blocks;
    if (p->max_partition_tokens_user > 0) {
        split_blocks = std::max(1, p->max_partition_tokens_user / CSV_BLOCK_SIZE);
    } else {
        // largest power-of-two split (<= 2^17 tokens) that still gives >= 6 items per CTA slot
        const int64_t slots = (int64_t)p->num_sms * 2;
        split_blocks = (1 << 17) / CSV_BLOCK_SIZE;
        while (split_blocks > 2048 / CSV_BLOCK_SIZE && count_items(split_blocks) < 6 * slots) split_blocks /= 2;
    }

    for (int b = 0; b < p->batch; ++b) {
        const int m = p->q_lens[b];
        if (m <= 1) continue;
        const int P = p->kv_lens[b] - m;
        const int rows = m * G;
        for (int g = 0; g < Hkv; ++g)
            for (int r0 = 0; r0 < rows; r0 += TR) {
                const int i_max = std::min(m - 1, (std::min(rows, r0 + TR) - 1) / G);
                const int nblk = (P + i_max + 1 + CSV_BLOCK_SIZE - 1) / CSV_BLOCK_SIZE;
                const int nparts = (nblk + split_blocks - 1) / split_blocks;
                MergeGroup mg{};
                mg.first = p->n_append_partials;
                mg.count = nparts;
                mg.conv = b;
                mg.head = g;
                mg.row_begin = r0;
                mg.q_start = p->q_start[b];
                mg.m = m;
                for (int k = 0; k < nparts; ++k) {
                    AppendItem it{};
                    it.conv = b;
                    it.head = g;
                    it.row_begin = r0;
                    it.q_start = p->q_start[b];
                    it.m = m;
                    it.kv_len = p->kv_lens[b];
                    it.blk_begin = k * split_blocks;
                    it.blk_end = std::min(nblk, (k + 1) * split_blocks);
                    it.direct = nparts == 1 ? 1 : 0;
                    it.partial = nparts == 1 ? -1 : p->n_append_partials++;
                    p->append_items.push_back(it);
                }
                if (nparts > 1) p->append_groups.push_back(mg);
            }
    }
    // longest first: with the kernel's work queue (CTAs take the next item when they finish one) this is LPT
    // scheduling; static round-robin left 5-8 % imbalance on config 3.  Stable => deterministic order
    std::stable_sort(p->append_items.begin(), p->append_items.end(), [](const AppendItem& a, const AppendItem& b) {
        return (a.blk_end - a.blk_begin) > (b.blk_end - b.blk_begin);
    });
}

static void plan_layout(csv_plan* p) {
    const int d = p->shape.head_dim;
    const int G = p->shape.num_q_heads / p->shape.num_kv_heads;
    PlanLayout& L = p->lay;
    size_t off = 0;
    auto take = [&](size_t bytes) {
        const size_t at = off;
        off = align_up(off + bytes, 128);
        return at;
    };
    L.decode_items = take(p->decode_items.size() * sizeof(DecodeItem));
    L.worker_begin = take(p->worker_begin.size() * sizeof(int32_t));
    L.decode_groups = take(p->decode_groups.size() * sizeof(MergeGroup));
    L.append_items = take(p->append_items.size() * sizeof(AppendItem));
    L.append_groups = take(p->append_groups.size() * sizeof(MergeGroup));
    L.zero_rows = take(p->zero_rows.size() * sizeof(int32_t));
    L.tail_items = take(p->tail_items.size() * sizeof(DecodeItem));
    L.tail_worker_begin = take(p->tail_worker_begin.size() * sizeof(int32_t));
    L.tail_groups = take(p->tail_groups.size() * sizeof(MergeGroup));
    L.append_sched = take(128);   // zero in the uploaded image; every launcher zeroes it again (cudaMemsetAsync) before its kernel
    std::vector<int32_t> meta;
    meta.insert(meta.end(), p->q_start.begin(), p->q_start.end());
    meta.insert(meta.end(), p->kv_lens.begin(), p->kv_lens.end());
    meta.insert(meta.end(), p->q_lens.begin(), p->q_lens.end());
    L.conv_meta = take(meta.size() * sizeof(int32_t));
    const size_t list_bytes = off;
    const size_t dec_partials = (size_t)std::max(p->n_decode_partials, p->tail_n_partials);   // the two lists never run together
    L.decode_po = take(dec_partials * G * d * sizeof(float));
    L.decode_pml = take(dec_partials * G * 2 * sizeof(float));
    L.append_po = take((size_t)p->n_append_partials * p->append_tile_rows * d * sizeof(float));
    L.append_pml = take((size_t)p->n_append_partials * p->append_tile_rows * 2 * sizeof(float));
    L.total = std::max<size_t>(off, 128);
    p->h_image.assign(list_bytes, 0);
    auto put = [&](size_t at, const void* src, size_t bytes) {
        if (bytes) memcpy(p->h_image.data() + at, src, bytes);
    };
    put(L.decode_items, p->decode_items.data(), p->decode_items.size() * sizeof(DecodeItem));
    put(L.worker_begin, p->worker_begin.data(), p->worker_begin.size() * sizeof(int32_t));
    put(L.decode_groups, p->decode_groups.data(), p->decode_groups.size() * sizeof(MergeGroup));
    put(L.append_items, p->append_items.data(), p->append_items.size() * sizeof(AppendItem));
    put(L.append_groups, p->append_groups.data(), p->append_groups.size() * sizeof(MergeGroup));
    put(L.conv_meta, meta.data(), meta.size() * sizeof(int32_t));
    put(L.zero_rows, p->zero_rows.data(), p->zero_rows.size() * sizeof(int32_t));
    put(L.tail_items, p->tail_items.data(), p->tail_items.size() * sizeof(DecodeItem));
    put(L.tail_worker_begin, p->tail_worker_begin.data(), p->tail_worker_begin.size() * sizeof(int32_t));
    put(L.tail_groups, p->tail_groups.data(), p->tail_groups.size() * sizeof(MergeGroup));
}

// Builds the host side of a plan.  Returns NULL on bad arguments.
csv_plan* csv_plan_build_host(const csv_attn_shape* shape, const int32_t* h_q_lens, const int32_t* h_kv_lens,
                              int32_t batch, int32_t max_partition_tokens, int* err) {
    *err = CSV_E_INVAL;
    if (!attn_shape_ok(shape) || batch < 0 || (batch > 0 && (!h_q_lens || !h_kv_lens))) return nullptr;
    if (max_partition_tokens < 0 || max_partition_tokens % CSV_BLOCK_SIZE != 0) return nullptr;
    int64_t total_q = 0;
    for (int b = 0; b < batch; ++b) {
        // q_len <= kv_len (a row's own K/V is in the cache), except the decode row on an EMPTY cache (q_len 1, kv_len 0):
        // nothing to attend to, O = 0 and LSE = -inf (conserve_kv.h a4)
        if (h_kv_lens[b] < 0 || h_q_lens[b] < 0) return nullptr;
        if (h_q_lens[b] > h_kv_lens[b] && !(h_q_lens[b] == 1 && h_kv_lens[b] == 0)) return nullptr;
        total_q += h_q_lens[b];
    }
    if (total_q > INT32_MAX) return nullptr;
    csv_plan* p = new (std::nothrow) csv_plan();
    if (!p) {
        *err = CSV_E_NOMEM;
        return nullptr;
    }
    p->shape = *shape;
    p->batch = batch;
    p->max_partition_tokens_user = max_partition_tokens;
    p->max_partition_tokens = max_partition_tokens > 0 ? max_partition_tokens : (1 << 30);   // 0: share cuts only
    p->num_sms = csv_query_num_sms();
    p->q_lens.assign(h_q_lens, h_q_lens + batch);
    p->kv_lens.assign(h_kv_lens, h_kv_lens + batch);
    p->q_start.assign((size_t)batch + 1, 0);
    for (int b = 0; b < batch; ++b) p->q_start[(size_t)b + 1] = p->q_start[(size_t)b] + h_q_lens[b];
    p->total_q = (int32_t)total_q;
    p->d_ws = nullptr;
    p->tail_two_kernels = csv_tuning().v[CSV_TUNE_TAIL_TWO_KERNELS] != 0;
    // d = 128: 7 warp-workers x 2 ring stages per SM (112 KB in flight).  Measured against 8 x 3 (192 KB): configs[1] 184.8
    // against 201.2 us, configs[2] 2.02 against 2.12 ms, configs[4] 1.25 against 1.31 ms per layer (6 x 2: 184.8 us / 2.02 /
    // 1.23 ms): more bytes in flight than the latency needs only queue up in the memory system.
    // 7 rather than 6 keeps configs[4] at >= 64 partitions per sequence (8 KV heads x 8.1 shares) without extra cuts.
    p->decode_warps = shape->head_dim == 128 ? kDecodeWarps128 : kDecodeWarps;
    plan_decode(p);
    plan_append(p);
    plan_tail(p);
    plan_layout(p);
    *err = CSV_OK;
    return p;
}

extern "C" {

size_t csv_plan_workspace_bytes(const csv_attn_shape* shape, const int32_t* h_q_lens, const int32_t* h_kv_lens,
                                int32_t batch, int32_t max_partition_tokens) {
    int err;
    csv_plan* p = csv_plan_build_host(shape, h_q_lens, h_kv_lens, batch, max_partition_tokens, &err);
    if (!p) return 0;
    const size_t n = p->lay.total;
    delete p;
    return n;
}

int csv_tuning_set(int32_t knob, int32_t value) {
    if (knob < 0 || knob >= CSV_TUNE_COUNT || value < 0 || value > (1 << 20)) return CSV_E_INVAL;
    csv_tuning().v[knob] = value;
    return CSV_OK;
}

int32_t csv_tuning_get(int32_t knob) {
    return (knob < 0 || knob >= CSV_TUNE_COUNT) ? -1 : csv_tuning().v[knob];
}

int csv_plan_destroy(csv_plan_t* plan) {
    if (!plan) return CSV_E_INVAL;
    delete plan;
    return CSV_OK;
}

int csv_plan_info(const csv_plan_t* plan, int32_t* n_decode_items, int32_t* n_decode_rows, int32_t* n_append_chunks,
                  int32_t* n_append_rows, int32_t* decode_grid) {
    if (!plan) return CSV_E_INVAL;
    if (n_decode_items) *n_decode_items = (int32_t)plan->decode_items.size();
    if (n_decode_rows) *n_decode_rows = plan->n_decode_rows;
    if (n_append_chunks) *n_append_chunks = plan->n_append_chunks;
    if (n_append_rows) *n_append_rows = plan->n_append_rows;
    if (decode_grid) *decode_grid = plan->decode_grid;
    return CSV_OK;
}

int32_t csv_plan_decode_workers(const csv_plan_t* plan) { return plan ? (int32_t)plan->worker_begin.size() - 1 : -1; }

int csv_plan_tail_split(const csv_plan_t* plan, int32_t* n_decode_ctas, int32_t* n_decode_shares) {
    if (!plan) return CSV_E_INVAL;
    if (n_decode_ctas) *n_decode_ctas = plan->tail_n_dec;
    if (n_decode_shares) *n_decode_shares = plan->tail_n_shares;
    return CSV_OK;
}

int32_t csv_plan_total_q(const csv_plan_t* plan) { return plan ? plan->total_q : -1; }

int32_t csv_plan_decode_items(const csv_plan_t* plan, int32_t* h_out, int32_t max_items, int32_t* h_worker_begin,
                              int32_t max_workers_plus_1) {
    if (!plan) return -1;
    const int32_t n = (int32_t)plan->decode_items.size();
    if (h_out)
        for (int32_t i = 0; i < n && i < max_items; ++i) memcpy(h_out + (size_t)i * 8, &plan->decode_items[(size_t)i], 32);   // first 8 fields
    if (h_worker_begin)
        for (int32_t i = 0; i < (int32_t)plan->worker_begin.size() && i < max_workers_plus_1; ++i)
            h_worker_begin[i] = plan->worker_begin[(size_t)i];
    return n;
}

int32_t csv_plan_append_items(const csv_plan_t* plan, int32_t* h_out, int32_t max_items) {
    if (!plan) return -1;
    const int32_t n = (int32_t)plan->append_items.size();
    if (h_out)
        for (int32_t i = 0; i < n && i < max_items; ++i) memcpy(h_out + (size_t)i * 12, &plan->append_items[(size_t)i], 48);
    return n;
}

}   // extern "C"
