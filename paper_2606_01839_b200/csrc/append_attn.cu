// append_attn.cu — append_prefill_attn (a5): causal attention of an m-token appended chunk
// (a tool output) against its cached prefix plus itself.  PAPER.md:94 §3.1: "relatively small
// prompts are appended to the whole history context ... only calculating new KV cache entries
// for the appended tokens"; §2.2: appends run on the decoder holding the prefix.
//
// Roofline: tensor cores when m*G >~ 213 stacked rows per KV byte, HBM below.
//
// The m query tokens x G heads of one KV head are stacked token-major (row r = i*G + hh) into
// tiles of 64 rows: one K/V tile read serves all G heads and the causal diagonal stays tight
// (a 16-row MMA tile spans 16/G tokens).  A CTA (4 warps x 16 rows) streams the visible KV
// blocks of its tile through a 3-stage ring of 4 blocks (64 tokens, 32 KiB) filled by 1-D
// bulk copies (UBLKCP), FA2-style register-resident S/P/O on mma.sync.m16n8k16.  Long
// prefixes are cut into KV partitions (plan.cpp) with the same (o, m, l) partial format as
// decode and a fixed-order merge.
#include <math.h>

#include "common.cuh"
#include "internal.h"

namespace {

constexpr int kAppendWarps = 4;
constexpr int kStageBlocks = 4;
constexpr int kAppendStages = 3;

struct AppendParams {
    const AppendItem* items;
    int32_t n_items;
    const uint8_t* pool_layer;
    const uint16_t* q;
    const int32_t* tables;
    uint16_t* out;
    float* lse;
    float* po;
    float* pml;
    int32_t max_blocks, Hq, Hkv, G;
    float scale_log2;
};

template <int D>
__global__ void __launch_bounds__(kAppendWarps * 32, 2) append_kernel(const __grid_constant__ AppendParams p) {
    constexpr int TB = 16 * D * 2;
    constexpr int SB = kStageBlocks * 2 * TB;
    constexpr int KS = D / 16;
    constexpr int NT = D / 8;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)kAppendStages * SB);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int row = lane >> 2, t4 = lane & 3;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kAppendStages; ++s) mbar_init(&bars[s], 1);
        fence_mbar_init();
    }
    __syncthreads();

    const int G = p.G;
    const size_t kv_stride = (size_t)p.Hkv * TB;
    const size_t blk_stride = 2 * kv_stride;
    const int mi = lane >> 3, r8 = lane & 7;
    const uint32_t k_lane_off = (uint32_t)((r8 + 8 * (mi >> 1)) * 128 + (((mi & 1) ^ r8) << 4));
    const uint32_t v_lane_off = (uint32_t)((r8 + 8 * (mi & 1)) * 128 + (((mi >> 1) ^ r8) << 4));
    const uint32_t smem_base = smem_u32(smem);

    uint32_t cnt = 0;   // stages consumed by this CTA (ring position), CTA-uniform
    for (int it = blockIdx.x; it < p.n_items; it += gridDim.x) {
        const int4 i0 = __ldg(reinterpret_cast<const int4*>(p.items + it));
        const int4 i1 = __ldg(reinterpret_cast<const int4*>(p.items + it) + 1);
        const int4 i2 = __ldg(reinterpret_cast<const int4*>(p.items + it) + 2);
        const int conv = i0.x, head = i0.y, row_begin = i0.z, q_start = i0.w;
        const int m = i1.x, kv_len = i1.y, blk_begin = i1.z, blk_end = i1.w;
        const int partial = i2.x, direct = i2.y;
        const int P = kv_len - m;
        const int rows_total = m * G;
        const int nblk = blk_end - blk_begin;
        const int nst = (nblk + kStageBlocks - 1) / kStageBlocks;
        const int32_t* tab = p.tables + (size_t)conv * p.max_blocks + blk_begin;
        const uint8_t* head_base = p.pool_layer + (size_t)head * TB;

        // rows of this thread: r_lo, r_hi = r_lo + 8 (stacked row index inside the chunk)
        const int r_lo = row_begin + warp * 16 + row, r_hi = r_lo + 8;
        const bool ok_lo = r_lo < rows_total, ok_hi = r_hi < rows_total;
        // last visible key of each row; rows past the chunk see everything (their Q is zero)
        const int lim_lo = ok_lo ? P + r_lo / G : kv_len - 1;
        const int lim_hi = ok_hi ? P + r_hi / G : kv_len - 1;
        const int w_first = row_begin + warp * 16;
        const int w_min_lim = w_first < rows_total ? P + w_first / G : kv_len - 1;
        const int w_last = min(w_first + 15, rows_total - 1);
        const int w_max_lim = w_first < rows_total ? P + w_last / G : -1;   // -1: warp has no row at all

        uint32_t qa[KS][4];
        {
            const uint16_t* q_lo = p.q + ((size_t)(q_start + (ok_lo ? r_lo / G : 0)) * p.Hq + (size_t)head * G + (ok_lo ? r_lo % G : 0)) * D;
            const uint16_t* q_hi = p.q + ((size_t)(q_start + (ok_hi ? r_hi / G : 0)) * p.Hq + (size_t)head * G + (ok_hi ? r_hi % G : 0)) * D;
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                qa[ks][0] = ok_lo ? *reinterpret_cast<const uint32_t*>(q_lo + ks * 16 + 2 * t4) : 0u;
                qa[ks][1] = ok_hi ? *reinterpret_cast<const uint32_t*>(q_hi + ks * 16 + 2 * t4) : 0u;
                qa[ks][2] = ok_lo ? *reinterpret_cast<const uint32_t*>(q_lo + ks * 16 + 8 + 2 * t4) : 0u;
                qa[ks][3] = ok_hi ? *reinterpret_cast<const uint32_t*>(q_hi + ks * 16 + 8 + 2 * t4) : 0u;
            }
        }
        float o[NT][4];
#pragma unroll
        for (int n = 0; n < NT; ++n) o[n][0] = o[n][1] = o[n][2] = o[n][3] = 0.f;
        float m_lo = -INFINITY, m_hi = -INFINITY, l_lo = 0.f, l_hi = 0.f;

        // producer state (thread 0): ids of the next stage to issue
        int nid[kStageBlocks];
        int next_issue = 0;
        auto load_ids = [&](int st) {
#pragma unroll
            for (int j = 0; j < kStageBlocks; ++j) {
                const int b = st * kStageBlocks + j;
                nid[j] = b < nblk ? __ldg(tab + b) : 0;
            }
        };
        auto issue_stage = [&](int st, uint32_t ring_pos) {
            const uint32_t stage = ring_pos % kAppendStages;
            const int nb = min(kStageBlocks, nblk - st * kStageBlocks);
            uint8_t* dst = smem + (size_t)stage * SB;
            mbar_expect_tx(&bars[stage], (uint32_t)nb * 2 * TB);
#pragma unroll
            for (int j = 0; j < kStageBlocks; ++j)
                if (j < nb) {
                    const uint8_t* src = head_base + (size_t)nid[j] * blk_stride;
                    bulk_g2s(dst + (size_t)j * 2 * TB, src, TB, &bars[stage]);
                    bulk_g2s(dst + (size_t)j * 2 * TB + TB, src + kv_stride, TB, &bars[stage]);
                }
        };
        if (threadIdx.x == 0) {
            load_ids(0);
            const int npro = nst < kAppendStages ? nst : kAppendStages;
            for (; next_issue < npro; ++next_issue) {
                issue_stage(next_issue, cnt + next_issue);
                load_ids(next_issue + 1);
            }
        }

        for (int st = 0; st < nst; ++st) {
            const uint32_t stage = cnt % kAppendStages, parity = (cnt / kAppendStages) & 1u;
            mbar_wait(&bars[stage], parity);
            const int nb = min(kStageBlocks, nblk - st * kStageBlocks);
            const int tok0 = (blk_begin + st * kStageBlocks) * 16;
            if (tok0 + nb * 16 > kv_len) {   // CTA-uniform: the conversation's partial last block
                const int nvalid = kv_len - (tok0 + (nb - 1) * 16);
                uint8_t* vtile = smem + (size_t)stage * SB + (size_t)(nb - 1) * 2 * TB + TB;
                for (int c = threadIdx.x; c < TB / 16; c += kAppendWarps * 32)
                    if (((c & 127) >> 3) >= nvalid) *reinterpret_cast<uint4*>(vtile + c * 16) = make_uint4(0, 0, 0, 0);
                fence_proxy_async();
                __syncthreads();
            }
            if (tok0 <= w_max_lim) {
                for (int jb = 0; jb < nb; ++jb) {
                    const int tokb = tok0 + jb * 16;
                    if (tokb > w_max_lim) break;   // warp-uniform: nothing visible from here on
                    const uint32_t kt = smem_base + stage * SB + jb * 2 * TB, vt = kt + TB;
                    float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                    for (int ks = 0; ks < KS; ++ks) {
                        uint32_t b[4];
                        ldsm_x4(b, kt + (ks >> 2) * 2048 + (k_lane_off ^ (((2 * ks) & 7) << 4)));
                        mma_bf16(s0, qa[ks], b[0], b[1]);
                        mma_bf16(s1, qa[ks], b[2], b[3]);
                    }
                    // [0],[1]: row lo; [2],[3]: row hi.  s0: tokens +0..7, s1: tokens +8..15
                    float sv[8] = {s0[0] * p.scale_log2, s0[1] * p.scale_log2, s1[0] * p.scale_log2, s1[1] * p.scale_log2,
                                   s0[2] * p.scale_log2, s0[3] * p.scale_log2, s1[2] * p.scale_log2, s1[3] * p.scale_log2};
                    if (tokb + 15 > w_min_lim) {
                        const int j0 = tokb + 2 * t4;
                        if (j0 > lim_lo) sv[0] = -INFINITY;
                        if (j0 + 1 > lim_lo) sv[1] = -INFINITY;
                        if (j0 + 8 > lim_lo) sv[2] = -INFINITY;
                        if (j0 + 9 > lim_lo) sv[3] = -INFINITY;
                        if (j0 > lim_hi) sv[4] = -INFINITY;
                        if (j0 + 1 > lim_hi) sv[5] = -INFINITY;
                        if (j0 + 8 > lim_hi) sv[6] = -INFINITY;
                        if (j0 + 9 > lim_hi) sv[7] = -INFINITY;
                    }
                    float mx_lo = fmaxf(fmaxf(sv[0], sv[1]), fmaxf(sv[2], sv[3]));
                    float mx_hi = fmaxf(fmaxf(sv[4], sv[5]), fmaxf(sv[6], sv[7]));
                    mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 1));
                    mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 1));
                    mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, 2));
                    mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, 2));
                    const float mn_lo = fmaxf(m_lo, mx_lo), mn_hi = fmaxf(m_hi, mx_hi);
                    if (__any_sync(0xffffffffu, mn_lo > m_lo || mn_hi > m_hi)) {
                        // a row that has seen no key yet keeps m = -inf: use 0 as its reference (all its p are 0)
                        const float a_lo = fast_exp2(m_lo - (mn_lo == -INFINITY ? 0.f : mn_lo));
                        const float a_hi = fast_exp2(m_hi - (mn_hi == -INFINITY ? 0.f : mn_hi));
                        l_lo *= a_lo;
                        l_hi *= a_hi;
#pragma unroll
                        for (int n = 0; n < NT; ++n) {
                            o[n][0] *= a_lo;
                            o[n][1] *= a_lo;
                            o[n][2] *= a_hi;
                            o[n][3] *= a_hi;
                        }
                        m_lo = mn_lo;
                        m_hi = mn_hi;
                    }
                    const float ref_lo = m_lo == -INFINITY ? 0.f : m_lo, ref_hi = m_hi == -INFINITY ? 0.f : m_hi;
                    float pv[8];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        pv[k] = fast_exp2(sv[k] - ref_lo);
                        pv[4 + k] = fast_exp2(sv[4 + k] - ref_hi);
                    }
                    l_lo += (pv[0] + pv[1]) + (pv[2] + pv[3]);
                    l_hi += (pv[4] + pv[5]) + (pv[6] + pv[7]);
                    uint32_t pa[4] = {pack_bf16(pv[0], pv[1]), pack_bf16(pv[4], pv[5]), pack_bf16(pv[2], pv[3]),
                                      pack_bf16(pv[6], pv[7])};
#pragma unroll
                    for (int n2 = 0; n2 < NT / 2; ++n2) {
                        uint32_t b[4];
                        ldsm_x4_trans(b, vt + (n2 >> 2) * 2048 + (v_lane_off ^ (((2 * n2) & 7) << 4)));
                        mma_bf16(o[2 * n2], pa, b[0], b[1]);
                        mma_bf16(o[2 * n2 + 1], pa, b[2], b[3]);
                    }
                }
            }
            __syncthreads();   // every warp is done with this stage
            ++cnt;
            if (threadIdx.x == 0 && next_issue < nst) {
                issue_stage(next_issue, cnt - 1 + kAppendStages);
                ++next_issue;
                load_ids(next_issue);
            }
        }

        // epilogue
        l_lo += __shfl_xor_sync(0xffffffffu, l_lo, 1);
        l_hi += __shfl_xor_sync(0xffffffffu, l_hi, 1);
        l_lo += __shfl_xor_sync(0xffffffffu, l_lo, 2);
        l_hi += __shfl_xor_sync(0xffffffffu, l_hi, 2);
        if (direct) {
            if (ok_lo) {
                const float inv = 1.f / l_lo;
                const size_t orow = (size_t)(q_start + r_lo / G) * p.Hq + (size_t)head * G + r_lo % G;
#pragma unroll
                for (int n = 0; n < NT; ++n)
                    *reinterpret_cast<uint32_t*>(p.out + orow * D + n * 8 + 2 * t4) = pack_bf16(o[n][0] * inv, o[n][1] * inv);
                if (t4 == 0) p.lse[orow] = (m_lo + log2f(l_lo)) * 0.6931471805599453f;
            }
            if (ok_hi) {
                const float inv = 1.f / l_hi;
                const size_t orow = (size_t)(q_start + r_hi / G) * p.Hq + (size_t)head * G + r_hi % G;
#pragma unroll
                for (int n = 0; n < NT; ++n)
                    *reinterpret_cast<uint32_t*>(p.out + orow * D + n * 8 + 2 * t4) = pack_bf16(o[n][2] * inv, o[n][3] * inv);
                if (t4 == 0) p.lse[orow] = (m_hi + log2f(l_hi)) * 0.6931471805599453f;
            }
        } else {
            const size_t prow = (size_t)partial * kAppendTileRows + warp * 16 + row;
#pragma unroll
            for (int n = 0; n < NT; ++n) {
                *reinterpret_cast<float2*>(p.po + prow * D + n * 8 + 2 * t4) = make_float2(o[n][0], o[n][1]);
                *reinterpret_cast<float2*>(p.po + (prow + 8) * D + n * 8 + 2 * t4) = make_float2(o[n][2], o[n][3]);
            }
            if (t4 == 0) {
                *reinterpret_cast<float2*>(p.pml + prow * 2) = make_float2(m_lo, l_lo);
                *reinterpret_cast<float2*>(p.pml + (prow + 8) * 2) = make_float2(m_hi, l_hi);
            }
        }
    }
}

// One warp per (merge group, tile row).
template <int D>
__global__ void __launch_bounds__(128) append_merge_kernel(const MergeGroup* groups, int n_groups, int TR, int G, int Hq,
                                                           const float* po, const float* pml, uint16_t* out,
                                                           float* lse) {
    constexpr int VEC = D / 32;
    const int w = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (w >= n_groups * TR) return;
    const MergeGroup g = groups[w / TR];
    const int tr = w % TR;
    const int r = g.row_begin + tr;
    if (r >= g.m * G) return;
    float M = -INFINITY;
    for (int k = 0; k < g.count; ++k) M = fmaxf(M, __ldg(pml + ((size_t)(g.first + k) * TR + tr) * 2));
    float L = 0.f, acc[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) acc[v] = 0.f;
    for (int k = 0; k < g.count; ++k) {
        const float2 ml = __ldg(reinterpret_cast<const float2*>(pml + ((size_t)(g.first + k) * TR + tr) * 2));
        if (ml.x == -INFINITY) continue;   // this partition held no visible key for the row
        const float wgt = fast_exp2(ml.x - M);
        L += ml.y * wgt;
        const float* src = po + ((size_t)(g.first + k) * TR + tr) * D + lane * VEC;
#pragma unroll
        for (int v = 0; v < VEC; ++v) acc[v] += __ldg(src + v) * wgt;
    }
    const float inv = 1.f / L;
    const size_t orow = (size_t)(g.q_start + r / G) * Hq + (size_t)g.head * G + r % G;
#pragma unroll
    for (int v = 0; v < VEC; v += 2)
        *reinterpret_cast<uint32_t*>(out + orow * D + lane * VEC + v) = pack_bf16(acc[v] * inv, acc[v + 1] * inv);
    if (lane == 0) lse[orow] = (M + log2f(L)) * 0.6931471805599453f;
}

template <int D>
int launch_append_t(const csv_plan* plan, const AppendParams& p, cudaStream_t stream) {
    constexpr int TB = 16 * D * 2;
    const size_t smem = (size_t)kAppendStages * kStageBlocks * 2 * TB + kAppendStages * 8;
    static PerDeviceOnce attr;
    CSV_CUDA_TRY(once_per_device(attr, [&] {
        return cudaFuncSetAttribute(append_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    }));
    const int cap = plan->num_sms * 2;
    const int grid = p.n_items < cap ? p.n_items : cap;
    append_kernel<D><<<grid, kAppendWarps * 32, smem, stream>>>(p);
    CSV_CUDA_TRY(cudaGetLastError());
    return CSV_OK;
}

template <int D>
int launch_append_merge(const csv_plan* plan, const AppendParams& p, cudaStream_t stream) {
    const int ng = (int)plan->append_groups.size();
    if (ng > 0) {
        const int warps = ng * plan->append_tile_rows;
        append_merge_kernel<D><<<(warps + 3) / 4, 128, 0, stream>>>(
            reinterpret_cast<const MergeGroup*>(plan->d_ws + plan->lay.append_groups), ng, plan->append_tile_rows, p.G,
            p.Hq, p.po, p.pml, p.out, p.lse);
        CSV_CUDA_TRY(cudaGetLastError());
    }
    return CSV_OK;
}

}   // namespace

int launch_append_merge_128(const csv_plan* plan, void* out, float* lse, void* stream) {
    AppendParams p = {};
    p.out = (uint16_t*)out;
    p.lse = lse;
    p.po = reinterpret_cast<float*>(plan->d_ws + plan->lay.append_po);
    p.pml = reinterpret_cast<float*>(plan->d_ws + plan->lay.append_pml);
    p.Hq = plan->shape.num_q_heads;
    p.Hkv = plan->shape.num_kv_heads;
    p.G = p.Hq / p.Hkv;
    return launch_append_merge<128>(plan, p, (cudaStream_t)stream);
}

int launch_append_attn(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                       int max_blocks, void* out, float* lse, void* stream) {
    if (plan->append_items.empty()) return CSV_OK;
    const kv_pool_desc& s = pool->desc;
    AppendParams p;
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
    if (s.head_dim == 128) {
        // d = 128: tcgen05 / TMEM kernel (append_attn_tc2.cu), two 128-row tiles per CTA
        const int rc = launch_append_attn_tc2(plan, pool, layer, q, tables, max_blocks, out, lse, stream);
        if (rc != CSV_OK) return rc;
        return launch_append_merge<128>(plan, p, (cudaStream_t)stream);
    }
    const int rc = launch_append_t<64>(plan, p, (cudaStream_t)stream);
    if (rc != CSV_OK) return rc;
    return launch_append_merge<64>(plan, p, (cudaStream_t)stream);
}
