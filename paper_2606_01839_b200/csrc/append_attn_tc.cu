// append_attn_tc.cu — append_prefill_attn for head_dim 128 on the 5th-generation tensor cores
// (tcgen05.mma, accumulators in TMEM).  PAPER.md:94 §3.1 / PAPER.md:60 §2.2 (see append_attn.cu).
//
// Roofline: tensor (bf16, fp32 accumulate) once m*G >~ 213 stacked rows; flops = 4*d*Hq*m*(P+(m+1)/2).
//
// One CTA = one tile of 128 stacked rows (token-major: row = token*G + head) of one KV head against a
// range of KV blocks, 2 CTAs per SM.  Six warps:
//   warps 0-3  softmax: thread r owns row r = TMEM lane r, so row max / sum need no shuffles.  Reads S
//              (128 x 64 fp32) with tcgen05.ld, writes P (bf16) back into the same TMEM columns with
//              tcgen05.st, rescales O lazily (only when a row max grows by more than 2^8), epilogue.
//   warp 4     producer: 1-D bulk copies (UBLKCP) of K half-tiles and V tiles into 2-stage rings.
//   warp 5     MMA issuer: S_j = Q K_j^T (A = Q in smem, B = the K tiles exactly as they sit in the pool:
//              the pool's 128-byte-swizzled tile image IS the UMMA SWIZZLE_128B K-major layout), then
//              O += P_j V_j with A = P from TMEM and B = the V tiles as an MN-major SWIZZLE_128B operand.
//              S is double-buffered in TMEM so S_{j+1} runs under softmax j.
// TMEM columns: [0,64) S/P buffer 0, [64,128) S/P buffer 1, [128,256) O.
#include <math.h>

#include "common.cuh"
#include "internal.h"
#include "tc5.cuh"

namespace {

constexpr int kTcThreads = 192;
constexpr int kTcRows = 128;      // stacked rows per item (UMMA M)
constexpr int kChunk = 64;        // KV tokens per pipeline step (UMMA N of the score MMA)
constexpr int kChunkBlocks = kChunk / 16;
constexpr uint32_t kTmemCols = 256;

struct AppendTcParams {
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

// shared memory map (offsets from a 1024-byte aligned base)
constexpr uint32_t kOffQ = 0;                       // [2 halves][128 rows][128 B]
constexpr uint32_t kOffK = 32768;                   // 2 stages x [2 halves][4 blocks][2048 B]
constexpr uint32_t kOffV = kOffK + 2 * 16384;       // 2 stages x [4 blocks][4096 B]
constexpr uint32_t kOffBar = kOffV + 2 * 16384;     // 13 mbarriers + TMEM slot
constexpr uint32_t kSmemBytes = kOffBar + 128 + 1024;

__global__ void __launch_bounds__(kTcThreads, 2) append_tc_kernel(const __grid_constant__ AppendTcParams p) {
    constexpr int D = 128;
    constexpr int TB = 4096;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kOffBar);
    uint64_t *k_full = bars, *k_empty = bars + 2, *v_full = bars + 4, *v_empty = bars + 6, *s_full = bars + 8,
             *p_full = bars + 10, *o_done = bars + 12;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 13);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int i = 0; i < 2; ++i) {
            mbar_init(&k_full[i], 1);
            mbar_init(&k_empty[i], 1);
            mbar_init(&v_full[i], 1);
            mbar_init(&v_empty[i], 1);
            mbar_init(&s_full[i], 1);
            mbar_init(&p_full[i], 128);
        }
        mbar_init(o_done, 1);
        fence_mbar_init();
    }
    if (warp == 5) tmem_alloc(tmem_slot, kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t tmem_O = tmem + 128;

    const int G = p.G;
    const size_t kv_stride = (size_t)p.Hkv * TB;
    const size_t blk_stride = 2 * kv_stride;
    uint32_t kc = 0;   // chunks this CTA has pushed through the pipeline so far (same in every role)

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
        const int nch = (nblk + kChunkBlocks - 1) / kChunkBlocks;

        // ---- stage this tile's Q rows into shared memory in the K-major SWIZZLE_128B image ----------
        if (warp < 4) {
            const int r = threadIdx.x, sr = row_begin + r;
            const bool ok = sr < rows_total;
            const uint4* src = reinterpret_cast<const uint4*>(
                p.q + ((size_t)(q_start + (ok ? sr / G : 0)) * p.Hq + (size_t)head * G + (ok ? sr % G : 0)) * D);
            uint4 v[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) v[c] = ok ? __ldg(src + c) : make_uint4(0, 0, 0, 0);
#pragma unroll
            for (int c = 0; c < 16; ++c)
                *reinterpret_cast<uint4*>(smem + kOffQ + (c >> 3) * 16384 + r * 128 + (((c & 7) ^ (r & 7)) << 4)) = v[c];
            fence_proxy_async();   // generic writes -> visible to the tensor core's async-proxy reads
        }
        tc_fence_before();
        __syncthreads();   // Q staged; previous item's epilogue has finished reading O
        tc_fence_after();

        if (warp == 4) {
            // ================= producer =================
            if (lane == 0) {
                const int32_t* tab = p.tables + (size_t)conv * p.max_blocks + blk_begin;
                const uint8_t* head_base = p.pool_layer + (size_t)head * TB;
                int ids[kChunkBlocks], nids[kChunkBlocks];
#pragma unroll
                for (int jb = 0; jb < kChunkBlocks; ++jb) nids[jb] = jb < nblk ? __ldg(tab + jb) : 0;
                for (int j = 0; j < nch; ++j) {
                    const uint32_t c = kc + j, b = c & 1, ph = (c >> 1) & 1;
                    const int nb = min(kChunkBlocks, nblk - j * kChunkBlocks);
#pragma unroll
                    for (int jb = 0; jb < kChunkBlocks; ++jb) {
                        ids[jb] = nids[jb];
                        const int nx = (j + 1) * kChunkBlocks + jb;
                        nids[jb] = nx < nblk ? __ldg(tab + nx) : 0;
                    }
                    uint8_t* kb = smem + kOffK + b * 16384;
                    uint8_t* vb = smem + kOffV + b * 16384;
                    mbar_wait(&k_empty[b], ph ^ 1);
                    mbar_expect_tx(&k_full[b], (uint32_t)nb * TB);
#pragma unroll
                    for (int jb = 0; jb < kChunkBlocks; ++jb)
                        if (jb < nb) {
                            const uint8_t* src = head_base + (size_t)ids[jb] * blk_stride;
                            bulk_g2s(kb + jb * 2048, src, 2048, &k_full[b]);
                            bulk_g2s(kb + 8192 + jb * 2048, src + 2048, 2048, &k_full[b]);
                        }
                    mbar_wait(&v_empty[b], ph ^ 1);
                    mbar_expect_tx(&v_full[b], (uint32_t)nb * TB);
#pragma unroll
                    for (int jb = 0; jb < kChunkBlocks; ++jb)
                        if (jb < nb)
                            bulk_g2s(vb + jb * TB, head_base + (size_t)ids[jb] * blk_stride + kv_stride, TB, &v_full[b]);
                }
            }
        } else if (warp == 5) {
            // ================= MMA issuer =================
            constexpr uint32_t idS = idesc_bf16(kTcRows, kChunk, 0, 0);
            constexpr uint32_t idO = idesc_bf16(kTcRows, D, 0, 1);
            auto issue_S = [&](int j) {
                const uint32_t c = kc + j, b = c & 1, ph = (c >> 1) & 1;
                mbar_wait(&k_full[b], ph);
                tc_fence_after();
                if (lane == 0) {
#pragma unroll
                    for (int hk = 0; hk < 8; ++hk) {   // hk = half * 4 + k-step inside the 64-element half
                        const uint32_t off = (hk >> 2) * 16384 + (hk & 3) * 32;
                        const uint32_t offk = (hk >> 2) * 8192 + (hk & 3) * 32;
                        mma_ss(tmem + b * 64, smem_desc_sw128(sbase + kOffQ + off, 16, 1024),
                               smem_desc_sw128(sbase + kOffK + b * 16384 + offk, 16, 1024), idS, hk != 0);
                    }
                    tc_commit(&k_empty[b]);
                    tc_commit(&s_full[b]);
                }
                __syncwarp();
            };
            issue_S(0);
            for (int j = 0; j < nch; ++j) {
                if (j + 1 < nch) issue_S(j + 1);
                const uint32_t c = kc + j, b = c & 1, ph = (c >> 1) & 1;
                const int nb = min(kChunkBlocks, nblk - j * kChunkBlocks);
                mbar_wait(&p_full[b], ph);
                mbar_wait(&v_full[b], ph);
                const int tok0 = (blk_begin + j * kChunkBlocks) * 16;
                if (tok0 + nb * 16 > kv_len) {   // slots past kv_len may hold NaN patterns: 0 * NaN must not reach O
                    const int nvalid = kv_len - (tok0 + (nb - 1) * 16);
                    uint8_t* vt = smem + kOffV + b * 16384 + (nb - 1) * TB;
                    for (int cidx = lane; cidx < TB / 16; cidx += 32)
                        if (((cidx & 127) >> 3) >= nvalid) *reinterpret_cast<uint4*>(vt + cidx * 16) = make_uint4(0, 0, 0, 0);
                    fence_proxy_async();
                    __syncwarp();
                }
                tc_fence_after();
                if (lane == 0) {
                    for (int kk = 0; kk < nb; ++kk)
                        mma_ts(tmem_O, tmem + b * 64 + kk * 8,
                               smem_desc_sw128(sbase + kOffV + b * 16384 + kk * TB, 2048, 1024), idO, (j | kk) != 0);
                    tc_commit(&v_empty[b]);
                    tc_commit(o_done);
                }
                __syncwarp();
            }
        } else {
            // ================= softmax (thread r owns stacked row r = TMEM lane r) =================
            const int r = threadIdx.x, sr = row_begin + r;
            const bool ok = sr < rows_total;
            const int lim = ok ? P + sr / G : kv_len - 1;   // last visible key; rows past the chunk see all (Q = 0)
            const uint32_t lane_base = tmem + ((uint32_t)(warp * 32) << 16);
            float m_used = -INFINITY, l_run = 0.f;
            for (int j = 0; j < nch; ++j) {
                const uint32_t c = kc + j, b = c & 1, ph = (c >> 1) & 1;
                mbar_wait(&s_full[b], ph);
                tc_fence_after();
                uint32_t s0[32], s1[32];
                tmem_ld32(lane_base + b * 64, s0);
                tmem_ld32(lane_base + b * 64 + 32, s1);
                tmem_wait_ld();
                const int tok0 = (blk_begin + j * kChunkBlocks) * 16;
                const int nb = min(kChunkBlocks, nblk - j * kChunkBlocks);
                // visible columns of this chunk for this row (<= 0: none).  Columns past the blocks actually loaded
                // hold stale shared memory and are masked too (a KV partition may end before the row's limit).
                const int nvis = min(lim - tok0 + 1, nb * 16);
                // raw scores stay unscaled: max on the raw values (scale > 0), and the scale folds into the
                // exponent's FFMA below: p = exp2(s * scale - ref)
                float x[64];
#pragma unroll
                for (int k = 0; k < 32; ++k) {
                    x[k] = __uint_as_float(s0[k]);
                    x[32 + k] = __uint_as_float(s1[k]);
                }
                if (nvis < kChunk) {
#pragma unroll
                    for (int k = 0; k < 64; ++k)
                        if (k >= nvis) x[k] = -INFINITY;
                }
                float mraw = x[0];
#pragma unroll
                for (int k = 1; k < 63; k += 2) mraw = fmax3(mraw, x[k], x[k + 1]);
                mraw = fmaxf(mraw, x[63]);
                const float mx = mraw * p.scale_log2;   // -inf stays -inf
                if (j == 0) {
                    m_used = mx;   // PV_0 overwrites O (accumulate = 0): nothing to rescale yet
                } else {
                    mbar_wait(o_done, (c - 1) & 1);   // PV_{j-1} has finished: O is stable, P buffer history is consumed
                    tc_fence_after();
                    const bool need = mx > m_used + 8.f;   // lazy rescale: exponents stay below 2^8 otherwise
                    if (__any_sync(0xffffffffu, need)) {
                        const float alpha = need ? fast_exp2(m_used - mx) : 1.f;   // exp2(-inf) = 0 for a row with no key yet
                        if (need) m_used = mx;
                        l_run *= alpha;
#pragma unroll
                        for (int piece = 0; piece < 4; ++piece) {
                            uint32_t o[32];
                            tmem_ld32(lane_base + 128 + piece * 32, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int k = 0; k < 32; ++k) o[k] = __float_as_uint(__uint_as_float(o[k]) * alpha);
                            tmem_st32(lane_base + 128 + piece * 32, o);
                        }
                        tmem_wait_st();
                    }
                }
                const float ref = m_used == -INFINITY ? 0.f : m_used;
                uint32_t pk[32];
                const float2 sc2 = make_float2(p.scale_log2, p.scale_log2), nref2 = make_float2(-ref, -ref);
                float2 acc2 = make_float2(0.f, 0.f);
#pragma unroll
                for (int k = 0; k < 32; ++k) {
                    const float2 t = ffma2(make_float2(x[2 * k], x[2 * k + 1]), sc2, nref2);
                    const float p0 = fast_exp2(t.x), p1 = fast_exp2(t.y);
                    acc2 = fadd2(acc2, make_float2(p0, p1));
                    pk[k] = pack_bf16(p0, p1);
                }
                const float lsum = acc2.x + acc2.y;
                l_run += lsum;
                tmem_st32(lane_base + b * 64, pk);   // P_j over the first 32 columns of S_j (this lane's row only)
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(&p_full[b]);
            }
            // ---- epilogue: wait for the last PV, normalise, write ----
            mbar_wait(o_done, (kc + nch - 1) & 1);
            tc_fence_after();
            const float inv = direct ? 1.f / l_run : 1.f;
            const size_t orow = (size_t)(q_start + (ok ? sr / G : 0)) * p.Hq + (size_t)head * G + (ok ? sr % G : 0);
            const size_t prow = (size_t)partial * kTcRows + r;
#pragma unroll
            for (int piece = 0; piece < 4; ++piece) {
                uint32_t o[32];
                tmem_ld32(lane_base + 128 + piece * 32, o);
                tmem_wait_ld();
                if (direct) {
                    if (ok) {
                        uint4* dst = reinterpret_cast<uint4*>(p.out + orow * D + piece * 32);
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4) {
                            uint4 w;
                            w.x = pack_bf16(__uint_as_float(o[8 * q4 + 0]) * inv, __uint_as_float(o[8 * q4 + 1]) * inv);
                            w.y = pack_bf16(__uint_as_float(o[8 * q4 + 2]) * inv, __uint_as_float(o[8 * q4 + 3]) * inv);
                            w.z = pack_bf16(__uint_as_float(o[8 * q4 + 4]) * inv, __uint_as_float(o[8 * q4 + 5]) * inv);
                            w.w = pack_bf16(__uint_as_float(o[8 * q4 + 6]) * inv, __uint_as_float(o[8 * q4 + 7]) * inv);
                            dst[q4] = w;
                        }
                    }
                } else {
                    uint4* dst = reinterpret_cast<uint4*>(p.po + prow * D + piece * 32);
#pragma unroll
                    for (int q4 = 0; q4 < 8; ++q4) dst[q4] = make_uint4(o[4 * q4], o[4 * q4 + 1], o[4 * q4 + 2], o[4 * q4 + 3]);
                }
            }
            if (direct) {
                if (ok) p.lse[orow] = (m_used + log2f(l_run)) * 0.6931471805599453f;
            } else {
                *reinterpret_cast<float2*>(p.pml + prow * 2) = make_float2(m_used, l_run);
            }
        }
        kc += nch;
        tc_fence_before();   // order this item's TMEM traffic before the next item's barrier
    }
    __syncthreads();
    if (warp == 5) tmem_dealloc(tmem, kTmemCols);
}

}   // namespace

int launch_append_attn_tc(const csv_plan* plan, const kv_pool* pool, int layer, const void* q, const int32_t* tables,
                          int max_blocks, void* out, float* lse, void* stream) {
    const kv_pool_desc& s = pool->desc;
    AppendTcParams p;
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
    static bool attr_set = false;
    if (!attr_set) {
        CSV_CUDA_TRY(cudaFuncSetAttribute(append_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
        attr_set = true;
    }
    const int cap = plan->num_sms * 2;
    const int grid = p.n_items < cap ? p.n_items : cap;
    append_tc_kernel<<<grid, kTcThreads, kSmemBytes, (cudaStream_t)stream>>>(p);
    CSV_CUDA_TRY(cudaGetLastError());
    return CSV_OK;
}
