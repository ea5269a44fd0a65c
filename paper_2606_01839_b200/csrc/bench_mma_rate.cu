// bench_mma_rate.cu — microbenchmark behind the tile-shape choices of append_attn_tc2.cu:
// cycles per tcgen05.mma (kind::f16, bf16 operands, fp32 accumulate, cta_group::1) by shape and operand source,
// one CTA per SM on all SMs, operands resident in shared memory / TMEM, issued back to back by one or two warps.
// Not part of libconserve_kv.so.  Build and run:
//   python -m paper_2606_01839_b200.build --microbench && paper_2606_01839_b200/bench_mma_rate
// Columns: cycles per unit measured by the issuing thread until its last instruction issued ("issue") and until
// tcgen05.commit reports completion ("total").  A unit is one MMA, or one mix (see the mode names).
#include <cstdio>
#include <cuda_runtime.h>

#include "tc5.cuh"

namespace {

struct Res {
    long long issue, total;
};

enum Mode {
    kSS64,        // M128 N64  K16, A and B from shared memory
    kSS128,       // M128 N128 K16
    kSS256,       // M128 N256 K16
    kTS128,       // M128 N128 K16, A from TMEM
    kRebuild64,   // N64 SS with the 64-bit descriptors rebuilt and a lane elected per MMA, one A half only
    kMix64x2,     // the 64-key step of append_tc2: 8 x SS N64 + 4 x TS N128, from each of two warps (two row tiles)
    kMix128x2,    // the 128-key step of the FlashAttention-4 tiling: 8 x SS N128 + 8 x TS N128, from each of two warps
    kModes
};
const char* kNames[kModes] = {"SS M128 N64 K16", "SS M128 N128 K16", "SS M128 N256 K16", "TS M128 N128 K16",
                              "SS N64, descriptor rebuilt per MMA", "mix 8 x SS N64 + 4 x TS N128, two warps",
                              "mix 8 x SS N128 + 8 x TS N128, two warps"};

__device__ __forceinline__ void mma_ss_elect_rebuild(uint32_t d, uint32_t a_addr, uint32_t b_addr, uint32_t idesc, uint32_t acc) {
    const uint64_t ad = smem_desc_sw128(a_addr, 0, 1024), bd = smem_desc_sw128(b_addr, 0, 1024);
    asm volatile(
        "{\n\t.reg .pred pe, pa;\n\telect.sync _|pe, 0xffffffff;\n\tsetp.ne.b32 pa, %4, 0;\n\t"
        "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, pa;\n\t}"
        ::"r"(d), "l"(ad), "l"(bd), "r"(idesc), "r"(acc)
        : "memory");
}

__global__ void __launch_bounds__(64, 1) mma_rate_kernel(int mode, int iters, Res* out) {
    extern __shared__ __align__(1024) uint8_t smem[];   // [0,64K) A tiles of the two warps, [64K,192K) B tiles
    __shared__ uint32_t tslot;
    __shared__ uint64_t bar[2];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < 192 * 1024 / 4; i += blockDim.x)
        reinterpret_cast<uint32_t*>(smem)[i] = 0x3f803f80u ^ ((uint32_t)i * 2654435761u & 0x007f007fu);   // bf16 values near 1
    if (warp == 0) tmem_alloc(&tslot, 512);
    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        fence_mbar_init();
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tslot, sbase = smem_u32(smem);
    const bool two = mode == kMix64x2 || mode == kMix128x2;
    if (warp == 0 || two) {
        const uint32_t d = tmem + warp * 256;
        const uint64_t ad = smem_desc_sw128(sbase + warp * 32768, 0, 1024), bd = smem_desc_sw128(sbase + 65536, 0, 1024);
        const uint64_t vd = smem_desc_sw128(sbase + 65536, 2048, 1024);
        const uint32_t alo = (uint32_t)ad, hi = (uint32_t)(ad >> 32), blo = (uint32_t)bd, vlo = (uint32_t)vd, vhi = (uint32_t)(vd >> 32);
        const int N = mode == kSS64 || mode == kRebuild64 ? 64 : mode == kSS256 ? 256 : 128;
        const uint32_t idS = idesc_bf16(128, mode == kMix64x2 ? 64 : N, 0, 0), idO = idesc_bf16(128, 128, 0, 1);
        long long t0 = clock64(), t1 = t0;
        if (mode == kRebuild64) {
            for (int i = 0; i < iters; ++i)
                mma_ss_elect_rebuild(d, sbase + (i & 3) * 32, sbase + 65536 + ((i >> 2) & 3) * 16384 + (i & 3) * 32, idS, i > 0);
            t1 = clock64();
            if (lane == 0) tc_commit(&bar[warp]);
        } else if (lane == 0) {
            for (int i = 0; i < iters; ++i) {
                const uint32_t st = (uint32_t)(i & 3) * 1024;   // rotate over four 16 KiB B stages
                if (mode == kTS128) {
#pragma unroll
                    for (int u = 0; u < 8; ++u) mma_ts_lohi(d + 128, d + u * 8, vlo + st + u * 256, vhi, idO, (i | u) != 0);
                } else if (two) {
                    const bool wide = mode == kMix128x2;
                    const uint32_t dS = wide ? d : d + (i & 1) * 64;
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        mma_ss_lohi(dS, alo + (u & 3) * 2 + (u >> 2) * 1024, hi, blo + st + (u & 3) * 2 + (u >> 2) * (wide ? 1024 : 512),
                                    hi, idS, u != 0);
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (wide || u < 4) mma_ts_lohi(d + 128, dS + u * 8, vlo + (wide ? (st & 1024) * 2 : st) + u * 256, vhi, idO, (i | u) != 0);
                } else {
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        mma_ss_lohi(d, alo + (u & 3) * 2 + (u >> 2) * 1024, hi, blo + (u & 3) * 2 + (u >> 2) * 512, hi, idS, (i | u) != 0);
                }
            }
            t1 = clock64();
            tc_commit(&bar[warp]);
        }
        __syncwarp();
        mbar_wait(&bar[warp], 0);
        const long long t2 = clock64();
        if (lane == 0 && blockIdx.x == 0 && warp == 0) {
            out->issue = t1 - t0;
            out->total = t2 - t0;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 512);
}

}   // namespace

int main() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        fprintf(stderr, "no CUDA device\n");
        return 1;
    }
    Res* d = nullptr;
    cudaMalloc(&d, sizeof(Res));
    const int smem = 192 * 1024;
    cudaFuncSetAttribute(mma_rate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    printf("tcgen05.mma rate, %d SMs, one CTA per SM (cycles of the issuing thread)\n", sms);
    for (int mode = 0; mode < kModes; ++mode) {
        const bool single = mode == kRebuild64;                        // one MMA per iteration
        const bool mix = mode == kMix64x2 || mode == kMix128x2;
        const int iters = single ? 512 : 64;
        Res h = {};
        cudaMemset(d, 0, sizeof(Res));
        mma_rate_kernel<<<sms, 64, smem>>>(mode, iters, d);
        const cudaError_t e = cudaDeviceSynchronize();
        cudaMemcpy(&h, d, sizeof(h), cudaMemcpyDeviceToHost);
        const double units = mix ? iters : single ? iters : iters * 8.0;
        printf("%-44s %8.1f issue  %8.1f total  cycles per %s%s%s\n", kNames[mode], h.issue / units, h.total / units,
               mix ? "mix" : "MMA", e == cudaSuccess ? "" : "  ERROR: ", e == cudaSuccess ? "" : cudaGetErrorString(e));
        if (e != cudaSuccess) return 1;
    }
    cudaFree(d);
    return 0;
}
