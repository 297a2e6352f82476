// common.cuh - PTX helpers shared by the libmopal kernels (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libmopal is written for sm_100a (B200) only"
#endif

namespace mopal {

constexpr int TJ = 128;                 // j-bodies per shared-memory tile
constexpr int STAGES = 4;               // TMA ring depth
constexpr int CONSUMER_THREADS = 128;   // 4 compute warps, one per SM sub-partition
constexpr int CTA_THREADS = CONSUMER_THREADS + 32;  // + 1 TMA producer warp
constexpr int ACC_TILE_BYTES = TJ * 32 + 16;        // TJ x {x,y,z,gm} + 16 B gate header
constexpr int SYM_TILE_BYTES = TJ * 32 + 16 + TJ * 8; // two-sided kernel: the same + TJ x rcrit (5136)
constexpr int SYM_RC_OFF = TJ * 32 + 16;
constexpr int BOX_TILE_BYTES = TJ * 32;             // TJ x {lox,hix,loy,hiy}
constexpr int ON_BLOCK = 256;           // block size of the O(N) kernels

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}

// A kernel launch that is recorded in the step's graph but only WORKS when a device flag says so (the resolving step has
// two ways of getting its closing accelerations, chosen on the device from the last step's encounter list: mopal.cu)
struct Gate { const int* flag; int want; };
__device__ __forceinline__ bool gate_closed(const Gate& g) { return g.flag != nullptr && *g.flag != g.want; }

// ---- mbarrier ----------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t addr = smem_u32(bar), ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(addr), "r"(parity)
            : "memory");
    } while (!ok);
}

// ---- TMA 1-D bulk copy global -> shared, completion on an mbarrier -------
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes,
                                            uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(smem_dst)),
        "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// ---- 22-bit reciprocal square root seed: one MUFU.RSQ64H on the high word --
__device__ __forceinline__ double rsqrt_seed(double a) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    return y;
}

// fixed-order block reduction of three doubles (warp shuffle tree, then warps in order)
template <int BLOCK>
__device__ __forceinline__ void block_sum3(double& s0, double& s1, double& s2, double (*sh)[3]) {
    const unsigned full = 0xffffffffu;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s0 += __shfl_down_sync(full, s0, o);
        s1 += __shfl_down_sync(full, s1, o);
        s2 += __shfl_down_sync(full, s2, o);
    }
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { sh[w][0] = s0; sh[w][1] = s1; sh[w][2] = s2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t0 = 0, t1 = 0, t2 = 0;
#pragma unroll
        for (int k = 0; k < BLOCK / 32; ++k) { t0 += sh[k][0]; t1 += sh[k][1]; t2 += sh[k][2]; }
        sh[0][0] = t0; sh[0][1] = t1; sh[0][2] = t2;
    }
    __syncthreads();
    s0 = sh[0][0]; s1 = sh[0][1]; s2 = sh[0][2];
}

}  // namespace mopal
