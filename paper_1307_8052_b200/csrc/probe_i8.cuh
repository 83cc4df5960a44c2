// tcgen05 int8 issue-rate probe with a self-check (the denominator of the planned int8-sliced rank-K).
// One CTA per SM: TMEM allocation, two operand tiles in shared memory in the canonical K-major no-swizzle layout
// (8-row x 16-byte core matrices; the two 16-byte K chunks of an MMA I8_LBO apart, 8-row groups I8_SBO apart), one
// tcgen05.mma.kind::i8 of 128 x 256 x 32 read back with tcgen05.ld and written out for the host to check, then `iters`
// accumulating MMAs issued by one thread and committed to an mbarrier.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

constexpr int I8_M = 128, I8_N = 256, I8_K = 32;
constexpr uint32_t I8_LBO = 128, I8_SBO = 256;
// instruction descriptor: D = s32 (bits 4-5 = 2), A and B signed 8-bit (bits 7-9, 10-12 = 1), both K-major, N/8 at bit 17,
// M/16 at bit 24
constexpr uint32_t I8_IDESC = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(I8_N >> 3) << 17) | ((uint32_t)(I8_M >> 4) << 24);

__device__ __forceinline__ uint32_t i8_saddr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared-memory matrix descriptor: address, leading (K) and stride (M/N) byte offsets in 16-byte units, version 1, no swizzle
__device__ __forceinline__ uint64_t i8_smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((saddr & 0x3FFFF) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void i8_mma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t accumulate) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(I8_IDESC), "r"(accumulate));
}
__device__ __forceinline__ void i8_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(i8_saddr(bar)) : "memory");
}
__device__ __forceinline__ void i8_bar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nI8W: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra I8D;\nbra I8W;\nI8D:\n}"
                 ::"r"(i8_saddr(bar)), "r"(parity) : "memory");
}

// A[128][32], B[256][32] int8 row-major (K contiguous); D[128][256] = A B^T written by CTA 0.  block 128.
__global__ void __launch_bounds__(128) i8_probe_kernel(const int8_t *__restrict__ A, const int8_t *__restrict__ B,
                                                      int32_t *__restrict__ D, int iters) {
    __shared__ __align__(128) int8_t sA[I8_M * I8_K];
    __shared__ __align__(128) int8_t sB[I8_N * I8_K];
    __shared__ __align__(8) uint64_t bar;
    __shared__ uint32_t tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < I8_M * I8_K; i += 128) {
        const int r = i / I8_K, k = i % I8_K;
        sA[(r % 8) * 16 + (r / 8) * I8_SBO + (k % 16) + (k / 16) * I8_LBO] = A[i];
    }
    for (int i = tid; i < I8_N * I8_K; i += 128) {
        const int r = i / I8_K, k = i % I8_K;
        sB[(r % 8) * 16 + (r / 8) * I8_SBO + (k % 16) + (k / 16) * I8_LBO] = B[i];
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(i8_saddr(&bar)));
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {   // 256 TMEM columns: one 128 x 256 s32 accumulator
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(i8_saddr(&tmem_base)), "r"(256));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the generic-proxy stores above -> the tensor core's reads
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t taddr = tmem_base;
    const uint64_t da = i8_smem_desc(i8_saddr(sA), I8_LBO, I8_SBO), db = i8_smem_desc(i8_saddr(sB), I8_LBO, I8_SBO);
    if (tid == 0) {
        i8_mma(taddr, da, db, 0);
        i8_commit(&bar);
    }
    i8_bar_wait(&bar, 0);
    asm volatile("tcgen05.fence::after_thread_sync;");
    if (blockIdx.x == 0) {   // D row = TMEM lane = thread, 8 columns per load
        for (int c0 = 0; c0 < I8_N; c0 += 8) {
            uint32_t r[8];
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                         : "r"(taddr + ((uint32_t)(warp * 32) << 16) + c0));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            for (int j = 0; j < 8; j++) D[(size_t)tid * I8_N + c0 + j] = (int32_t)r[j];
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    if (tid == 0) {
        for (int it = 0; it < iters; it++) i8_mma(taddr, da, db, 1);
        i8_commit(&bar);
    }
    i8_bar_wait(&bar, 1);
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(256));
}
