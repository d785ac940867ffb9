// umma.cuh -- thin inline-PTX wrappers for the 5th-generation tensor cores (tcgen05): shared-memory
// matrix descriptors (no swizzle), mbarriers, MMA issue/commit and TMEM loads.  Shared by the
// gridding kernel (k_grid_mma.cu) and the DFT-as-GEMM transforms (tcfft.cuh).
//
// No-swizzle operand layout (validated against a host matmul before use): blocks of 8 x 8 halves
// (128 contiguous bytes).  K-major operand: block = 8 mn-rows x 8 k (k contiguous);  MN-major operand:
// block = 8 k-rows x 8 mn (mn contiguous).  In both, the descriptor's leading byte offset is the
// distance between blocks adjacent in K and the stride byte offset between blocks adjacent in M/N.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

namespace tcpk {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// shared-memory matrix descriptor, no swizzle: start >> 4, leading (k-block) and stride (mn-block) byte offsets >> 4
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) |
           ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity, int tag = 0, int info = 0) {
    uint32_t done = 0;
#ifdef TCP_MBAR_WATCHDOG
    unsigned spins = 0;
#endif
    while (!done) {
        asm volatile("{.reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p;}"
                     : "=r"(done)
                     : "r"(smem_u32(b)), "r"(parity)
                     : "memory");
#ifdef TCP_MBAR_WATCHDOG
        if (!done && ++spins > (1u << 22)) {
            if ((threadIdx.x & 31) == 0)
                printf("mbar stuck: block %d,%d warp %d tag %d parity %u info %d\n", blockIdx.x, blockIdx.y, threadIdx.x >> 5, tag, parity, info);
            __trap();
        }
#endif
    }
}
__device__ __forceinline__ void umma_commit(uint64_t* b) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{.reg .pred p; setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;}" ::"r"(tmem_d),
                 "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
                 : "memory");
}

template <int NN> struct TmemLd;
template <> struct TmemLd<16> {
    static __device__ __forceinline__ void run(uint32_t taddr, uint32_t* r) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                       "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                     : "r"(taddr));
    }
};
template <> struct TmemLd<32> {
    static __device__ __forceinline__ void run(uint32_t taddr, uint32_t* r) {
        TmemLd<16>::run(taddr, r);
        TmemLd<16>::run(taddr + 16, r + 16);
    }
};

// ---- bulk asynchronous copies (TMA, 1D): global -> shared completes on an mbarrier, shared -> global in bulk groups
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* b) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(b))
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
// generic-proxy accesses to shared memory before / after asynchronous-proxy accesses to the same bytes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}

}  // namespace tcpk
