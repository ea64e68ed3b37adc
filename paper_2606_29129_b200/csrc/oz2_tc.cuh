// oz2_tc.cuh -- sm_100a plumbing shared by the tensor-core kernels (oz2_gemm.cu, oz2_crt.cu): mbarrier, TMA,
// tcgen05 fences / commit / kind::i8 MMA, and the driver entry point for tensor-map encoding.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>
#include <atomic>
#include <mutex>

namespace {

// A stuck mbarrier must not hang the GPU box, and a legitimately long stall (debugger, MPS time slicing, deep clock
// throttling) must not kill the context: the waits below spin freely for SPIN_FAST polls, then back off with
// __nanosleep and give up (trap) only after STALL_NS of wall time by %globaltimer.  -DOZ2_TRAP_ON_STALL=0 removes
// the trap altogether.
#ifndef OZ2_TRAP_ON_STALL
#define OZ2_TRAP_ON_STALL 1
#endif
constexpr uint32_t SPIN_FAST = 1u << 14;
constexpr unsigned long long STALL_NS = 20ull * 1000ull * 1000ull * 1000ull;     // 20 s
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// slow side of every wait: called once the fast spin budget is used up
__device__ __noinline__ void mbar_wait_slow(uint32_t addr, uint32_t parity)
{
    const unsigned long long t0 = globaltimer_ns();
    uint32_t done = 0;
    while (true) {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(addr), "r"(parity)
                     : "memory");
        if (done) return;
        __nanosleep(1000);
#if OZ2_TRAP_ON_STALL
        if (globaltimer_ns() - t0 > STALL_NS) __trap();
#endif
    }
}

// SM count of the CURRENT device, cached per device (first calls that race store the same value)
inline int oz2_num_sms()
{
    static std::atomic<int> cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 1;
    if (dev < 0 || dev >= 64) {
        int v = 1;
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
        return v;
    }
    int v = cache[dev].load(std::memory_order_relaxed);
    if (!v) {
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v < 1) return 1;
        cache[dev].store(v, std::memory_order_relaxed);
    }
    return v;
}

// tensor memory -> registers: 32 lanes x 32 consecutive columns of 32-bit accumulators, 32 registers per thread.
// tc_ld32_nowait leaves the load in flight (the caller issues tcgen05.wait::ld before it reads v); tc_ld32 waits.
__device__ __forceinline__ void tc_ld32_nowait(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    tc_ld32_nowait(taddr, v);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done = 0, spins = 0;
    const uint32_t addr = smem_u32(bar);
    while (true) {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(addr), "r"(parity)
                     : "memory");
        if (done) break;
        if (++spins > SPIN_FAST) { mbar_wait_slow(addr, parity); break; }
    }
}
__device__ __forceinline__ void tma_load_3d(const CUtensorMap *map, uint64_t *bar, void *dst, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_mma_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "setp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
                 : "memory");
}


// the same primitives on 32-bit shared-space addresses (keeps address conversions out of persistent loops)
__device__ __forceinline__ void mbar_wait_a(uint32_t addr, uint32_t parity)
{
    uint32_t done = 0, spins = 0;
    while (true) {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(addr), "r"(parity)
                     : "memory");
        if (done) break;
        if (++spins > SPIN_FAST) { mbar_wait_slow(addr, parity); break; }
    }
}
// wait of a warp that is expected to idle for a long time (an epilogue warp waiting for the next accumulator):
// sleep between polls so that the idle warps do not burn issue slots (and power) next to the MMA warp
__device__ __forceinline__ void mbar_wait_idle(uint32_t addr, uint32_t parity)
{
    uint32_t done = 0, spins = 0;
    while (true) {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(addr), "r"(parity)
                     : "memory");
        if (done) break;
        __nanosleep(200);
        if (++spins > SPIN_FAST) { mbar_wait_slow(addr, parity); break; }
    }
}
__device__ __forceinline__ void mbar_arrive_a(uint32_t addr)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx_a(uint32_t addr, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(addr), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_3d_a(const CUtensorMap *map, uint32_t bar, uint32_t dst, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void tc_commit_a(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn get_encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// Encoded tensor maps are pure functions of (base, dims, strides, box, swizzle): a small cache keeps the host from
// re-encoding the same three maps on every ozaki2_dgemm call (cuTensorMapEncodeTiled costs a few microseconds,
// which shows at small sizes).  Uniform key: 3-D UINT8 maps only, which is all this library uses.
struct TensorMapKey {
    const void *base;
    uint64_t d0, d1, d2, s1, s2;
    uint32_t b0, b1, b2, swizzle;
};
inline int encode_u8_3d_cached(CUtensorMap *out, const TensorMapKey &key)
{
    constexpr int SLOTS = 16;
    static TensorMapKey keys[SLOTS];
    static CUtensorMap maps[SLOTS];
    static int used = 0, next = 0;
    static std::mutex mu;
    std::lock_guard<std::mutex> lk(mu);
    for (int t = 0; t < used; t++)
        if (memcmp(&keys[t], &key, sizeof(key)) == 0) { *out = maps[t]; return 0; }
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return (int)cudaErrorNotSupported;
    cuuint64_t dims[3] = { key.d0, key.d1, key.d2 };
    cuuint64_t strides[2] = { key.s1, key.s2 };
    cuuint32_t box[3] = { key.b0, key.b1, key.b2 };
    cuuint32_t estr[3] = { 1u, 1u, 1u };
    CUtensorMap m;
    CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void *>(key.base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, (CUtensorMapSwizzle)key.swizzle, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return (int)cudaErrorInvalidValue;
    const int slot = used < SLOTS ? used++ : (next = (next + 1) % SLOTS);
    keys[slot] = key;
    maps[slot] = m;
    *out = m;
    return 0;
}

} // namespace
