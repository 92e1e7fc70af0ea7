// fx_stream.cuh -- per-thread asynchronous staging of streamed vectors (cp.async / LDGSTS into shared memory).
//
// The streaming kernels (exact dot, the fused CG vector update) do 25-30 dependent fp64 operations per element, so a
// thread that loads into registers and then computes keeps nothing in flight while it computes.  Here every thread
// copies ITS OWN elements of the next FX_STAGES-1 tiles into its own shared-memory slots with cp.async and reads them
// back when their group has completed: no barrier is needed (a thread only reads what it copied itself), no
// registers are held by data in flight, and ~200 KB per SM stay in flight ("bytes in flight").
// Out-of-range elements are zero-filled by the copy itself (src-size 0).

#ifndef FX_STREAM_CUH
#define FX_STREAM_CUH

#define FX_STAGES 4

// -DFX_CHECKED: bounds and ownership asserts in every staging routine (compute-sanitizer is closed on the pool the library is
// developed on).  A failing assert prints its location and traps; the parity suite is run against this build once per round.
#ifdef FX_CHECKED
#include <stdio.h>
#define FX_ASSERT(cond)                                                                                          \
    do {                                                                                                         \
        if (!(cond)) {                                                                                           \
            printf("FX_ASSERT failed: %s  (%s:%d, block %d thread %d)\n", #cond, __FILE__, __LINE__, (int)blockIdx.x, (int)threadIdx.x); \
            __trap();                                                                                            \
        }                                                                                                        \
    } while (0)
#else
#define FX_ASSERT(cond) do { } while (0)
#endif

__device__ __forceinline__ unsigned fx_smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void fx_cp_async8(unsigned dst, const void* src, bool valid) {
    const int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void fx_cp_async4(unsigned dst, const void* src, bool valid) {
    const int sz = valid ? 4 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void fx_cp_async16(unsigned dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void fx_cp_async16_full(unsigned dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void fx_lds128(double2& v, unsigned addr) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
}
__device__ __forceinline__ void fx_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void fx_cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- TMA (1-D bulk copy, cp.async.bulk) with mbarrier completion: one thread moves a whole tile -------------------------
__device__ __forceinline__ void fx_mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fx_mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fx_mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void fx_mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void fx_mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completion counted on `bar`
__device__ __forceinline__ void fx_tma_load_1d(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

#endif
