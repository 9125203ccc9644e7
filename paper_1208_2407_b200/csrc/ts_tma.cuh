// ts_tma.cuh -- PTX wrappers shared by the kernels that stream rows through shared memory:
// mbarrier, 1-D bulk async copies (TMA engine: SASS UBLKCP), vector shared-memory loads and
// elect.sync.  Device code only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ts {
namespace tma {

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t"
        "}" ::"r"(bar), "r"(parity)
        : "memory");
}
// global -> shared bulk copy; bytes % 16 == 0, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes,
                                         uint32_t bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

// global -> shared copy of one box of a 2-D tensor map (TMA, SASS UTMALDG): coordinates in
// elements (c0 = fastest dimension); elements of the box outside the tensor arrive as zeros and
// count towards the transaction bytes like any others
__device__ __forceinline__ void tensor2d_g2s(uint32_t dst, const void* tmap, int c0, int c1,
                                             uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}

__device__ __forceinline__ void lds4(uint32_t addr, float (&v)[4]) {
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]) : "r"(addr));
}
// fp64: a lane's four sites are 32 bytes, so two 16-byte loads at stride 32 over the lanes are
// 2-way bank conflicts (39 % of the shared-memory wavefronts of the C5 kernel, ncu r2).  A 128-bit
// load is served eight lanes at a time: lanes 0-3 of each eight read their first half first,
// lanes 4-7 their second half -- 128 distinct bytes per eight lanes in both loads -- and the
// halves are put back in order by selects.  addr is 32 * lane beyond a 128-byte aligned row.
#ifndef TS_F64_PLAIN_LDS
__device__ __forceinline__ void lds4(uint32_t addr, double (&v)[4]) {
    const bool sw = (addr & 128u) != 0;
    double a0, a1, b0, b1;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a0), "=d"(a1) : "r"(addr + (sw ? 16u : 0u)));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(b0), "=d"(b1) : "r"(addr + (sw ? 0u : 16u)));
    v[0] = sw ? b0 : a0; v[1] = sw ? b1 : a1;
    v[2] = sw ? a0 : b0; v[3] = sw ? a1 : b1;
}
#else
__device__ __forceinline__ void lds4(uint32_t addr, double (&v)[4]) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v[0]), "=d"(v[1]) : "r"(addr));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v[2]), "=d"(v[3]) : "r"(addr + 16));
}
#endif

// one lane per warp, known to the compiler as a single active lane (no per-lane issue loops)
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t"
        ".reg .pred P;\n\t"
        "elect.sync _|P, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, P;\n\t"
        "}" : "=r"(pred));
    return pred != 0;
}

}  // namespace tma
}  // namespace ts
