// ddsp_dev.cuh -- device helpers of the lanes kernels (ddsp_lanes.cu): shared-memory vector loads, mbarrier
// operations with a BOUNDED wait, the copy-engine bulk copy (cp.async.bulk -> SASS UBLKCP) and the global
// reduction store.  Inline PTX for sm_100a; 32-bit shared-window addresses throughout.
//
// The CPU emulation (tests/emu) replaces this header by host stand-ins with the same names, so everything a
// kernel does to memory or to a barrier goes through a function declared here.
#pragma once

#include <cstdint>

namespace ddsp_dev {

// ---- shared memory ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void lds64(uint32_t addr, uint32_t* v) {
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v[0]), "=r"(v[1]) : "r"(addr));
}
__device__ __forceinline__ void lds128(uint32_t addr, uint32_t* v) {
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(addr));
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// ---- integer adds routed to a chosen pipe ------------------------------------------------------------------
// acc += v as IMAD (FMA pipe); `one` is a kernel argument equal to 1 so that the multiply is not folded away.
// The ALU pipe (PRMT, IADD3, LOP3: 64 lanes/clk/SM) is the busier one in the uint8 hot loop.
__device__ __forceinline__ void add_fma_pipe(uint32_t& acc, uint32_t v, uint32_t one) {
    asm("mad.lo.u32 %0, %1, %2, %0;" : "+r"(acc) : "r"(v), "r"(one));
}
// bytes 1 and 3 of w as two 16-bit lanes: (b1, 0, b3, 0)
__device__ __forceinline__ uint32_t odd_bytes(uint32_t w) { return __byte_perm(w, 0u, 0x4341u); }

// ---- mbarrier ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ long long clock_now() { return clock64(); }
// Wait for the phase of parity `parity`, but never forever: after `budget` SM clocks without completion, or as
// soon as another thread of the CTA has given up (*abort_flag != 0), return false.  A mismatch between the
// expected and the delivered byte count of a bulk copy then ends the kernel with an error code instead of
// hanging the GPU until the process is killed.
__device__ __forceinline__ bool mbar_wait(uint32_t bar, uint32_t parity, uint32_t abort_flag, long long budget) {
    if (mbar_try_wait(bar, parity)) return true;
    const long long t0 = clock_now();
    for (;;) {
        if (mbar_try_wait(bar, parity)) return true;
        if (lds32(abort_flag) != 0u) return false;
        if (clock_now() - t0 > budget) { sts32(abort_flag, 1u); return false; }
    }
}
// makes freshly initialised mbarriers visible to the copy engine (async proxy)
__device__ __forceinline__ void fence_barrier_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

// ---- copy engine -------------------------------------------------------------------------------------------
// global -> shared bulk copy; dst, src and bytes are multiples of 16; completion is counted in bytes on `bar`.
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// ---- global memory -----------------------------------------------------------------------------------------
__device__ __forceinline__ void st_global_u32(uint32_t* p, uint32_t v) { *p = v; }
__device__ __forceinline__ void st_global_f32(float* p, float v) { *p = v; }
// *p += v on an element that only this thread ever touches.  Default: a reduction store (SASS RED: no return
// value, the issuing thread does not wait).  -DDDSP_LANES_FLUSH_RMW=1: plain load / add / store instead (tuning
// knob, in case the L2's atomic units turn out to be the narrower path).
#ifndef DDSP_LANES_FLUSH_RMW
#define DDSP_LANES_FLUSH_RMW 0
#endif
__device__ __forceinline__ void red_add_u32(uint32_t* p, uint32_t v) {
#if DDSP_LANES_FLUSH_RMW
    *p += v;
#else
    asm volatile("red.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
#endif
}
// plain loads / stores of output elements: named so that the CPU emulation can range-check them
__device__ __forceinline__ uint32_t ld_global_u32(const uint32_t* p) { return *p; }
__device__ __forceinline__ uint4 ld_global_v4(const void* p) { return *reinterpret_cast<const uint4*>(p); }
__device__ __forceinline__ void report_status(int* status, int code) { atomicCAS(status, 0, code); }
__device__ __forceinline__ uint32_t ldg_u8(const uint8_t* p) { return (uint32_t)__ldg(p); }
__device__ __forceinline__ float ldg_f32(const float* p) { return __ldg(p); }
__device__ __forceinline__ void st_global_v2(void* p, uint32_t a, uint32_t b) { *reinterpret_cast<uint2*>(p) = make_uint2(a, b); }
__device__ __forceinline__ void st_global_v4(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    *reinterpret_cast<uint4*>(p) = make_uint4(a, b, c, d);
}

}  // namespace ddsp_dev
