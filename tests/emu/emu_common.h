// Host stand-ins for paper_2511_02328_b200/csrc/ddsp_dev.cuh (same names, same semantics): shared-memory
// accesses go to the emulated CTA's buffer (range-checked), mbarriers are counted with the PTX rules (arrive =
// release, successful wait = acquire), bulk copies are carried out by a separate "copy engine" thread, and
// every global access is checked against the registered device-memory extents.  Test infrastructure only.
#pragma once

#include <chrono>
#include <cstdint>
#include <cstring>

#include "cuda_runtime.h"

namespace emu {
void mbar_init(uint32_t bar, int count);
void mbar_arrive(uint32_t bar, uint32_t expect_tx_bytes);
bool mbar_test(uint32_t bar, uint32_t parity);
void bulk_copy(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar);
void yield();
uint8_t* smem_at(uint32_t addr, uint32_t n, uint32_t align);    // faults on a range or alignment violation
void check_aligned(const void* p, size_t align);
}  // namespace emu

namespace ddsp_dev {

inline uint32_t smem_addr(const void* p) { return (uint32_t)((const uint8_t*)p - emu::smem()); }
inline uint32_t lds32(uint32_t addr) { uint32_t v; std::memcpy(&v, emu::smem_at(addr, 4, 4), 4); return v; }
inline uint32_t lds8(uint32_t addr) { return *emu::smem_at(addr, 1, 1); }
inline void lds64(uint32_t addr, uint32_t* v) { std::memcpy(v, emu::smem_at(addr, 8, 8), 8); }
inline void lds128(uint32_t addr, uint32_t* v) { std::memcpy(v, emu::smem_at(addr, 16, 16), 16); }
inline void sts32(uint32_t addr, uint32_t v) { std::memcpy(emu::smem_at(addr, 4, 4), &v, 4); }
inline void sts128(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    const uint32_t v[4] = {a, b, c, d};
    std::memcpy(emu::smem_at(addr, 16, 16), v, 16);
}
inline void add_fma_pipe(uint32_t& acc, uint32_t v, uint32_t one) { acc += v * one; }
inline void add_wide(uint64_t& acc, uint32_t v, uint32_t one) { acc += (uint64_t)v * one; }
inline uint32_t odd_bytes(uint32_t w) { return __byte_perm(w, 0u, 0x4341u); }
inline void mbar_init(uint32_t bar, int count) { emu::mbar_init(bar, count); }
inline void mbar_arrive(uint32_t bar) { emu::mbar_arrive(bar, 0); }
inline void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) { emu::mbar_arrive(bar, bytes); }
inline bool mbar_try_wait(uint32_t bar, uint32_t parity) { return emu::mbar_test(bar, parity); }
inline long long clock_now() {     // "SM clocks": nanoseconds of the host's steady clock
    return (long long)std::chrono::duration_cast<std::chrono::nanoseconds>(std::chrono::steady_clock::now().time_since_epoch()).count();
}
// The abort flag is shared memory that any thread may write while others poll it: relaxed atomics here, a
// plain ld/st.shared on the device (the flag only ever goes from 0 to 1).
inline uint32_t abort_load(uint32_t flag) { return __atomic_load_n((uint32_t*)emu::smem_at(flag, 4, 4), __ATOMIC_RELAXED); }
inline void abort_store(uint32_t flag) { __atomic_store_n((uint32_t*)emu::smem_at(flag, 4, 4), 1u, __ATOMIC_RELAXED); }
inline bool mbar_wait(uint32_t bar, uint32_t parity, uint32_t abort_flag, long long budget) {
    if (emu::mbar_test(bar, parity)) return true;
    const long long t0 = clock_now();
    for (;;) {
        if (emu::mbar_test(bar, parity)) return true;
        if (abort_load(abort_flag) != 0u) return false;
        if (clock_now() - t0 > budget * 8) { abort_store(abort_flag); return false; }   // 512 host threads are slow
        emu::yield();
    }
}
inline void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) { emu::bulk_copy(dst, src, bytes, bar); }
inline void fence_barrier_init() {}
inline void fence_proxy_async_smem() {}
inline void st_global_u32(uint32_t* p, uint32_t v) { emu::check_global(p, 4, true); *p = v; }
inline void st_global_f32(float* p, float v) { emu::check_global(p, 4, true); *p = v; }
inline void red_add_u32(uint32_t* p, uint32_t v) { emu::check_global(p, 4, true); __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
inline uint32_t ld_global_u32(const uint32_t* p) { emu::check_global(p, 4, false); return *p; }
inline uint4 ld_global_v4(const void* p) {
    emu::check_global(p, 16, false);
    emu::check_aligned(p, 16);
    uint4 v;
    std::memcpy(&v, p, 16);
    return v;
}
inline void report_status(int* status, int code) {
    emu::check_global(status, 4, true);
    int zero = 0;
    __atomic_compare_exchange_n(status, &zero, code, false, __ATOMIC_RELAXED, __ATOMIC_RELAXED);
}
inline uint32_t ldg_u8(const uint8_t* p) { emu::check_global(p, 1, false); return *p; }
inline float ldg_f32(const float* p) { emu::check_global(p, 4, false); return *p; }
inline void st_global_v2(void* p, uint32_t a, uint32_t b) {
    emu::check_global(p, 8, true);
    emu::check_aligned(p, 8);
    const uint32_t v[2] = {a, b};
    std::memcpy(p, v, 8);
}
inline void st_global_v4(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    emu::check_global(p, 16, true);
    emu::check_aligned(p, 16);
    const uint32_t v[4] = {a, b, c, d};
    std::memcpy(p, v, 16);
}

}  // namespace ddsp_dev
