// Host stand-ins for paper_2511_02328_b200/csrc/ddsp_ring_common.cuh (same names, same semantics):
// shared-memory accesses go to the emulated CTA's buffer, mbarriers are counted under a mutex (arrive =
// release, wait = acquire, as in the PTX memory model), bulk copies are carried out by a separate
// "copy engine" thread.  Test infrastructure only (tests/emu).
#pragma once

#include <cstdint>
#include <cstring>

#include "cuda_runtime.h"

namespace emu {
void mbar_init(uint32_t bar, int count);
void mbar_arrive(uint32_t bar, uint32_t expect_tx_bytes);
bool mbar_test(uint32_t bar, uint32_t parity);
void bulk_copy(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar);
void yield();
}  // namespace emu

namespace ddsp_dev {

inline uint32_t smem_addr(const void* p) { return (uint32_t)((const uint8_t*)p - emu::smem()); }
inline uint32_t lds32(uint32_t addr) { uint32_t v; std::memcpy(&v, emu::smem() + addr, 4); return v; }
inline uint32_t lds8(uint32_t addr) { return emu::smem()[addr]; }
inline void lds128(uint32_t addr, uint32_t* v) { std::memcpy(v, emu::smem() + addr, 16); }
inline void sts32(uint32_t addr, uint32_t v) { std::memcpy(emu::smem() + addr, &v, 4); }
inline void sts128(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    const uint32_t v[4] = {a, b, c, d};
    std::memcpy(emu::smem() + addr, v, 16);
}
inline void add_fma_pipe(uint32_t& acc, uint32_t v, uint32_t one) { acc += v * one; }
inline void add_wide(uint64_t& acc, uint32_t v, uint32_t one) { acc += (uint64_t)v * one; }
inline void mbar_init(uint32_t bar, int count) { emu::mbar_init(bar, count); }
inline void mbar_arrive(uint32_t bar) { emu::mbar_arrive(bar, 0); }
inline void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) { emu::mbar_arrive(bar, bytes); }
inline void mbar_wait(uint32_t bar, uint32_t parity) {
    while (!emu::mbar_test(bar, parity)) emu::yield();
}
inline void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) { emu::bulk_copy(dst, src, bytes, bar); }
inline void fence_barrier_init() {}
inline void fence_proxy_async_smem() {}
inline void st_global_v2(uint32_t* p, uint32_t a, uint32_t b) { p[0] = a; p[1] = b; }

}  // namespace ddsp_dev
