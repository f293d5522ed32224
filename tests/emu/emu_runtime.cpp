// Runtime of the CPU emulation harness: one std::thread per CUDA thread of a CTA, CTAs one after another,
// a copy-engine thread for cp.async.bulk, mbarriers with the PTX counting rules.  The alignment and size rules
// of the real instructions are checked (16-byte bulk copies, 8-byte mbarriers, aligned vector accesses), and so
// is the RANGE of every access: shared-memory accesses against the CTA's dynamic shared memory, global accesses
// and bulk-copy sources against the registered device-memory extents (cudaMalloc stand-in + ddsp_emu_register).
// Test infrastructure only.
#include <pthread.h>
#include <unistd.h>

#include <atomic>
#include <chrono>
#include <condition_variable>
#include <cstdio>
#include <cstdlib>
#include <deque>
#include <mutex>
#include <thread>
#include <vector>

#include "emu_common.h"

namespace emu {

thread_local Ctx ctx;

namespace {

// One 64-bit atomic per mbarrier: phase (bits 48..), pending arrivals (bits 32..47), transaction bytes + 2^30
// (bits 0..31).  Every update is one acq_rel read-modify-write and a successful wait is an acquire load, so
// the only happens-before edges are those of the PTX model (arrive / complete_tx = release on THIS barrier,
// wait = acquire on THIS barrier) -- a shared mutex would order everything and hide races from TSan.
struct MBar { std::atomic<uint64_t> state{0}; int count = 0; std::atomic<bool> init{false}; };
constexpr uint64_t kTxBias = 1u << 30;
inline uint64_t pack(uint64_t phase, uint64_t pending, int64_t tx) { return (phase << 48) | (pending << 32) | (uint64_t)(tx + (int64_t)kTxBias); }
inline uint64_t ph_of(uint64_t v) { return v >> 48; }
inline uint64_t pend_of(uint64_t v) { return (v >> 32) & 0xffff; }
inline int64_t tx_of(uint64_t v) { return (int64_t)(v & 0xffffffffu) - (int64_t)kTxBias; }
struct Copy { uint32_t dst; const void* src; uint32_t bytes; uint32_t bar; };

struct Cta {
    std::vector<uint8_t> smem;
    size_t smem_bytes = 0;
    unsigned nthreads = 0;
    pthread_barrier_t cta_bar;
    std::vector<pthread_barrier_t> warp_bar;
    std::vector<unsigned> shfl;         // [nthreads]
    MBar mbar[128];                     // mbarriers live in the first 1 KB of shared memory
    std::mutex q_mutex;
    std::deque<Copy> queue;
    bool stop = false;
    std::atomic<long> faults{0};
};
Cta* cta = nullptr;
std::atomic<long> total_faults{0};
std::atomic<long> printed{0};

void fault(const char* what, long a = 0, long b = 0) {
    if (printed.fetch_add(1) < 20) std::fprintf(stderr, "EMU FAULT: %s (%ld, %ld)\n", what, a, b);
    if (cta) ++cta->faults; else ++total_faults;
}

// registered device-memory extents: changed only between launches (cudaMalloc / cudaFree / register)
struct Extent { uintptr_t lo, hi; };
std::mutex ext_mutex;
std::vector<Extent> extents;

// pending -= arrivals, tx += dtx; the phase completes when both reach zero
bool update(MBar& m, int arrivals, int64_t dtx) {
    uint64_t old = m.state.load(std::memory_order_relaxed), nv;
    do {
        uint64_t phase = ph_of(old), pending = pend_of(old);
        int64_t tx = tx_of(old) + dtx;
        if ((int64_t)pending < arrivals) return false;
        pending -= arrivals;
        if (pending == 0 && tx == 0) { phase = (phase + 1) & 0xffff; pending = (uint64_t)m.count; }
        nv = pack(phase, pending, tx);
    } while (!m.state.compare_exchange_weak(old, nv, std::memory_order_acq_rel, std::memory_order_relaxed));
    return true;
}

void engine_main(int delay_us) {
    for (;;) {
        Copy c;
        {
            std::unique_lock<std::mutex> l(cta->q_mutex);
            if (cta->queue.empty()) {
                if (cta->stop) return;
                l.unlock();
                std::this_thread::yield();
                continue;
            }
            c = cta->queue.front();
            cta->queue.pop_front();
        }
        if (delay_us > 0) usleep(delay_us);
        check_global(c.src, c.bytes, false);
        std::memcpy(cta->smem.data() + c.dst, c.src, c.bytes);
        update(cta->mbar[c.bar / 8], 0, -(int64_t)c.bytes);
    }
}

}  // namespace

uint8_t* smem() { return cta->smem.data(); }

uint8_t* smem_at(uint32_t addr, uint32_t n, uint32_t align) {
    if ((size_t)addr + n > cta->smem_bytes) { fault("shared-memory access out of range", addr, n); return cta->smem.data() + cta->smem_bytes; }
    if (addr % align) fault("misaligned shared-memory access", addr, align);
    return cta->smem.data() + addr;
}

void* dev_alloc(size_t n) {
    void* p = nullptr;
    if (posix_memalign(&p, 256, n ? n : 1)) return nullptr;
    std::lock_guard<std::mutex> l(ext_mutex);
    extents.push_back(Extent{(uintptr_t)p, (uintptr_t)p + n});
    return p;
}
void dev_free(void* p) {
    if (!p) return;
    {
        std::lock_guard<std::mutex> l(ext_mutex);
        for (size_t i = 0; i < extents.size(); ++i)
            if (extents[i].lo == (uintptr_t)p) { extents.erase(extents.begin() + i); break; }
    }
    std::free(p);
}
void check_global(const void* p, size_t n, bool write) {
    const uintptr_t a = (uintptr_t)p;
    for (const Extent& e : extents)          // a handful of entries; only read while a launch is running
        if (a >= e.lo && a + n <= e.hi) return;
    fault(write ? "global WRITE outside every registered device buffer" : "global READ outside every registered device buffer",
          (long)a, (long)n);
}
void check_aligned(const void* p, size_t align) {
    if ((uintptr_t)p % align) fault("misaligned global vector access", (long)(uintptr_t)p, (long)align);
}
void yield() { std::this_thread::yield(); }

void mbar_init(uint32_t bar, int count) {
    if (bar % 8 || bar >= 1024) { fault("mbarrier address", bar); return; }
    MBar& m = cta->mbar[bar / 8];
    m.count = count;
    m.state.store(pack(0, (uint64_t)count, 0), std::memory_order_relaxed);
    m.init.store(true, std::memory_order_relaxed);
}

void mbar_arrive(uint32_t bar, uint32_t expect_tx_bytes) {
    if (bar % 8 || bar >= 1024 || !cta->mbar[bar / 8].init.load(std::memory_order_relaxed)) { fault("arrive on a bad mbarrier", bar); return; }
    if (!update(cta->mbar[bar / 8], 1, (int64_t)expect_tx_bytes)) fault("more arrivals than the mbarrier's count", bar);
}

bool mbar_test(uint32_t bar, uint32_t parity) {
    if (bar % 8 || bar >= 1024 || !cta->mbar[bar / 8].init.load(std::memory_order_relaxed)) { fault("wait on a bad mbarrier", bar); return true; }
    return (ph_of(cta->mbar[bar / 8].state.load(std::memory_order_acquire)) & 1u) != (parity & 1u);
}

void bulk_copy(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    if (dst % 16 || (uintptr_t)src % 16 || bytes % 16 || bytes == 0) fault("cp.async.bulk alignment/size", dst, bytes);
    if ((size_t)dst + bytes > cta->smem_bytes) { fault("cp.async.bulk beyond shared memory", dst, bytes); return; }
    check_global(src, bytes, false);
    std::lock_guard<std::mutex> l(cta->q_mutex);
    cta->queue.push_back(Copy{dst, src, bytes, bar});
}

void syncthreads() { pthread_barrier_wait(&cta->cta_bar); }
void syncwarp() { pthread_barrier_wait(&cta->warp_bar[ctx.tid / 32]); }
unsigned shfl_xor(unsigned v, int lane_mask) {
    cta->shfl[ctx.tid] = v;
    syncwarp();
    const unsigned r = cta->shfl[(ctx.tid & ~31u) | ((ctx.tid ^ (unsigned)lane_mask) & 31u)];
    syncwarp();
    return r;
}

long faults() { return total_faults.load(); }

void launch_seq(unsigned grid, unsigned nthreads, const std::function<void()>& body) {
    const unsigned nworkers = std::max(1u, std::min(8u, std::thread::hardware_concurrency()));
    std::atomic<unsigned> next{0};
    std::vector<std::thread> th;
    for (unsigned w = 0; w < nworkers; ++w)
        th.emplace_back([&]() {
            for (unsigned b = next.fetch_add(1); b < grid; b = next.fetch_add(1))
                for (unsigned t = 0; t < nthreads; ++t) {
                    ctx.tid = t;
                    ctx.bid = b;
                    body();
                }
        });
    for (auto& t : th) t.join();
}

void launch(unsigned grid, unsigned nthreads, size_t smem_bytes, const std::function<void()>& body) {
    const char* d = getenv("DDSP_EMU_TMA_DELAY_US");
    const int delay_us = d ? atoi(d) : 0;
    for (unsigned b = 0; b < grid; ++b) {
        Cta c;
        c.smem.assign(smem_bytes + 64, 0xA5);       // shared memory starts as garbage, not zero
        c.smem_bytes = smem_bytes;
        c.nthreads = nthreads;
        c.shfl.assign(nthreads, 0);
        pthread_barrier_init(&c.cta_bar, nullptr, nthreads);
        c.warp_bar.resize((nthreads + 31) / 32);
        for (unsigned w = 0; w < c.warp_bar.size(); ++w)
            pthread_barrier_init(&c.warp_bar[w], nullptr, std::min(32u, nthreads - 32 * w));
        cta = &c;
        std::thread engine(engine_main, delay_us);
        std::vector<std::thread> th;
        th.reserve(nthreads);
        for (unsigned t = 0; t < nthreads; ++t)
            th.emplace_back([&, t]() {
                ctx.tid = t;
                ctx.bid = b;
                body();
            });
        for (auto& t : th) t.join();
        {
            std::lock_guard<std::mutex> l(c.q_mutex);
            if (!c.queue.empty()) fault("CTA exited with bulk copies in flight");
            c.stop = true;
        }
        engine.join();
        for (int i = 0; i < 128; ++i)
            if (c.mbar[i].init.load() && tx_of(c.mbar[i].state.load()) != 0) fault("mbarrier with outstanding transaction bytes", i * 8, tx_of(c.mbar[i].state.load()));
        total_faults += c.faults;
        pthread_barrier_destroy(&c.cta_bar);
        for (auto& wb : c.warp_bar) pthread_barrier_destroy(&wb);
        cta = nullptr;
    }
}

}  // namespace emu

extern "C" long ddsp_emu_faults(void) { return emu::faults(); }
// caller-owned "device" buffers (the tests' input / output arrays): exact extents, so that a kernel that reads or
// writes one byte outside them is reported
extern "C" void ddsp_emu_register(const void* p, size_t n) {
    std::lock_guard<std::mutex> l(emu::ext_mutex);
    emu::extents.push_back(emu::Extent{(uintptr_t)p, (uintptr_t)p + n});
}
extern "C" void ddsp_emu_unregister(const void* p) {
    std::lock_guard<std::mutex> l(emu::ext_mutex);
    for (size_t i = 0; i < emu::extents.size(); ++i)
        if (emu::extents[i].lo == (uintptr_t)p) { emu::extents.erase(emu::extents.begin() + i); break; }
}
