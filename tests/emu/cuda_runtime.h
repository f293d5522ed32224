// Fake <cuda_runtime.h> of the CPU emulation harness (tests/emu): just enough of the CUDA runtime API and
// of the device-side keywords for the kernels' sources (paper_2511_02328_b200/csrc/*.cu and ddsp_plan.cpp) to
// compile with g++ and run with one std::thread per CUDA thread.  Test infrastructure only: nothing in the
// product includes this file.  "Device memory" is host memory whose extents are registered, so that the
// stand-ins of the device helpers can check every global access against them (emu::check_global).
#pragma once

#include <cstddef>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <functional>

// ---- keywords --------------------------------------------------------------------------------------
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __launch_bounds__(...)
#define __align__(n)
#define __grid_constant__

// ---- vector types ----------------------------------------------------------------------------------
struct int2 { int x, y; };
struct uint2 { unsigned x, y; };
struct uint3 { unsigned x, y, z; };
struct uint4 { unsigned x, y, z, w; };
inline uint2 make_uint2(unsigned x, unsigned y) { return uint2{x, y}; }
inline uint4 make_uint4(unsigned x, unsigned y, unsigned z, unsigned w) { return uint4{x, y, z, w}; }

// ---- runtime API -----------------------------------------------------------------------------------
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2, cudaErrorInvalidConfiguration = 9 };
enum cudaMemcpyKind { cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
typedef void* cudaStream_t;
struct cudaDeviceProp { int multiProcessorCount; size_t sharedMemPerBlockOptin; };

inline cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
inline cudaError_t cudaGetDeviceProperties(cudaDeviceProp* p, int) {
    p->multiProcessorCount = 148;
    p->sharedMemPerBlockOptin = 232448;
    return cudaSuccess;
}
namespace emu {
void* dev_alloc(size_t n);                         // registers [p, p + n) as device memory
void dev_free(void* p);
void check_global(const void* p, size_t n, bool write);   // faults unless [p, p + n) lies inside one registered extent
}
inline cudaError_t cudaMalloc(void** p, size_t n) { *p = emu::dev_alloc(n); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
inline cudaError_t cudaFree(void* p) { emu::dev_free(p); return cudaSuccess; }
inline cudaError_t cudaMemset(void* p, int v, size_t n) { std::memset(p, v, n); return cudaSuccess; }
inline cudaError_t cudaMemcpy(void* d, const void* s, size_t n, cudaMemcpyKind) { std::memcpy(d, s, n); return cudaSuccess; }
inline cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t) { std::memcpy(d, s, n); return cudaSuccess; }
inline cudaError_t cudaMemcpy2DAsync(void* d, size_t dp, const void* s, size_t sp, size_t w, size_t h, cudaMemcpyKind, cudaStream_t) {
    for (size_t r = 0; r < h; ++r) std::memcpy((char*)d + r * dp, (const char*)s + r * sp, w);
    return cudaSuccess;
}
inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
// streams and events: everything runs synchronously in issue order, which is one legal schedule
typedef void* cudaEvent_t;
enum { cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2 };
inline cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned) { *s = std::malloc(1); return cudaSuccess; }
inline cudaError_t cudaStreamDestroy(cudaStream_t s) { std::free(s); return cudaSuccess; }
inline cudaError_t cudaEventCreateWithFlags(cudaEvent_t* e, unsigned) { *e = std::malloc(1); return cudaSuccess; }
inline cudaError_t cudaEventDestroy(cudaEvent_t e) { std::free(e); return cudaSuccess; }
inline cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t) { return cudaSuccess; }
inline cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned) { return cudaSuccess; }
inline cudaError_t cudaGetLastError() { return cudaSuccess; }
template <class F> cudaError_t cudaFuncSetAttribute(F, cudaFuncAttribute, int) { return cudaSuccess; }

// ---- the emulated CTA (emu_runtime.cpp) ------------------------------------------------------------
namespace emu {
struct Ctx { unsigned tid, bid, bidy, gdimy, gdimx; };
extern thread_local Ctx ctx;
uint8_t* smem();                                   // dynamic shared memory of the running CTA
void launch(unsigned grid, unsigned nthreads, size_t smem_bytes, const std::function<void()>& body);
// kernels without shared memory, barriers or shuffles: the CUDA threads of a block run one after another
void launch_seq(unsigned grid, unsigned nthreads, const std::function<void()>& body);
void syncthreads();
void syncwarp();
unsigned shfl_xor(unsigned v, int lane_mask);
}  // namespace emu

struct EmuIdx { unsigned x, y; };
struct dim3 {
    unsigned x, y, z;
    dim3(unsigned x_ = 1, unsigned y_ = 1, unsigned z_ = 1) : x(x_), y(y_), z(z_) {}
};
#define threadIdx (EmuIdx{emu::ctx.tid, 0u})
#define blockIdx (EmuIdx{emu::ctx.bid, emu::ctx.bidy})
#define gridDim (EmuIdx{emu::ctx.gdimx, emu::ctx.gdimy})

// one argument (a struct): a 1-D or 2-D grid, one emulated launch per grid row
template <class F, class A>
void emu_launch(F fn, dim3 grid, unsigned nthreads, size_t smem_bytes, cudaStream_t, const A& a) {
    for (unsigned y = 0; y < grid.y; ++y)
        emu::launch(grid.x, nthreads, smem_bytes, [&]() { emu::ctx.bidy = y; emu::ctx.gdimy = grid.y; emu::ctx.gdimx = grid.x; fn(a); });
}
// 2-D grid, any argument list, no synchronisation inside the kernel (the direct kernel, the interleave pass)
template <class F, class... A>
void emu_launch_v(F fn, dim3 grid, unsigned nthreads, size_t smem_bytes, cudaStream_t, A... a) {
    for (unsigned y = 0; y < grid.y; ++y)
        emu::launch_seq(grid.x, nthreads, [&]() { emu::ctx.bidy = y; emu::ctx.gdimy = grid.y; emu::ctx.gdimx = grid.x; fn(a...); });
}

// ---- device intrinsics -----------------------------------------------------------------------------
inline void __syncthreads() { emu::syncthreads(); }
inline void __syncwarp() { emu::syncwarp(); }
inline unsigned __shfl_xor_sync(unsigned, unsigned v, int m) { return emu::shfl_xor(v, m); }
template <class T> inline T __ldg(const T* p) { emu::check_global(p, sizeof(T), false); return *p; }
inline int min(int a, int b) { return a < b ? a : b; }
inline unsigned __byte_perm(unsigned x, unsigned y, unsigned s) {       // PTX prmt, default mode
    const uint64_t src = ((uint64_t)y << 32) | x;
    unsigned r = 0;
    for (int i = 0; i < 4; ++i) {
        const unsigned sel = (s >> (4 * i)) & 0xf;
        unsigned b = (unsigned)(src >> (8 * (sel & 7))) & 0xff;
        if (sel & 8) b = (b & 0x80) ? 0xff : 0x00;
        r |= b << (8 * i);
    }
    return r;
}
inline unsigned __dp4a(unsigned a, unsigned b, unsigned c) {
    for (int i = 0; i < 4; ++i) c += ((a >> (8 * i)) & 0xff) * ((b >> (8 * i)) & 0xff);
    return c;
}
inline float __fadd_rn(float a, float b) { return a + b; }
inline float __uint_as_float(unsigned u) { float f; std::memcpy(&f, &u, 4); return f; }
inline unsigned __float_as_uint(float f) { unsigned u; std::memcpy(&u, &f, 4); return u; }
