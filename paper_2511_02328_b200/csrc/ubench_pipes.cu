// ubench_pipes.cu -- per-SM issue rates of the instructions the dedispersion hot loops are made of, and the
// shared-memory load bandwidth per load width.  These numbers fix the roofline denominator P_add
// (148 SM x 128 thread-adds/clk/SM x f_SM) and show which pipe binds a given mix.
//
//   build + run:  python -m paper_2511_02328_b200.ubench        (nvcc, sm_100a; prints one table)
//
// Method: one CTA per SM, every thread runs `kIters` iterations of an unrolled body of independent dependency
// chains (8 accumulators) made of ONE opcode class, forced through inline PTX so that ptxas cannot fold it;
// cycles = clock64 difference of the slowest CTA; rate = threads x iters x ops / cycles per SM.  Shared-memory
// loads read a different, conflict-free address every iteration (volatile asm, so nothing is hoisted) and feed
// an XOR chain.  Nothing here touches global memory except one result word per thread.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

#define CHECK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { std::printf("CUDA error %s at %s:%d\n", cudaGetErrorString(e_), __FILE__, __LINE__); return 1; } } while (0)

enum Op { kIadd3, kIadd2, kImad, kLop3, kPrmt, kFadd, kIadd3Imad, kHotMix, kNumOps };
const char* kOpName[kNumOps] = {"IADD3 (a+b+c)", "IADD (a+b)", "IMAD (a*one+c)", "LOP3", "PRMT", "FADD",
                                "IADD3 + IMAD 1:1", "2 PRMT + 2 IMAD + 1 IADD3 (uint8 hot mix, no loads)"};
const int kOpsPerBody[kNumOps] = {8, 8, 8, 8, 8, 8, 16, 40};

constexpr int kIters = 4096;

template <int OP>
__global__ void __launch_bounds__(1024) pipe_kernel(uint32_t* out, long long* cycles, uint32_t one, uint32_t seed) {
    uint32_t a[8], b[8];
    float f[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) { a[k] = seed + threadIdx.x * 8 + k; b[k] = seed * 3 + k; f[k] = (float)(seed + k); }
    const float fone = (float)one;
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (OP == kIadd3) asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(a[k]) : "r"(b[k]), "r"(one));
            if (OP == kIadd2) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[k]) : "r"(b[k]));
            if (OP == kImad) asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a[k]) : "r"(b[k]), "r"(one));
            if (OP == kLop3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[k]) : "r"(b[k]), "r"(one));
            if (OP == kPrmt) asm volatile("prmt.b32 %0, %0, %1, 0x4341;" : "+r"(a[k]) : "r"(b[k]));
            if (OP == kFadd) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(f[k]) : "f"(fone));
            if (OP == kIadd3Imad) {
                asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(a[k]) : "r"(b[k]), "r"(one));
                asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(b[k]) : "r"(a[k]), "r"(one));
            }
            if (OP == kHotMix) {     // per pair of 32-bit words w0 = a[k], w1 = b[k]: what the lanes kernel issues
                uint32_t p0, p1;
                asm volatile("prmt.b32 %0, %1, 0, 0x4341;" : "=r"(p0) : "r"(a[k]));
                asm volatile("prmt.b32 %0, %1, 0, 0x4341;" : "=r"(p1) : "r"(b[k]));
                asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a[k]) : "r"(b[k]), "r"(one));
                asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(b[k]) : "r"(a[k]), "r"(one));
                asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(a[k]) : "r"(p0), "r"(p1));
            }
        }
    }
    const long long t1 = clock64();
    uint32_t r = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) r ^= a[k] ^ b[k] ^ __float_as_uint(f[k]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

// WIDTH = 4, 8, 16 bytes per lane per load; a warp reads 32 * WIDTH contiguous bytes (conflict-free)
template <int WIDTH>
__global__ void __launch_bounds__(1024) lds_kernel(uint32_t* out, long long* cycles, uint32_t step) {
    extern __shared__ __align__(16) uint8_t smem[];
    const uint32_t bytes = 64 * 1024;
    for (uint32_t i = threadIdx.x; i < bytes / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(smem)[i] = i * 2654435761u;
    __syncthreads();
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t lane_off = (threadIdx.x & 31) * WIDTH + (threadIdx.x >> 5) * 32 * WIDTH;
    uint32_t acc[4] = {0, 0, 0, 0};
    uint32_t pos = 0;
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uint32_t addr = base + ((pos + lane_off + k * 1024u * WIDTH / 4) & (bytes - 1) & ~(uint32_t)(WIDTH - 1));
            uint32_t v[4] = {0, 0, 0, 0};
            if (WIDTH == 4) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v[0]) : "r"(addr));
            if (WIDTH == 8) asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v[0]), "=r"(v[1]) : "r"(addr));
            if (WIDTH == 16) asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(addr));
            acc[k & 3] ^= v[0] ^ v[1] ^ v[2] ^ v[3];
        }
        pos += step * WIDTH;
    }
    const long long t1 = clock64();
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc[0] ^ acc[1] ^ acc[2] ^ acc[3];
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

typedef void (*PipeKernel)(uint32_t*, long long*, uint32_t, uint32_t);
const PipeKernel kPipe[kNumOps] = {pipe_kernel<kIadd3>, pipe_kernel<kIadd2>, pipe_kernel<kImad>, pipe_kernel<kLop3>,
                                   pipe_kernel<kPrmt>, pipe_kernel<kFadd>, pipe_kernel<kIadd3Imad>, pipe_kernel<kHotMix>};

int main() {
    cudaDeviceProp prop;
    CHECK(cudaGetDeviceProperties(&prop, 0));
    const int sms = prop.multiProcessorCount;
    std::printf("# %s, %d SMs, clock %d kHz\n", prop.name, sms, prop.clockRate);
    uint32_t* out = nullptr;
    long long* cyc = nullptr;
    CHECK(cudaMalloc(&out, (size_t)sms * 1024 * 4));
    CHECK(cudaMalloc(&cyc, (size_t)sms * 8));
    std::vector<long long> h(sms);
    std::printf("| instruction mix | threads/SM | thread-instr/clk/SM |\n|---|---|---|\n");
    for (int threads : {256, 512, 1024})
        for (int op = 0; op < kNumOps; ++op) {
            for (int rep = 0; rep < 2; ++rep) kPipe[op]<<<sms, threads>>>(out, cyc, 1u, 12345u);
            CHECK(cudaDeviceSynchronize());
            CHECK(cudaMemcpy(h.data(), cyc, (size_t)sms * 8, cudaMemcpyDeviceToHost));
            const long long worst = *std::max_element(h.begin(), h.end());
            std::printf("| %s | %d | %.2f |\n", kOpName[op], threads, (double)threads * kIters * kOpsPerBody[op] / (double)worst);
        }
    std::printf("\n| shared-memory load | threads/SM | bytes/clk/SM | warp-loads/clk/SM |\n|---|---|---|---|\n");
    CHECK(cudaFuncSetAttribute(lds_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
    CHECK(cudaFuncSetAttribute(lds_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
    CHECK(cudaFuncSetAttribute(lds_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
    for (int threads : {256, 512, 1024})
        for (int width : {4, 8, 16}) {
            for (int rep = 0; rep < 2; ++rep) {
                if (width == 4) lds_kernel<4><<<sms, threads, 64 * 1024>>>(out, cyc, 37u);
                if (width == 8) lds_kernel<8><<<sms, threads, 64 * 1024>>>(out, cyc, 37u);
                if (width == 16) lds_kernel<16><<<sms, threads, 64 * 1024>>>(out, cyc, 37u);
            }
            CHECK(cudaDeviceSynchronize());
            CHECK(cudaMemcpy(h.data(), cyc, (size_t)sms * 8, cudaMemcpyDeviceToHost));
            const long long worst = *std::max_element(h.begin(), h.end());
            const double loads = (double)threads * kIters * 8;
            std::printf("| LDS.%d | %d | %.1f | %.3f |\n", width * 8, threads, loads * width / (double)worst, loads / 32.0 / (double)worst);
        }
    cudaFree(out);
    cudaFree(cyc);
    return 0;
}
