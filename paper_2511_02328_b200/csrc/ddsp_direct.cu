// ddsp_direct.cu -- DDSP_KERNEL_DIRECT: the plain definition on the GPU, one thread per output element.
//
//   D[i][t] = sum over unmasked c (ascending) of x_ds[c][t + d(i,c)]
//   x_ds[c][u] = sum_{k<ds} x[c][ds*u + k], zero beyond nsamp
//
// It runs every plan (any pitch, alignment, downsample factor, mask, DM order) and is the fallback
// and the in-library cross-check of the tiled kernels.  Each warp reads 32 consecutive samples of a
// channel row (coalesced); the delay d(i,c) is uniform over the block.  All element offsets are 64-bit
// (config 2's input is 6.25e9 bytes).
#include "ddsp_internal.h"
#include "ddsp_dev.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kPerThread = 4;  // output samples per thread, strided by kThreads (keeps loads coalesced)

template <typename TIn, typename TAcc>
__device__ __forceinline__ TAcc bin_sum(const TIn* __restrict__ row, int64_t nsamp, int ds, int64_t u);

// uint8: exact in uint32.
template <>
__device__ __forceinline__ uint32_t bin_sum<uint8_t, uint32_t>(const uint8_t* __restrict__ row,
                                                               int64_t nsamp, int ds, int64_t u) {
    const int64_t j0 = (int64_t)ds * u;
    uint32_t s = 0;
    for (int k = 0; k < ds; ++k) {
        const int64_t j = j0 + k;
        if (j < nsamp) s += __ldg(row + j);
    }
    return s;
}

// float32: ((x0 + x1) + x2) + ... in fp32, missing samples are +0 (R8, R9).
template <>
__device__ __forceinline__ float bin_sum<float, float>(const float* __restrict__ row, int64_t nsamp,
                                                       int ds, int64_t u) {
    const int64_t j0 = (int64_t)ds * u;
    float s = (j0 < nsamp) ? __ldg(row + j0) : 0.0f;
    for (int k = 1; k < ds; ++k) {
        const int64_t j = j0 + k;
        const float v = (j < nsamp) ? __ldg(row + j) : 0.0f;
        s = __fadd_rn(s, v);
    }
    return s;
}

__device__ __forceinline__ void store_out(uint32_t* p, uint32_t v) { ddsp_dev::st_global_u32(p, v); }
__device__ __forceinline__ void store_out(float* p, float v) { ddsp_dev::st_global_f32(p, v); }
__device__ __forceinline__ void accumulate(uint32_t& acc, uint32_t v) { acc += v; }
__device__ __forceinline__ void accumulate(float& acc, float v) { acc = __fadd_rn(acc, v); }  // never an FMA

template <typename TIn, typename TAcc, bool kDs1>
__global__ void __launch_bounds__(kThreads)
ddsp_direct_kernel(const TIn* __restrict__ in, TAcc* __restrict__ out, const int32_t* __restrict__ delays,
                   const int32_t* __restrict__ chan_list, int nlist, int nchan, int ndm, int64_t nsamp, int ds,
                   int64_t nsamp_out, int64_t in_pitch, int64_t out_pitch) {
    const int64_t t0 = (int64_t)blockIdx.x * (kThreads * kPerThread) + threadIdx.x;
    for (int i = blockIdx.y; i < ndm; i += gridDim.y) {  // trial (dm_list order)
    const int32_t* __restrict__ drow = delays + (size_t)i * nchan;
    TAcc acc[kPerThread];
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) acc[k] = TAcc(0);
    for (int l = 0; l < nlist; ++l) {
        const int c = __ldg(chan_list + l);
        const int64_t d = __ldg(drow + c);
        const TIn* __restrict__ row = in + (size_t)c * (size_t)in_pitch;
#pragma unroll
        for (int k = 0; k < kPerThread; ++k) {
            const int64_t t = t0 + (int64_t)k * kThreads;
            if (t < nsamp_out) {
                TAcc v;
                if (kDs1) v = (TAcc)__ldg(row + t + d);
                else v = bin_sum<TIn, TAcc>(row, nsamp, ds, t + d);
                accumulate(acc[k], v);
            }
        }
    }
    TAcc* __restrict__ orow = out + (size_t)i * (size_t)out_pitch;
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
        const int64_t t = t0 + (int64_t)k * kThreads;
        if (t < nsamp_out) store_out(orow + t, acc[k]);
    }
    }
}

}  // namespace

cudaError_t ddsp_launch_direct(const ddsp_plan* p, const void* d_in, void* d_out, cudaStream_t s) {
    const int64_t per_block = (int64_t)kThreads * kPerThread;
    const int64_t gx = (p->nsamp_out + per_block - 1) / per_block;
    if (gx > 2147483647LL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)gx, (unsigned)(p->ndm < 65535 ? p->ndm : 65535));
    const int nlist = (int)p->chan_list.size();
    if (p->in_dtype == DDSP_IN_U8) {
        auto in = (const uint8_t*)d_in;
        auto out = (uint32_t*)d_out;
        if (p->ds == 1)
            ddsp_direct_kernel<uint8_t, uint32_t, true><<<grid, kThreads, 0, s>>>(
                in, out, p->d_delays, p->d_chan_list, nlist, p->nchan, p->ndm, p->nsamp, p->ds, p->nsamp_out,
                p->in_pitch, p->out_pitch);
        else
            ddsp_direct_kernel<uint8_t, uint32_t, false><<<grid, kThreads, 0, s>>>(
                in, out, p->d_delays, p->d_chan_list, nlist, p->nchan, p->ndm, p->nsamp, p->ds, p->nsamp_out,
                p->in_pitch, p->out_pitch);
    } else {
        auto in = (const float*)d_in;
        auto out = (float*)d_out;
        if (p->ds == 1)
            ddsp_direct_kernel<float, float, true><<<grid, kThreads, 0, s>>>(
                in, out, p->d_delays, p->d_chan_list, nlist, p->nchan, p->ndm, p->nsamp, p->ds, p->nsamp_out,
                p->in_pitch, p->out_pitch);
        else
            ddsp_direct_kernel<float, float, false><<<grid, kThreads, 0, s>>>(
                in, out, p->d_delays, p->d_chan_list, nlist, p->nchan, p->ndm, p->nsamp, p->ds, p->nsamp_out,
                p->in_pitch, p->out_pitch);
    }
    return cudaGetLastError();
}
