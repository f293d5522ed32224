// ddsp_tiled.cu -- DDSP_KERNEL_TILED: shared-memory tiled brute-force dedispersion.
//
//   D[i][t] = sum over unmasked c of x[c][t + d(i,c)]
//
// One CTA computes a tile of BDM consecutive (DM-sorted) trials x T output samples and loops over the
// unmasked channels in chunks.  For every chunk the needed window of each channel row,
// [t0 + d(i_first,c), t0 + T + d(i_last,c)), is staged once into shared memory and serves all BDM
// trials ("shared-memory tiling" is the prior art; tile shapes, the phase copies and
// the packed accumulators below are ours).
//
// uint8 path (ds = 1).  The shifted read x[c][t + d] lands on an arbitrary byte of the row, but a
// 32-bit shared-memory load must be 4-byte aligned.  The row is therefore staged as FOUR phase copies,
// copy_p[i] = row[i + p]; a trial whose offset is q reads word (q >> 2) of copy (q & 3): always
// aligned, always conflict-free (lanes read consecutive words), no per-load realignment.  A loaded
// word holds 4 consecutive samples; it is split into even and odd bytes (two registers of 2 x 16-bit
// lanes) and added to packed accumulators: 4 sample-adds for 2 integer adds.  The 16-bit lanes are
// flushed to the uint32 output rows (global memory, L2-resident, owned by this thread) every 256
// channels (255 * 257 < 65536).
//
// float32 path.  One staged copy (4-byte elements are always aligned); one fp32 register accumulator
// per output element, channels added in ascending order with __fadd_rn: bit-identical to the
// sequential sum (R9).  With ds > 1 the bins ((x0 + x1) + x2) + ... are formed at staging.
#include <algorithm>
#include <cstdio>
#include <vector>

#include "ddsp_internal.h"

namespace {

// ------------------------------------------------------------------------------------------------
// compile-time geometry
// ------------------------------------------------------------------------------------------------
constexpr int kThreads = 512;          // 16 warps = 4 time slabs x 4 trial groups
constexpr int kSlabs = 4;
constexpr int kGroups = 4;
constexpr int kWT = 4;                 // 32-bit words per thread per trial (strided by 32 lanes)
constexpr int kTileT = kSlabs * kWT * 128;   // 2048 output samples per CTA (uint8 path)
constexpr int kFlushEvery = 256;       // channels between flushes of the 16-bit lanes
constexpr int kMaxUnits = 4;           // 16-byte staging units per thread per chunk
constexpr int kMaxChunkC = 32;

struct TiledArgs {
    const uint8_t* in;
    uint32_t* out;
    const int32_t* base;      // [nblk][nch_pad] 16-byte-aligned first byte of each row window (rel. to t0)
    const uint32_t* off;      // [nblk][nch_pad][bdm] phase * row_stride + (q >> 2) * 4
    const int32_t* rows;      // [nblk * bdm] output row of each sorted trial, -1 = padding
    const int32_t* chan;      // [nch_pad] channel index of each listed channel (padding repeats the last)
    int64_t in_pitch, out_pitch, nsamp_out, in_bytes;
    int nlist, nch_pad, nblk, chunk_c, nchunk, row_stride, units_per_row, out_vec, in_vec;
};

__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// ------------------------------------------------------------------------------------------------
// uint8, ds = 1
// ------------------------------------------------------------------------------------------------
template <int BDM_T>   // trials per thread; BDM = kGroups * BDM_T
__global__ void __launch_bounds__(kThreads, 1) ddsp_tiled_u8_kernel(const TiledArgs a) {
    constexpr int BDM = kGroups * BDM_T;
    extern __shared__ __align__(16) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slab = warp & (kSlabs - 1), grp = warp / kSlabs;
    const int blk = blockIdx.x % a.nblk;
    const int64_t tile = blockIdx.x / a.nblk;
    const int64_t t0 = tile * kTileT;

    const int stage_rows_bytes = a.chunk_c * 4 * a.row_stride;
    const int stage_bytes = stage_rows_bytes + a.chunk_c * BDM * 4;
    const uint32_t smem_base = (uint32_t)__cvta_generic_to_shared(smem);

    const int32_t* __restrict__ base_b = a.base + (size_t)blk * a.nch_pad;
    const uint32_t* __restrict__ off_b = a.off + (size_t)blk * a.nch_pad * BDM;

    // packed accumulators: E = samples (0,2), O = samples (1,3) of each owned word, 16-bit lanes
    uint32_t accE[BDM_T][kWT], accO[BDM_T][kWT];
#pragma unroll
    for (int j = 0; j < BDM_T; ++j)
#pragma unroll
        for (int k = 0; k < kWT; ++k) accE[j][k] = accO[j][k] = 0;

    // staging registers: kMaxUnits x (16 bytes + the following word), and the chunk's offset table
    uint4 pre[kMaxUnits];
    uint32_t nxt[kMaxUnits];
    uint32_t ptab[2];
    const int units_total = a.chunk_c * a.units_per_row;
    const uint8_t* in_end = a.in + a.in_bytes;

    auto prefetch = [&](int chunk) {
#pragma unroll
        for (int u = 0; u < kMaxUnits; ++u) {
            const int unit = tid + u * kThreads;
            pre[u] = make_uint4(0, 0, 0, 0);
            nxt[u] = 0;
            if (unit < units_total) {
                const int r = unit / a.units_per_row, p = unit - r * a.units_per_row;
                const int l = chunk * a.chunk_c + r;
                const int c = __ldg(a.chan + l);
                const uint8_t* src = a.in + (size_t)c * (size_t)a.in_pitch + (t0 + __ldg(base_b + l)) + p * 16;
                if (a.in_vec) {
                    if (src + 16 <= in_end) pre[u] = __ldg(reinterpret_cast<const uint4*>(src));
                    if (src + 20 <= in_end) nxt[u] = __ldg(reinterpret_cast<const uint32_t*>(src + 16));
                } else {   // unaligned base pointer or row pitch: gather the 20 bytes one by one
                    uint32_t w[5];
#pragma unroll
                    for (int q = 0; q < 5; ++q) {
                        w[q] = 0;
#pragma unroll
                        for (int b = 0; b < 4; ++b)
                            if (src + q * 4 + b < in_end) w[q] |= (uint32_t)__ldg(src + q * 4 + b) << (8 * b);
                    }
                    pre[u] = make_uint4(w[0], w[1], w[2], w[3]);
                    nxt[u] = w[4];
                }
            }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int e = tid + u * kThreads;
            ptab[u] = (e < a.chunk_c * BDM) ? __ldg(off_b + (size_t)chunk * a.chunk_c * BDM + e) : 0u;
        }
    };

    auto commit = [&](int stage) {
        uint8_t* sb = smem + (size_t)stage * stage_bytes;
#pragma unroll
        for (int u = 0; u < kMaxUnits; ++u) {
            const int unit = tid + u * kThreads;
            if (unit < units_total) {
                const int r = unit / a.units_per_row, p = unit - r * a.units_per_row;
                uint8_t* dst = sb + (size_t)(r * 4) * a.row_stride + p * 16;
                const uint32_t w0 = pre[u].x, w1 = pre[u].y, w2 = pre[u].z, w3 = pre[u].w, w4 = nxt[u];
                *reinterpret_cast<uint4*>(dst) = pre[u];
                *reinterpret_cast<uint4*>(dst + a.row_stride) =
                    make_uint4(__byte_perm(w0, w1, 0x4321), __byte_perm(w1, w2, 0x4321),
                               __byte_perm(w2, w3, 0x4321), __byte_perm(w3, w4, 0x4321));
                *reinterpret_cast<uint4*>(dst + 2 * a.row_stride) =
                    make_uint4(__byte_perm(w0, w1, 0x5432), __byte_perm(w1, w2, 0x5432),
                               __byte_perm(w2, w3, 0x5432), __byte_perm(w3, w4, 0x5432));
                *reinterpret_cast<uint4*>(dst + 3 * a.row_stride) =
                    make_uint4(__byte_perm(w0, w1, 0x6543), __byte_perm(w1, w2, 0x6543),
                               __byte_perm(w2, w3, 0x6543), __byte_perm(w3, w4, 0x6543));
            }
        }
        uint32_t* tb = reinterpret_cast<uint32_t*>(sb + stage_rows_bytes);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int e = tid + u * kThreads;
            if (e < a.chunk_c * BDM) tb[e] = ptab[u];
        }
    };

    bool first_flush = true;
    auto flush = [&]() {
#pragma unroll
        for (int j = 0; j < BDM_T; ++j) {
            const int row = __ldg(a.rows + blk * BDM + grp * BDM_T + j);
#pragma unroll
            for (int k = 0; k < kWT; ++k) {
                const int64_t t = t0 + slab * (kWT * 128) + k * 128 + lane * 4;
                const uint32_t e = accE[j][k], o = accO[j][k];
                accE[j][k] = accO[j][k] = 0;
                if (row < 0 || t >= a.nsamp_out) continue;
                uint32_t* p = a.out + (size_t)row * (size_t)a.out_pitch + t;
                uint32_t v0 = e & 0xffffu, v1 = o & 0xffffu, v2 = e >> 16, v3 = o >> 16;
                if (a.out_vec && t + 3 < a.nsamp_out) {
                    if (!first_flush) {
                        const uint4 old = *reinterpret_cast<const uint4*>(p);
                        v0 += old.x; v1 += old.y; v2 += old.z; v3 += old.w;
                    }
                    *reinterpret_cast<uint4*>(p) = make_uint4(v0, v1, v2, v3);
                } else {
                    const uint32_t v[4] = {v0, v1, v2, v3};
#pragma unroll
                    for (int s = 0; s < 4; ++s)
                        if (t + s < a.nsamp_out) p[s] = first_flush ? v[s] : p[s] + v[s];
                }
            }
        }
        first_flush = false;
    };

    // byte offset of this thread's first word inside a phase copy (relative to the row window start)
    const uint32_t lane_off = (uint32_t)(slab * (kWT * 128) + lane * 4);

    prefetch(0);
    commit(0);
    __syncthreads();
    int since_flush = 0;
    for (int chunk = 0; chunk < a.nchunk; ++chunk) {
        const int stage = chunk & 1;
        const bool more = chunk + 1 < a.nchunk;
        if (more) prefetch(chunk + 1);
        const int nrow = min(a.chunk_c, a.nlist - chunk * a.chunk_c);
        if (since_flush + nrow > kFlushEvery) { flush(); since_flush = 0; }
        since_flush += nrow;

        const uint32_t sbase = smem_base + (uint32_t)stage * stage_bytes;
        const uint32_t tbase = sbase + stage_rows_bytes + grp * (BDM_T * 4);
        uint32_t rbase = sbase + lane_off;
#pragma unroll 2
        for (int r = 0; r < nrow; ++r) {
            uint32_t offs[BDM_T];
#pragma unroll
            for (int j = 0; j < BDM_T; j += 4) {
                asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                             : "=r"(offs[j]), "=r"(offs[j + 1]), "=r"(offs[j + 2]), "=r"(offs[j + 3])
                             : "r"(tbase + (uint32_t)(r * BDM * 4 + j * 4)));
            }
#pragma unroll
            for (int j = 0; j < BDM_T; ++j) {
                const uint32_t addr = rbase + offs[j];
#pragma unroll
                for (int k = 0; k < kWT; ++k) {
                    const uint32_t w = lds32(addr + k * 128);
                    accE[j][k] += w & 0x00ff00ffu;
                    accO[j][k] += __byte_perm(w, 0, 0x4341);
                }
            }
            rbase += 4 * a.row_stride;
        }
        if (more) commit(stage ^ 1);
        __syncthreads();
    }
    flush();
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
namespace {

template <typename T>
cudaError_t upload(T** dptr, const std::vector<T>& h) {
    cudaError_t e = cudaMalloc((void**)dptr, std::max<size_t>(h.size(), 1) * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
}

}  // namespace

int ddsp_tiled_plan(ddsp_plan* p) {
    ddsp_tiled& g = p->tiled;
    g.ok = false;
    const int nlist = (int)p->chan_list.size();
    if (p->in_dtype != DDSP_IN_U8 || p->ds != 1 || nlist < 1) return DDSP_OK;   // other paths: direct kernel
    const int smem_budget = (p->smem_optin > 0 ? p->smem_optin : 232448) - 1024;

    // Try the wide DM block first; fall back to the narrow one when the delay spread of a block
    // makes the staged rows too long for shared memory.
    for (int bdm_t : {8, 4}) {
        const int bdm = kGroups * bdm_t;
        const int nblk = (p->ndm + bdm - 1) / bdm;
        // spread of each block/channel and the longest row window
        int64_t max_len = 0;
        for (int b = 0; b < nblk; ++b) {
            const int i0 = p->order[(size_t)b * bdm];
            const int i1 = p->order[std::min<size_t>((size_t)b * bdm + bdm, (size_t)p->ndm) - 1];
            for (int l = 0; l < nlist; ++l) {
                const int c = p->chan_list[l];
                const int64_t lo = p->delays[(size_t)i0 * p->nchan + c] & ~15;
                const int64_t hi = p->delays[(size_t)i1 * p->nchan + c];
                max_len = std::max<int64_t>(max_len, hi - lo);
            }
        }
        // row window: offsets up to max_len, plus T samples, plus 3 bytes of phase shift, in 16-byte units
        const int64_t units = (max_len + kTileT + 3 + 15) / 16 + 1;
        if (units * 16 > 60000) continue;
        const int row_stride = (int)units * 16;
        int chunk_c = std::min(kMaxChunkC, (kMaxUnits * kThreads) / (int)units);
        chunk_c = std::min(chunk_c, (2 * kThreads) / bdm);
        while (chunk_c >= 2 && 2 * (chunk_c * (4 * row_stride + bdm * 4)) > smem_budget) --chunk_c;
        if (chunk_c < 2) continue;
        chunk_c = std::min(chunk_c, std::max(2, nlist));
        g.variant = bdm_t == 8 ? 0 : 1;
        g.bdm = bdm;
        g.tile_t = kTileT;
        g.nblk = nblk;
        g.ntile_t = (p->nsamp_out + kTileT - 1) / kTileT;
        g.chunk_c = chunk_c;
        g.nstage = 2;
        g.row_stride = row_stride;
        g.smem_bytes = 2 * (chunk_c * (4 * row_stride + bdm * 4));
        g.nchunk = (nlist + chunk_c - 1) / chunk_c;
        g.nch_pad = g.nchunk * chunk_c;
        g.ok = true;
        break;
    }
    if (!g.ok) return DDSP_OK;
    if ((int64_t)g.ntile_t * g.nblk > 2147483647LL) { g.ok = false; return DDSP_OK; }

    // tables
    const int bdm = g.bdm;
    std::vector<int32_t> base((size_t)g.nblk * g.nch_pad), rows((size_t)g.nblk * bdm, -1), chan((size_t)g.nch_pad);
    std::vector<uint32_t> off((size_t)g.nblk * g.nch_pad * bdm);
    for (int l = 0; l < g.nch_pad; ++l) chan[l] = p->chan_list[std::min(l, nlist - 1)];
    for (int b = 0; b < g.nblk; ++b) {
        for (int j = 0; j < bdm; ++j) {
            const size_t s = (size_t)b * bdm + j;
            if (s < (size_t)p->ndm) rows[s] = p->order[s];
        }
        const int i0 = p->order[(size_t)b * bdm];
        for (int l = 0; l < g.nch_pad; ++l) {
            const int c = chan[l];
            const int32_t lo = p->delays[(size_t)i0 * p->nchan + c] & ~15;
            base[(size_t)b * g.nch_pad + l] = lo;
            for (int j = 0; j < bdm; ++j) {
                const size_t s = std::min<size_t>((size_t)b * bdm + j, (size_t)p->ndm - 1);
                const int32_t q = p->delays[(size_t)p->order[s] * p->nchan + c] - lo;
                off[((size_t)b * g.nch_pad + l) * bdm + j] = (uint32_t)((q & 3) * g.row_stride + (q >> 2) * 4);
            }
        }
    }
    if (p->device < 0) return DDSP_OK;   // host-only plan: geometry only
    cudaError_t e = upload(&g.d_base, base);
    if (e == cudaSuccess) e = upload(&g.d_off, off);
    if (e == cudaSuccess) e = upload(&g.d_rows, rows);
    if (e == cudaSuccess) e = upload(&g.d_chan, chan);
    if (e == cudaSuccess) {
        // the attribute belongs to the function, not to a plan: always opt in to the device maximum
        e = cudaFuncSetAttribute(ddsp_tiled_u8_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_optin);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(ddsp_tiled_u8_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_optin);
    }
    if (e != cudaSuccess) {
        p->last_cuda = (int)e;
        (void)cudaGetLastError();
        ddsp_tiled_free(p);
        g.ok = false;
        return e == cudaErrorMemoryAllocation ? DDSP_ERR_ALLOC : DDSP_ERR_CUDA;
    }
    return DDSP_OK;
}

void ddsp_tiled_free(ddsp_plan* p) {
    ddsp_tiled& g = p->tiled;
    if (g.d_base) cudaFree(g.d_base);
    if (g.d_off) cudaFree(g.d_off);
    if (g.d_rows) cudaFree(g.d_rows);
    if (g.d_chan) cudaFree(g.d_chan);
    g.d_base = nullptr; g.d_off = nullptr; g.d_rows = nullptr; g.d_chan = nullptr;
}

bool ddsp_tiled_can_run(const ddsp_plan* p, const void* d_in, const void* d_out) {
    // any alignment is correct; 16-byte aligned base and row pitch take the vector staging path
    return p->tiled.ok && d_in != nullptr && d_out != nullptr;
}

cudaError_t ddsp_launch_tiled(const ddsp_plan* p, const void* d_in, void* d_out, cudaStream_t s) {
    const ddsp_tiled& g = p->tiled;
    TiledArgs a;
    a.in = (const uint8_t*)d_in;
    a.out = (uint32_t*)d_out;
    a.base = g.d_base; a.off = g.d_off; a.rows = g.d_rows; a.chan = g.d_chan;
    a.in_pitch = p->in_pitch; a.out_pitch = p->out_pitch; a.nsamp_out = p->nsamp_out;
    a.in_bytes = (int64_t)p->nchan * p->in_pitch;
    a.nlist = (int)p->chan_list.size(); a.nch_pad = g.nch_pad; a.nblk = g.nblk;
    a.chunk_c = g.chunk_c; a.nchunk = g.nchunk; a.row_stride = g.row_stride;
    a.units_per_row = g.row_stride / 16;
    a.out_vec = ((uintptr_t)d_out % 16 == 0) && (p->out_pitch % 4 == 0);
    a.in_vec = ((uintptr_t)d_in % 16 == 0) && (p->in_pitch % 16 == 0);
    const unsigned grid = (unsigned)(g.ntile_t * g.nblk);
    if (g.variant == 0)
        ddsp_tiled_u8_kernel<8><<<grid, kThreads, g.smem_bytes, s>>>(a);
    else
        ddsp_tiled_u8_kernel<4><<<grid, kThreads, g.smem_bytes, s>>>(a);
    return cudaGetLastError();
}
