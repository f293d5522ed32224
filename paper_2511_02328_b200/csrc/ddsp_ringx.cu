// ddsp_ringx.cu -- the ring kernel (ddsp_ring.cu) for the other two input kinds:
//
//   float32, ds = 1   D[i][t] = sum over unmasked c, ascending, of x[c][t + d(i,c)], one fp32 accumulator per
//                     output element, __fadd_rn in channel order: bit-identical to the sequential sum
//                     (R9).  One staged copy per row (4-byte samples are
//                     always aligned), 32 trials x 1024 samples per CTA, LDS.32 + FADD per add.
//   uint8, ds > 1     x_ds[c][u] = sum_{k<ds} x[c][ds*u + k], zero beyond nsamp,
//                     formed ONCE per staged row, shared memory to shared memory, as 16-bit bins in two
//                     phase copies (bins[i], bins[i+1]); the hot loop adds words of two bins into 2 x 16-bit
//                     lane accumulators (two rows per IADD3) and flushes them every floor(65535 / (255 ds))
//                     channels.  32 trials x 2048 samples per CTA.
//
// Both use the same pipeline as ddsp_ring.cu: rows arrive by cp.async.bulk on `raw` mbarriers, all
// warps mark progress on split-phase `built` mbarriers, warp 0 issues the copies two chunks ahead.
// Both are selected only for DDSP_KERNEL_RING and are opt-in (DDSP_ENABLE_RING) until they have run on
// hardware.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "ddsp_internal.h"
#include "ddsp_ring_common.cuh"

namespace {

using namespace ddsp_dev;

constexpr int kBdm = 32;            // trials per CTA tile
constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int kBarBytes = 1024;
constexpr int kMaxStages = 12;
constexpr int kTileF = 1024;        // float32: output samples per tile
constexpr int kTileB = 2048;        // uint8 bins: output samples per tile

struct RingXArgs {
    const uint8_t* in;        // bytes (uint8 or float32 samples)
    void* out;
    const int64_t* meta;      // [nblk][nch_pad] bits 0..47: byte offset of the row window at t0 = 0; bits 48..: 16-byte units
    const uint32_t* tbl;      // [nblk][nchunk][tblw]
    const int32_t* rows;      // [nblk * 32]
    int64_t out_pitch, nsamp_out, in_valid, nsamp;
    int64_t tile0;            // first time tile of this launch
    int nlist, nch_pad, nblk, nchunk, raw_stride, bins_stride, raw_slot_bytes, bins_slot_bytes, nraw, nbins;
    int tblw, ds, flush_every, out_vec;
};

// Issue the bulk copies of one chunk (warp 0, all lanes; lane r < C owns row r).  scale: bytes of input per
// unit of t0 (ds for uint8, 4 for float32).
template <int C>
__device__ __forceinline__ void issue_chunk(const RingXArgs& a, uint8_t* smem, int lane, int64_t meta_pref, int64_t t0_bytes,
                                            int slot, uint32_t slot_base, uint32_t bar, const uint32_t* tbl_chunk) {
    const int64_t so = (meta_pref & 0xffffffffffffLL) + t0_bytes;
    const uint32_t bytes = (uint32_t)(meta_pref >> 48) * 16u;
    uint32_t cp = bytes;
    const int64_t room = a.in_valid - so;
    if ((int64_t)bytes > room) {        // the window runs past the end of the input buffer
        cp = room > 0 ? (uint32_t)(room & ~(int64_t)15) : 0u;
        const int tail = room > 0 ? (int)(room - cp) : 0;
        for (int i = 0; i < tail; ++i)
            smem[kBarBytes + (size_t)slot * a.raw_slot_bytes + (size_t)lane * a.raw_stride + cp + i] = a.in[so + cp + i];
        fence_proxy_async_smem();
    }
    uint32_t total = cp;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);
    __syncwarp();
    if (lane == 0) mbar_arrive_expect_tx(bar, total + (uint32_t)a.tblw * 4u);
    __syncwarp();
    if (cp) bulk_g2s(slot_base + (uint32_t)lane * (uint32_t)a.raw_stride, a.in + so, cp, bar);
    if (lane == 0) bulk_g2s(slot_base + (uint32_t)(C * a.raw_stride), tbl_chunk, (uint32_t)a.tblw * 4u, bar);
}

// ------------------------------------------------------------------------------------------------
// float32, ds = 1
// ------------------------------------------------------------------------------------------------
// Thread = BDM_T trials x KWT samples (strided by 32 lanes); tile = 32 trials x (16 / GROUPS) * KWT * 32 samples.
// Stage = C raw rows + the chunk's table (C x 32 byte offsets (slot * raw_stride + 4 q), then C unit counts).
template <int BDM_T, int KWT, int C>
__global__ void __launch_bounds__(kThreads, 1) ddsp_ringf_kernel(const RingXArgs a) {
    constexpr int GROUPS = kBdm / BDM_T;
    constexpr int SLABS = kWarps / GROUPS;
    static_assert(SLABS * KWT * 32 == kTileF, "tile length");
    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slab = warp % SLABS, grp = warp / SLABS;
    const int blk = blockIdx.x % a.nblk;
    const int64_t t0 = ((int64_t)(blockIdx.x / a.nblk) + a.tile0) * kTileF;
    const int NS = a.nraw;
    const uint32_t smem_base = smem_addr(smem);
    const uint32_t rows_bytes = (uint32_t)(C * a.raw_stride);

    auto bar_raw = [&](int s) { return smem_base + (uint32_t)s * 8u; };
    auto bar_built = [&](int s) { return smem_base + 512u + (uint32_t)s * 8u; };
    auto stage_base = [&](int s) { return smem_base + (uint32_t)kBarBytes + (uint32_t)s * (uint32_t)a.raw_slot_bytes; };

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(bar_raw(s), 1);
            mbar_init(bar_built(s), kWarps);
        }
        fence_barrier_init();
    }
    __syncthreads();

    float acc[BDM_T][KWT];
#pragma unroll
    for (int j = 0; j < BDM_T; ++j)
#pragma unroll
        for (int k = 0; k < KWT; ++k) acc[j][k] = 0.0f;

    const int64_t* __restrict__ meta_b = a.meta + (size_t)blk * a.nch_pad;
    const uint32_t* __restrict__ tbl_b = a.tbl + (size_t)blk * a.nchunk * a.tblw;
    int64_t meta_pref = 0;
    auto load_meta = [&](int chunk) {
        meta_pref = (lane < C && chunk < a.nchunk) ? __ldg(meta_b + chunk * C + lane) : 0;
    };
    auto issue = [&](int chunk) {
        const int s = chunk % NS;
        issue_chunk<C>(a, smem, lane, meta_pref, t0 * 4, s, stage_base(s), bar_raw(s), tbl_b + (size_t)chunk * a.tblw);
    };

    const uint32_t lane_off = (uint32_t)((slab * (KWT * 32) + lane) * 4);
    auto hot = [&](int chunk) {
        const uint32_t sb = stage_base(chunk % NS);
        const int nrow = min(C, a.nlist - chunk * C);
        uint32_t tptr = sb + rows_bytes + (uint32_t)(grp * (BDM_T * 4));
        const uint32_t rbase = sb + lane_off;
#pragma unroll 1
        for (int r = 0; r < nrow; ++r) {         // channels strictly in ascending order (R9)
            uint32_t o[BDM_T];
#pragma unroll
            for (int j = 0; j < BDM_T; j += 4) lds128(tptr + (uint32_t)(j * 4), &o[j]);
            tptr += kBdm * 4;
#pragma unroll
            for (int j = 0; j < BDM_T; ++j) {
                const uint32_t a0 = rbase + o[j];
#pragma unroll
                for (int k = 0; k < KWT; ++k)
                    acc[j][k] = __fadd_rn(acc[j][k], __uint_as_float(lds32(a0 + k * 128)));
            }
        }
    };

    const int ahead = NS - 2;
    if (warp == 0) {
        for (int c = 0; c < ahead && c < a.nchunk; ++c) { load_meta(c); issue(c); }
        load_meta(ahead);
    }
    if (lane == 0) mbar_arrive(bar_built(0));
    for (int chunk = 0; chunk < a.nchunk; ++chunk) {
        // built[k] complete <=> every warp is past its hot loop of chunk k-2: that stage is free
        mbar_wait(bar_built(chunk % NS), (uint32_t)(chunk / NS) & 1u);
        if (warp == 0) {
            if (chunk + ahead < a.nchunk) issue(chunk + ahead);
            load_meta(chunk + ahead + 1);
        }
        __syncwarp();
        if (lane == 0 && chunk + 1 < a.nchunk) mbar_arrive(bar_built((chunk + 1) % NS));
        mbar_wait(bar_raw(chunk % NS), (uint32_t)(chunk / NS) & 1u);
        hot(chunk);
    }

    float* out = reinterpret_cast<float*>(a.out);
#pragma unroll 1
    for (int j = 0; j < BDM_T; ++j) {
        const int row = __ldg(a.rows + blk * kBdm + grp * BDM_T + j);
#pragma unroll
        for (int k = 0; k < KWT; ++k) {
            float v = 0.0f;
#pragma unroll
            for (int jj = 0; jj < BDM_T; ++jj)
                if (jj == j) v = acc[jj][k];
            const int64_t t = t0 + slab * (KWT * 32) + k * 32 + lane;
            if (row >= 0 && t < a.nsamp_out) out[(size_t)row * (size_t)a.out_pitch + t] = v;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// uint8, ds > 1: 16-bit bins
// ------------------------------------------------------------------------------------------------
// Shared memory: [mbarriers][nraw raw slots: C raw rows + table][nbins bin slots: C rows x 2 phase copies of
// 16-bit bins + the chunk's C x 32 offsets].  A raw slot is free again as soon as its chunk is binned, a
// bin slot when every warp is past the hot loop of its chunk.
// Table of a chunk: C x 32 byte offsets ((slot * 2 + (q & 1)) * bins_stride + (q >> 1) * 4), C counts of 8-bin
// units to form, C raw byte indices (within the channel row) of the window start at tile 0.
// DS: compile-time downsample factor of the fast binning paths (2, 4), 0 = any factor (byte loop)
template <int BDM_T, int KWT, int C, int DS>
__global__ void __launch_bounds__(kThreads, 1) ddsp_ringb_kernel(const RingXArgs a) {
    constexpr int GROUPS = kBdm / BDM_T;
    constexpr int SLABS = kWarps / GROUPS;
    static_assert(SLABS * KWT * 64 == kTileB, "tile length");
    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slab = warp % SLABS, grp = warp / SLABS;
    const int blk = blockIdx.x % a.nblk;
    const int64_t t0 = ((int64_t)(blockIdx.x / a.nblk) + a.tile0) * kTileB;
    const int NR = a.nraw, NB = a.nbins, ds = DS ? DS : a.ds;
    const int Sr = a.raw_stride, Sb = a.bins_stride;
    const uint32_t smem_base = smem_addr(smem);
    const uint32_t raw_rows_bytes = (uint32_t)(C * Sr), bin_rows_bytes = (uint32_t)(C * 2 * Sb);

    auto bar_raw = [&](int s) { return smem_base + (uint32_t)s * 8u; };
    auto bar_built = [&](int s) { return smem_base + 512u + (uint32_t)s * 8u; };
    auto raw_base = [&](int s) { return smem_base + (uint32_t)kBarBytes + (uint32_t)s * (uint32_t)a.raw_slot_bytes; };
    auto bin_base = [&](int s) {
        return smem_base + (uint32_t)kBarBytes + (uint32_t)NR * (uint32_t)a.raw_slot_bytes + (uint32_t)s * (uint32_t)a.bins_slot_bytes;
    };

    if (tid == 0) {
        for (int s = 0; s < NR; ++s) mbar_init(bar_raw(s), 1);
        for (int s = 0; s < NB; ++s) mbar_init(bar_built(s), kWarps);
        fence_barrier_init();
    }
    __syncthreads();

    uint32_t acc[BDM_T][KWT];      // two 16-bit lanes: samples (2i, 2i+1) of the owned word
#pragma unroll
    for (int j = 0; j < BDM_T; ++j)
#pragma unroll
        for (int k = 0; k < KWT; ++k) acc[j][k] = 0;

    const int64_t* __restrict__ meta_b = a.meta + (size_t)blk * a.nch_pad;
    const uint32_t* __restrict__ tbl_b = a.tbl + (size_t)blk * a.nchunk * a.tblw;
    int64_t meta_pref = 0;
    auto load_meta = [&](int chunk) {
        meta_pref = (lane < C && chunk < a.nchunk) ? __ldg(meta_b + chunk * C + lane) : 0;
    };
    auto issue = [&](int chunk) {
        const int s = chunk % NR;
        issue_chunk<C>(a, smem, lane, meta_pref, t0 * ds, s, raw_base(s), bar_raw(s), tbl_b + (size_t)chunk * a.tblw);
    };

    // ---- bin the raw rows of a chunk: 8 bins (+1 for the shifted copy) per unit, units spread over all threads ----
    auto build = [&](int chunk) {
        const uint32_t rs = raw_base(chunk % NR), bs = bin_base(chunk % NB);
        mbar_wait(bar_raw(chunk % NR), (uint32_t)(chunk / NR) & 1u);
        const uint32_t tb = rs + raw_rows_bytes;
        // row r of the chunk is binned by threads [r * TPR, (r + 1) * TPR) (whole warps per row); the partial
        // last pass alternates between the group's first and last warps so that no warp is always the slow one
        constexpr uint32_t TPR = kThreads / C;
        const uint32_t r = (uint32_t)tid / TPR;
        const uint32_t n = lds32(tb + (uint32_t)((C * kBdm) * 4) + r * 4u);
        const uint32_t j0 = lds32(tb + (uint32_t)((C * kBdm + C) * 4) + r * 4u);
        // the offsets of the chunk move to the bin slot: the raw slot is refilled before the hot loop runs
        if (tid < C * kBdm) {
            const uint32_t v = lds32(tb + (uint32_t)tid * 4u);
            sts32(bs + bin_rows_bytes + (uint32_t)tid * 4u, v);
        }
        uint32_t u = (uint32_t)tid % TPR;
        if (chunk & 1) u = TPR - 1u - u;
        for (; u < n; u += TPR) {
            const uint32_t rb = rs + r * (uint32_t)Sr + u * (uint32_t)(8 * ds);
            // raw bytes of this row at window index >= limit lie beyond nsamp: they count as zero
            const int64_t limit = a.nsamp - ((int64_t)j0 + t0 * ds) - (int64_t)u * (8 * ds);
            uint32_t b[9];
            if (DS == 4 && limit >= 36) {
                uint32_t w[9];
                lds128(rb, &w[0]);
                lds128(rb + 16, &w[4]);
                w[8] = lds32(rb + 32);
#pragma unroll
                for (int i = 0; i < 9; ++i) b[i] = __dp4a(w[i], 0x01010101u, 0u);
            } else if (DS == 2 && limit >= 18) {
                uint32_t w[5];
                lds128(rb, &w[0]);
                w[4] = lds32(rb + 16);
#pragma unroll
                for (int i = 0; i < 5; ++i) {
                    const uint32_t e = (w[i] & 0x00ff00ffu) + ((w[i] >> 8) & 0x00ff00ffu);   // (B0+B1) | (B2+B3) << 16
                    b[2 * i] = e & 0xffffu;
                    if (2 * i + 1 < 9) b[2 * i + 1] = e >> 16;
                }
            } else {
#pragma unroll 1
                for (int i = 0; i < 9; ++i) {
                    uint32_t sum = 0;
                    for (int k = 0; k < ds; ++k) {
                        const int idx = i * ds + k;
                        if (idx < limit) sum += lds8(rb + (uint32_t)idx);
                    }
#pragma unroll
                    for (int ii = 0; ii < 9; ++ii)
                        if (ii == i) b[ii] = sum;
                }
            }
            const uint32_t d0 = bs + (r * 2u) * (uint32_t)Sb + u * 16u;
            sts128(d0, __byte_perm(b[0], b[1], 0x5410), __byte_perm(b[2], b[3], 0x5410),
                   __byte_perm(b[4], b[5], 0x5410), __byte_perm(b[6], b[7], 0x5410));
            sts128(d0 + (uint32_t)Sb, __byte_perm(b[1], b[2], 0x5410), __byte_perm(b[3], b[4], 0x5410),
                   __byte_perm(b[5], b[6], 0x5410), __byte_perm(b[7], b[8], 0x5410));
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_built(chunk % NB));
    };

    bool first_flush = true;
    auto flush = [&]() {
        uint32_t* out = reinterpret_cast<uint32_t*>(a.out);
#pragma unroll 1
        for (int j = 0; j < BDM_T; ++j) {
            const int row = __ldg(a.rows + blk * kBdm + grp * BDM_T + j);
#pragma unroll
            for (int k = 0; k < KWT; ++k) {
                const int64_t t = t0 + slab * (KWT * 64) + k * 64 + lane * 2;
                uint32_t v = 0;
#pragma unroll
                for (int jj = 0; jj < BDM_T; ++jj)
                    if (jj == j) { v = acc[jj][k]; acc[jj][k] = 0; }
                if (row < 0 || t >= a.nsamp_out) continue;
                uint32_t* p = out + (size_t)row * (size_t)a.out_pitch + t;
                uint32_t v0 = v & 0xffffu, v1 = v >> 16;
                if (a.out_vec && t + 1 < a.nsamp_out) {
                    if (!first_flush) {
                        const uint2 old = *reinterpret_cast<const uint2*>(p);
                        v0 += old.x; v1 += old.y;
                    }
                    *reinterpret_cast<uint2*>(p) = make_uint2(v0, v1);
                } else {
                    p[0] = first_flush ? v0 : p[0] + v0;
                    if (t + 1 < a.nsamp_out) p[1] = first_flush ? v1 : p[1] + v1;
                }
            }
        }
        first_flush = false;
    };

    const uint32_t lane_off = (uint32_t)(slab * (KWT * 128) + lane * 4);
    auto hot = [&](int chunk) {
        const uint32_t sb = bin_base(chunk % NB);
        const int nrow = min(C, a.nlist - chunk * C);
        uint32_t tptr = sb + bin_rows_bytes + (uint32_t)(grp * (BDM_T * 4));
        const uint32_t rbase = sb + lane_off;
        int r = 0;
#pragma unroll 1
        for (; r + 2 <= nrow; r += 2) {
            uint32_t o0[BDM_T], o1[BDM_T];
#pragma unroll
            for (int j = 0; j < BDM_T; j += 4) {
                lds128(tptr + (uint32_t)(j * 4), &o0[j]);
                lds128(tptr + (uint32_t)(kBdm * 4 + j * 4), &o1[j]);
            }
            tptr += 2 * kBdm * 4;
#pragma unroll
            for (int j = 0; j < BDM_T; ++j) {
                const uint32_t a0 = rbase + o0[j], a1 = rbase + o1[j];
#pragma unroll
                for (int k = 0; k < KWT; ++k) acc[j][k] = acc[j][k] + lds32(a0 + k * 128) + lds32(a1 + k * 128);
            }
        }
        if (r < nrow) {
            uint32_t o0[BDM_T];
#pragma unroll
            for (int j = 0; j < BDM_T; j += 4) lds128(tptr + (uint32_t)(j * 4), &o0[j]);
#pragma unroll
            for (int j = 0; j < BDM_T; ++j) {
                const uint32_t a0 = rbase + o0[j];
#pragma unroll
                for (int k = 0; k < KWT; ++k) acc[j][k] += lds32(a0 + k * 128);
            }
        }
    };

    const int ahead = NR;                        // chunk k + NR is issued in iteration k (its raw slot was binned)
    if (warp == 0) {
        for (int c = 0; c < ahead && c < a.nchunk; ++c) { load_meta(c); issue(c); }
        load_meta(ahead);
    }
    build(0);
    int since_flush = 0;
    for (int chunk = 0; chunk < a.nchunk; ++chunk) {
        mbar_wait(bar_built(chunk % NB), (uint32_t)(chunk / NB) & 1u);
        if (warp == 0) {
            if (chunk + ahead < a.nchunk) issue(chunk + ahead);
            load_meta(chunk + ahead + 1);
        }
        if (chunk + 1 < a.nchunk) build(chunk + 1);
        const int nrow = min(C, a.nlist - chunk * C);
        if (since_flush + nrow > a.flush_every) { flush(); since_flush = 0; }
        since_flush += nrow;
        hot(chunk);
    }
    flush();
}

typedef void (*RingXKernel)(const RingXArgs);
struct VariantX { int kind, c, ds; RingXKernel fn; };
const VariantX kVariants[] = {
    {2, 4, 1, ddsp_ringf_kernel<8, 8, 4>},
    {1, 4, 4, ddsp_ringb_kernel<8, 8, 4, 4>},
    {1, 4, 2, ddsp_ringb_kernel<8, 8, 4, 2>},
    {1, 4, 0, ddsp_ringb_kernel<8, 8, 4, 0>},
    {1, 2, 4, ddsp_ringb_kernel<8, 8, 2, 4>},
    {1, 2, 2, ddsp_ringb_kernel<8, 8, 2, 2>},
    {1, 2, 0, ddsp_ringb_kernel<8, 8, 2, 0>},
};
constexpr int kNumVariants = sizeof(kVariants) / sizeof(kVariants[0]);

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

int gcd_int(int a, int b) { return b ? gcd_int(b, a % b) : a; }
int align_up(int v, int a) { return (v + a - 1) / a * a; }

// Window start (in samples of the delay grid) of channel c in block b: the first delay of the block moved
// down so that the byte address of the window start is a multiple of 16.
//   float32: (c * pitch + lo) * 4 % 16 == 0 for any pitch (lo may be negative for c > 0: previous row);
//   uint8 bins: pitch % 16 == 0 is required, lo is a multiple of 16 / gcd(ds, 16).
int64_t window_lo(const ddsp_plan* p, int kind, int b, int c) {
    const int i0 = p->order[(size_t)b * kBdm];
    const int64_t d0 = p->delays[(size_t)i0 * p->nchan + c];
    if (kind == 2) return d0 - ((int64_t)c * p->in_pitch + d0) % 4;
    const int g = 16 / gcd_int(p->ds, 16);
    return d0 - d0 % g;
}

// largest in-window offset q over all (block, channel) of the plan, for the worst window alignment
int64_t max_offset(const ddsp_plan* p, int slack) {
    const int nlist = (int)p->chan_list.size();
    const int nblk = (p->ndm + kBdm - 1) / kBdm;
    int64_t max_q = 0;
    for (int b = 0; b < nblk; ++b) {
        const int i0 = p->order[(size_t)b * kBdm];
        const int i1 = p->order[std::min<size_t>((size_t)b * kBdm + kBdm, (size_t)p->ndm) - 1];
        for (int l = 0; l < nlist; ++l) {
            const int c = p->chan_list[l];
            max_q = std::max<int64_t>(max_q, (int64_t)p->delays[(size_t)i1 * p->nchan + c] -
                                                 p->delays[(size_t)i0 * p->nchan + c] + slack);
        }
    }
    return max_q;
}

bool ringx_geometry(const ddsp_plan* p, int v, ddsp_ringx& g) {
    const VariantX& var = kVariants[v];
    const int nlist = (int)p->chan_list.size();
    const int budget = (p->smem_optin > 0 ? p->smem_optin : 232448) - kBarBytes;
    const int C = var.c;
    g.kind = var.kind;
    g.variant = v;
    g.c_rows = C;
    g.nblk = (p->ndm + kBdm - 1) / kBdm;
    g.nchunk = (nlist + C - 1) / C;
    g.nch_pad = g.nchunk * C;
    if (var.kind == 2) {
        g.tile_t = kTileF;
        const int64_t units = (max_offset(p, 3) + kTileF + 3) / 4;
        if (units > 8000) return false;
        g.raw_stride = (int)units * 16;
        g.bins_stride = 0;
        g.tblw = C * kBdm + 4;
        g.raw_slot_bytes = align_up(C * g.raw_stride + g.tblw * 4, 128);
        g.bins_slot_bytes = 0;
        g.nbins = 0;
        g.nraw = std::min(kMaxStages, budget / g.raw_slot_bytes);
        if (g.nraw < 4) return false;
        g.flush_every = 0;
        g.smem_bytes = kBarBytes + g.nraw * g.raw_slot_bytes;
    } else {
        g.tile_t = kTileB;
        const int align = 16 / gcd_int(p->ds, 16);
        const int64_t nb = (max_offset(p, align - 1) + kTileB + 7) / 8;      // 8-bin units
        if (nb * 8 * p->ds > 60000) return false;
        g.raw_stride = align_up((int)(8 * nb + 1) * p->ds, 16);
        g.bins_stride = (int)nb * 16;
        g.tblw = align_up(C * kBdm + 2 * C, 4);
        g.raw_slot_bytes = align_up(C * g.raw_stride + g.tblw * 4, 128);
        g.bins_slot_bytes = align_up(C * 2 * g.bins_stride + C * kBdm * 4, 128);
        g.nraw = 2;
        g.nbins = std::min(kMaxStages, (budget - g.nraw * g.raw_slot_bytes) / g.bins_slot_bytes);
        if (g.nbins < 3) return false;
        g.flush_every = std::min(256, 65535 / (255 * p->ds));
        if (g.flush_every < 2 * C) return false;
        g.smem_bytes = kBarBytes + g.nraw * g.raw_slot_bytes + g.nbins * g.bins_slot_bytes;
    }
    g.ntile_t = (p->nsamp_out + g.tile_t - 1) / g.tile_t;
    return (int64_t)g.ntile_t * g.nblk <= 2147483647LL;
}

}  // namespace

int ddsp_ringx_set_pitch(ddsp_plan* p) {
    ddsp_ringx& g = p->ringx;
    if (!g.kind) return DDSP_OK;
    const int nlist = (int)p->chan_list.size();
    const int C = g.c_rows, T = g.tile_t;
    const int64_t esize = g.kind == 2 ? 4 : 1;
    g.ok = false;
    if (g.kind == 1 && p->in_pitch % 16 != 0) return DDSP_OK;        // bins need 16-byte aligned rows
    if ((int64_t)p->nchan * p->in_pitch * esize >= ((int64_t)1 << 47)) return DDSP_OK;
    std::vector<int64_t> meta((size_t)g.nblk * g.nch_pad, 0);
    std::vector<uint32_t> tbl((size_t)g.nblk * g.nchunk * g.tblw, 0);
    for (int b = 0; b < g.nblk; ++b)
        for (int l = 0; l < nlist; ++l) {
            const int c = p->chan_list[l];
            const int chunk = l / C, slot = l % C;
            const int64_t lo = window_lo(p, g.kind, b, c);
            uint32_t* t = &tbl[((size_t)b * g.nchunk + chunk) * g.tblw];
            int64_t qmax = 0;
            for (int j = 0; j < kBdm; ++j) {
                const size_t s = std::min<size_t>((size_t)b * kBdm + j, (size_t)p->ndm - 1);
                const int64_t q = p->delays[(size_t)p->order[s] * p->nchan + c] - lo;
                qmax = std::max(qmax, q);
                t[slot * kBdm + j] = g.kind == 2 ? (uint32_t)(slot * g.raw_stride + q * 4)
                                                 : (uint32_t)((slot * 2 + (q & 1)) * g.bins_stride + (q >> 1) * 4);
            }
            if (g.kind == 2) {
                const int64_t units = (qmax + T + 3) / 4;
                if (units * 16 > g.raw_stride) return DDSP_OK;           // cannot happen (geometry)
                t[C * kBdm + slot] = (uint32_t)units;
                meta[(size_t)b * g.nch_pad + l] = (((int64_t)c * p->in_pitch + lo) * 4) | (units << 48);
            } else {
                const int64_t nb = (qmax + T + 7) / 8;
                if (nb * 16 > g.bins_stride) return DDSP_OK;             // cannot happen (geometry)
                const int64_t raw16 = (8 * nb * p->ds + 15) / 16;
                t[C * kBdm + slot] = (uint32_t)nb;
                t[C * kBdm + C + slot] = (uint32_t)(p->ds * lo);
                meta[(size_t)b * g.nch_pad + l] = ((int64_t)c * p->in_pitch + p->ds * lo) | (raw16 << 48);
            }
        }
    g.h_meta = meta;
    g.h_tbl = tbl;
    g.ok = true;
    if (p->device < 0) return DDSP_OK;
    cudaError_t e = cudaSuccess;
    if (!g.d_meta) e = cudaMalloc((void**)&g.d_meta, meta.size() * sizeof(int64_t));
    if (e == cudaSuccess && !g.d_tbl) e = cudaMalloc((void**)&g.d_tbl, tbl.size() * sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMemcpy(g.d_meta, meta.data(), meta.size() * sizeof(int64_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(g.d_tbl, tbl.data(), tbl.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { g.ok = false; p->last_cuda = (int)e; (void)cudaGetLastError(); return DDSP_ERR_CUDA; }
    return DDSP_OK;
}

int ddsp_ringx_plan(ddsp_plan* p) {
    ddsp_ringx& g = p->ringx;
    g.ok = false;
    g.kind = 0;
    const int nlist = (int)p->chan_list.size();
    if (nlist < 1) return DDSP_OK;
    int kind = 0;
    if (p->in_dtype == DDSP_IN_F32 && p->ds == 1) kind = 2;
    if (p->in_dtype == DDSP_IN_U8 && p->ds > 1 && p->ds <= 32) kind = 1;
    if (!kind) return DDSP_OK;
    const char* en = getenv("DDSP_ENABLE_RING");      // opt-in until run on hardware (see ddsp_ring.cu)
    if (!en || atoi(en) == 0) return DDSP_OK;
    bool found = false;
    for (int v = 0; v < kNumVariants && !found; ++v) {
        if (kVariants[v].kind != kind) continue;
        if (kind == 1 && kVariants[v].ds != ((p->ds == 2 || p->ds == 4) ? p->ds : 0)) continue;
        found = ringx_geometry(p, v, g);
    }
    if (!found) { g.kind = 0; return DDSP_OK; }
    std::vector<int32_t> rows((size_t)g.nblk * kBdm, -1);
    for (size_t s = 0; s < (size_t)p->ndm; ++s) rows[s] = p->order[s];
    g.h_rows = rows;
    if (p->device >= 0) {
        cudaError_t e = upload(&g.d_rows, rows);
        for (int v = 0; v < kNumVariants && e == cudaSuccess; ++v)
            e = cudaFuncSetAttribute(kVariants[v].fn, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_optin);
        if (e != cudaSuccess) {
            p->last_cuda = (int)e;
            (void)cudaGetLastError();
            ddsp_ringx_free(p);
            g.kind = 0;
            return e == cudaErrorMemoryAllocation ? DDSP_ERR_ALLOC : DDSP_ERR_CUDA;
        }
    }
    return ddsp_ringx_set_pitch(p);
}

void ddsp_ringx_free(ddsp_plan* p) {
    ddsp_ringx& g = p->ringx;
    if (g.d_meta) cudaFree(g.d_meta);
    if (g.d_tbl) cudaFree(g.d_tbl);
    if (g.d_rows) cudaFree(g.d_rows);
    g.d_meta = nullptr; g.d_tbl = nullptr; g.d_rows = nullptr;
}

bool ddsp_ringx_can_run(const ddsp_plan* p, const void* d_in, const void* d_out) {
    return p->ringx.ok && d_in != nullptr && d_out != nullptr && ((uintptr_t)d_in % 16 == 0);
}

cudaError_t ddsp_launch_ringx(const ddsp_plan* p, const void* d_in, void* d_out, cudaStream_t s, int64_t tile0,
                              int64_t ntile) {
    const ddsp_ringx& g = p->ringx;
    const int64_t esize = g.kind == 2 ? 4 : 1;
    RingXArgs a;
    a.in = (const uint8_t*)d_in;
    a.out = d_out;
    a.meta = g.d_meta; a.tbl = g.d_tbl; a.rows = g.d_rows;
    a.out_pitch = p->out_pitch; a.nsamp_out = p->nsamp_out; a.nsamp = p->nsamp;
    a.in_valid = ((int64_t)(p->nchan - 1) * p->in_pitch + p->nsamp) * esize;
    a.nlist = (int)p->chan_list.size(); a.nch_pad = g.nch_pad; a.nblk = g.nblk; a.nchunk = g.nchunk;
    a.raw_stride = g.raw_stride; a.bins_stride = g.bins_stride;
    a.raw_slot_bytes = g.raw_slot_bytes; a.bins_slot_bytes = g.bins_slot_bytes; a.nraw = g.nraw; a.nbins = g.nbins;
    a.tblw = g.tblw; a.ds = p->ds; a.flush_every = g.flush_every;
    a.out_vec = ((uintptr_t)d_out % 8 == 0) && (p->out_pitch % 2 == 0);
    if (ntile < 0) ntile = g.ntile_t - tile0;
    if (tile0 < 0 || ntile < 1 || tile0 + ntile > g.ntile_t) return cudaErrorInvalidConfiguration;
    a.tile0 = tile0;
    const unsigned grid = (unsigned)(ntile * g.nblk);
    kVariants[g.variant].fn<<<grid, kThreads, g.smem_bytes, s>>>(a);
    return cudaGetLastError();
}

// Introspection for the CPU tests of the plan-time geometry (tests/test_ring_tables_cpu.py).
extern "C" {

int ddsp_plan_ringx_geometry(const ddsp_plan* p, int32_t* geom) {
    if (!p || !geom) return DDSP_ERR_INVALID_ARG;
    const ddsp_ringx& g = p->ringx;
    if (!g.ok) return DDSP_ERR_UNSUPPORTED;
    const int32_t v[14] = {g.kind, g.c_rows, g.nblk, g.nchunk, g.nch_pad, g.raw_stride, g.bins_stride, g.tblw,
                           g.nraw, g.nbins, g.smem_bytes, g.tile_t, g.flush_every, g.raw_slot_bytes};
    for (int i = 0; i < 14; ++i) geom[i] = v[i];
    return DDSP_OK;
}

int ddsp_plan_ringx_tables(const ddsp_plan* p, int64_t* meta, uint32_t* tbl, int32_t* rows) {
    if (!p || !meta || !tbl || !rows) return DDSP_ERR_INVALID_ARG;
    const ddsp_ringx& g = p->ringx;
    if (!g.ok) return DDSP_ERR_UNSUPPORTED;
    std::copy(g.h_meta.begin(), g.h_meta.end(), meta);
    std::copy(g.h_tbl.begin(), g.h_tbl.end(), tbl);
    std::copy(g.h_rows.begin(), g.h_rows.end(), rows);
    return DDSP_OK;
}

}  // extern "C"
