// ddsp_lanes.cu -- DDSP_KERNEL_LANES: brute-force dedispersion on a segment-interleaved copy of the input
// (DESIGN.md section 6).
//
//   D[i][t] = sum over unmasked c (ascending) of x_ds[c][t + d(i,c)]
//   x_ds[c][u] = sum_{k<ds} x[c][ds*u + k], zero beyond nsamp
//
// The difficulty of the shifted sum on a GPU is that x[c][t + d] starts on an arbitrary byte while wide
// shared-memory loads need aligned addresses.  Here the alignment problem is removed before the hot loop:
// the output columns [0, nout) are cut into W long SEGMENTS of Q columns, and a first kernel (A5a/A6,
// "interleave") rewrites every unmasked channel row as a row of WORDS
//
//   y[l][m] = ( x_ds[c_l][0*Q + m], x_ds[c_l][1*Q + m], ..., x_ds[c_l][(W-1)*Q + m] )   m = 0 .. Q + d_max
//
// (the fused x ds bin sum is formed here, once per sample).  A delay d moves ALL lanes of a word by d words:
// y[l][m + d] holds the samples that the W outputs t = k*Q + m (k < W) need from channel c_l, so every
// shifted read is one aligned 8- or 16-byte shared-memory load whatever d is.  The lanes of a word are W
// independent stretches of the observation that happen to share a register.
//
// The second kernel (A5b/A7/A8) is persistent (one CTA of 512 threads per SM).  A work item is 16
// DM-consecutive trials x 512 words (x W lanes = 65536 outputs for the integer kinds); for every unmasked
// channel the window y[l][tau*512 + d(first trial) ... + 512 + d(last trial)] is brought into a ring of
// shared-memory stages by the copy engine (cp.async.bulk, completion counted on an mbarrier) and serves the
// 16 trials.  A thread owns 4 trials x 4 words; accumulators stay in registers for the whole channel loop.
//
//   uint8, ds = 1   8 lanes of 8 bits per 64-bit word.  Per 32-bit half w: accE += w (whole word, mod 2^32),
//                   accO += (b1, 0, b3, 0) (PRMT); at flush accE - (accO << 8) = b0-sum + 2^16 b2-sum exactly
//                   (<= 257 channels between flushes).  LDS.64 + 2 PRMT + 2 adds per 8 sample-adds.
//   uint8, ds > 1   8 lanes of 16 bits per 128-bit word (bins <= 255*ds); acc += w; flush every
//                   floor(65535 / (255 ds)) channels.
//   float32         4 lanes per 128-bit word; one fp32 accumulator per output, channels added in ascending
//                   order with __fadd_rn: bit-identical to the sequential sum (R9).
//
// 16-bit lanes are flushed into the uint32 output rows: the first flush of an item stores, later flushes add
// with a reduction store (RED, no return value, nobody waits).  Every output element is owned by one thread.
#include <algorithm>
#include <climits>
#include <type_traits>
#include <vector>

#include "ddsp_internal.h"
#include "ddsp_dev.cuh"

using namespace ddsp_dev;

namespace {

// ------------------------------------------------------------------------------------------------
// compile-time geometry
// ------------------------------------------------------------------------------------------------
// Compile-time tuning knobs (build.py --define NAME=VALUE); the defaults are what ships.  kSlabs * kGroups = 16
// warps always; (slabs, groups) = (4, 4): 16 trials x 512 words per item; (2, 8): 32 trials x 256 words (half the
// passes over the interleaved copy, windows twice as long).
#ifndef DDSP_LANES_SLABS
#define DDSP_LANES_SLABS 4
#endif
#ifndef DDSP_LANES_GROUPS
#define DDSP_LANES_GROUPS 4
#endif
#ifndef DDSP_LANES_ROWS
#define DDSP_LANES_ROWS 4                      // channel rows per chunk (ring stage); even; 6 or 8 trade ring depth for
#endif                                         // fewer barrier rounds per row
#ifndef DDSP_LANES_FMA_E
#define DDSP_LANES_FMA_E 1                     // uint8: whole-word adds as IMAD (FMA pipe); 0: IADD3 (ALU pipe)
#endif
constexpr int kDT = 4;                          // trials per thread
constexpr int kMW = 4;                          // words per thread per trial, strided by 32 lanes
constexpr int kSlabs = DDSP_LANES_SLABS;        // slabs of kMW * 32 = 128 words
constexpr int kGroups = DDSP_LANES_GROUPS;      // trial groups
constexpr int kBDM = kGroups * kDT;             // trials per work item
constexpr int kWarps = kSlabs * kGroups;        // 16
constexpr int kThreads = 32 * kWarps;           // 512
constexpr int kTW = kSlabs * kMW * 32;          // words per work item
static_assert(kWarps == 16, "512 threads x 128 registers = the register file");
constexpr int kC = DDSP_LANES_ROWS;              // channel rows per chunk (one ring stage)
static_assert(kC >= 2 && kC % 2 == 0 && kC <= 16, "rows per chunk: even, producer lanes 0..kC");
constexpr int kTblWords = kC * kBDM;            // per-chunk table: shared-memory offset of every (row, trial)
constexpr int kTblBytes = kTblWords * 4;
constexpr int kBarBytes = 1024;                 // mbarriers and the abort flag live in the first 1 KB
constexpr int kMaxStages = 8;
constexpr int kPreThreads = 256;

enum { kKindU8 = DDSP_LANES_U8, kKindU16 = DDSP_LANES_U16, kKindF32 = DDSP_LANES_F32 };
template <int KIND> struct Kind;
template <> struct Kind<kKindU8>  { static constexpr int W = 8, WB = 8,  NR = 2; };   // NR: 32-bit registers per word
template <> struct Kind<kKindU16> { static constexpr int W = 8, WB = 16, NR = 4; };
template <> struct Kind<kKindF32> { static constexpr int W = 4, WB = 16, NR = 4; };

// status codes written to *status by the kernels
enum { kStatusOk = 0, kStatusTimeout = 1, kStatusTable = 2 };

struct PreArgs {
    const void* in;             // x[c][t], in_pitch elements per row
    uint8_t* y;                 // [nlist][M] words
    const int32_t* chan_list;   // unmasked channels, ascending
    int64_t in_pitch, nsamp, u_begin, Q, M;
    int nlist, ds;
};

struct LanesArgs {
    const uint8_t* y;           // interleaved rows, M words each
    void* out;                  // D[i][t], out_pitch elements per row
    const int2* win;            // [nblk][nchunk * kC]  {first word of the window (relative to the tile), words}
    const uint32_t* off;        // [nblk][nchunk][kC * kBDM]  stage-relative byte offset of (row, trial)
    const int32_t* rows;        // [nblk * kBDM]  output row of each DM-sorted trial, -1 = padding
    int* status;
    int64_t out_pitch, u_begin, nout, Q, M, y_bytes;
    long long wait_budget;
    int nlist, nchunk, nblk, ndm, NT, RS, NS, stage_bytes, flush_rows;
    uint32_t one;               // 1: multiplier that routes an add through the FMA pipe
};

// ------------------------------------------------------------------------------------------------
// A5a / A6: interleave (and bin-sum) the unmasked channel rows
// ------------------------------------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(kPreThreads) ddsp_interleave_kernel(const PreArgs a) {
    using K = Kind<KIND>;
    const int64_t m = (int64_t)blockIdx.x * kPreThreads + threadIdx.x;
    if (m >= a.M) return;
    for (int l = blockIdx.y; l < a.nlist; l += gridDim.y) {
        const int c = __ldg(a.chan_list + l);
        uint32_t w[K::NR];
#pragma unroll
        for (int h = 0; h < K::NR; ++h) w[h] = 0;
        if constexpr (KIND == kKindF32) {
            const float* __restrict__ row = (const float*)a.in + (size_t)c * (size_t)a.in_pitch;
#pragma unroll
            for (int seg = 0; seg < K::W; ++seg) {
                const int64_t j0 = (a.u_begin + (int64_t)seg * a.Q + m) * a.ds;
                float s = j0 < a.nsamp ? ldg_f32(row + j0) : 0.0f;
                for (int k = 1; k < a.ds; ++k) {          // ((x0 + x1) + x2) + ..., missing samples are +0
                    const float v = j0 + k < a.nsamp ? ldg_f32(row + j0 + k) : 0.0f;
                    s = __fadd_rn(s, v);
                }
                w[seg] = __float_as_uint(s);
            }
        } else {
            const uint8_t* __restrict__ row = (const uint8_t*)a.in + (size_t)c * (size_t)a.in_pitch;
#pragma unroll
            for (int seg = 0; seg < K::W; ++seg) {
                const int64_t j0 = (a.u_begin + (int64_t)seg * a.Q + m) * a.ds;
                uint32_t s = 0;
                if constexpr (KIND == kKindU8) {
                    if (j0 < a.nsamp) s = ldg_u8(row + j0);
                    w[seg >> 2] |= s << (8 * (seg & 3));
                } else {
                    for (int k = 0; k < a.ds; ++k)
                        if (j0 + k < a.nsamp) s += ldg_u8(row + j0 + k);
                    w[seg >> 1] |= s << (16 * (seg & 1));
                }
            }
        }
        uint8_t* dst = a.y + ((int64_t)l * a.M + m) * K::WB;
        if constexpr (K::NR == 2) st_global_v2(dst, w[0], w[1]);
        else st_global_v4(dst, w[0], w[1], w[2], w[3]);
    }
}

// ------------------------------------------------------------------------------------------------
// A5b / A7 / A8: staged windows, shifted accumulate, write-out
// ------------------------------------------------------------------------------------------------
// FMA_E (uint8 only): 1 = the whole-word adds are IMADs (FMA pipe), 0 = one IADD3 per row pair (ALU pipe)
template <int KIND, int FMA_E>
__global__ void __launch_bounds__(kThreads, 1) ddsp_lanes_kernel(const LanesArgs a) {
    using K = Kind<KIND>;
    constexpr int kNAcc = KIND == kKindU8 ? 2 : 1;      // accumulator registers per loaded register
    constexpr int kLB = K::NR == 2 ? 4 : 2;             // words per row loaded before their adds are issued
    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slab = warp % kSlabs, grp = warp / kSlabs;
    const uint32_t sbase = smem_addr(smem);
    const uint32_t bar_full = sbase, bar_empty = sbase + 8 * kMaxStages, abort_flag = sbase + 16 * kMaxStages;
    const uint32_t stages = sbase + kBarBytes;

    if (tid == 0) {
        for (int s = 0; s < a.NS; ++s) {
            mbar_init(bar_full + 8 * s, kC + 1);        // kC row copies + the table copy, one arrival each
            mbar_init(bar_empty + 8 * s, kWarps);       // one arrival per consumer warp
        }
        sts32(abort_flag, 0u);
        fence_barrier_init();
    }
    __syncthreads();

    // 32-bit bookkeeping throughout (the plan guarantees nblk * NT * nchunk < 2^31): registers are for accumulators
    const int nitems = a.nblk * a.NT;
    const int first = (int)blockIdx.x, stride = (int)gridDim.x;
    const int n_my = first < nitems ? (nitems - first + stride - 1) / stride : 0;
    const int nchunks_my = n_my * a.nchunk;

    // ---- producer (warp 0): lane r < kC copies row r of a chunk, lane kC copies the chunk's table ----------
    int p_issued = 0, p_item = first;
    int p_k = 0, p_stage = 0;
    uint32_t p_phase = 0;                                // parity of the use of p_stage that is being filled
    auto issue = [&]() {
        const int b = p_item / a.NT;
        const int tau = p_item - b * a.NT;
        const uint32_t st = stages + (uint32_t)p_stage * (uint32_t)a.stage_bytes;
        const uint32_t fb = bar_full + 8 * p_stage;
        if (lane < kC) {
            const int l = p_k * kC + lane;
            bool sent = false;
            if (l < a.nlist) {
                const int2 w = __ldg(a.win + (size_t)b * (size_t)(a.nchunk * kC) + l);
                const int64_t bytes = (int64_t)w.y * K::WB;
                const int64_t so = ((int64_t)l * a.M + (int64_t)tau * kTW + w.x) * K::WB;
                // belt and braces: the plan guarantees all of this; a bad table must not become a bad access
                if (w.y > 0 && bytes <= a.RS && w.x >= 0 && so >= 0 && so + bytes <= a.y_bytes) {
                    mbar_arrive_expect_tx(fb, (uint32_t)bytes);
                    bulk_g2s(st + (uint32_t)(lane * a.RS), a.y + so, (uint32_t)bytes, fb);
                    sent = true;
                } else {
                    report_status(a.status, kStatusTable);
                    sts32(abort_flag, 1u);
                }
            }
            if (!sent) mbar_arrive(fb);
        } else if (lane == kC) {
            const uint32_t* src = a.off + ((size_t)b * (size_t)a.nchunk + (size_t)p_k) * kTblWords;
            mbar_arrive_expect_tx(fb, kTblBytes);
            bulk_g2s(st + (uint32_t)(kC * a.RS), src, kTblBytes, fb);
        }
        ++p_issued;
        if (++p_k == a.nchunk) { p_k = 0; p_item += stride; }
        if (++p_stage == a.NS) { p_stage = 0; p_phase ^= 1u; }
    };
    if (warp == 0)
        while (p_issued < nchunks_my && p_issued < a.NS - 2) issue();      // fresh stages: nothing to wait for

    // ---- accumulators --------------------------------------------------------------------------------------
    uint32_t acc[kDT][kMW][K::NR][kNAcc];
    float accf[KIND == kKindF32 ? kDT : 1][KIND == kKindF32 ? kMW : 1][K::NR];
    const uint32_t lane_off = (uint32_t)((slab * (kMW * 32) + lane) * K::WB);
    const uint32_t one = a.one;

    int c_stage = 0;
    uint32_t c_phase = 0;
    bool aborted = false;
    for (int it = 0; it < n_my && !aborted; ++it) {
        const int item = first + it * stride;
        const int b = item / a.NT;
        const int tau = item - b * a.NT;
#pragma unroll
        for (int j = 0; j < kDT; ++j)
#pragma unroll
            for (int k = 0; k < kMW; ++k)
#pragma unroll
                for (int h = 0; h < K::NR; ++h) {
                    if constexpr (KIND == kKindF32) accf[j][k][h] = 0.0f;
                    else
#pragma unroll
                        for (int e = 0; e < kNAcc; ++e) acc[j][k][h][e] = 0u;
                }

        bool first_flush = true;
        // FIRST: plain stores, else reductions; CHECKED: test every column against the end of the output
        auto flush_body = [&](auto first_tag, auto checked_tag) {
            constexpr bool FIRST = decltype(first_tag)::value, CHECKED = decltype(checked_tag)::value;
            const int64_t m0 = (int64_t)tau * kTW + slab * (kMW * 32) + lane;   // word of this thread, k = 0
            const int64_t lim64 = a.nout - m0;                                  // column offset c is valid iff c < lim
            const uint32_t lim = lim64 <= 0 ? 0u : (lim64 > 0x7fffffffLL ? 0x7fffffffu : (uint32_t)lim64);
            const uint32_t q32 = (uint32_t)a.Q;
            auto emit = [&](char* base, uint32_t col, uint32_t v) {
                if (CHECKED && col >= lim) return;
                uint32_t* p = reinterpret_cast<uint32_t*>(base + (size_t)col * 4u);     // col is warp-uniform
                if (FIRST) st_global_u32(p, v);
                else red_add_u32(p, v);
            };
#pragma unroll
            for (int j = 0; j < kDT; ++j) {
                int row = __ldg(a.rows + b * kBDM + grp * kDT + j);
                if (row >= a.ndm) row = -1;
                char* const base = (char*)a.out + ((int64_t)(row < 0 ? 0 : row) * a.out_pitch + a.u_begin + m0) * 4;
                const bool live = row >= 0 && lim > 0u;
#pragma unroll
                for (int k = 0; k < kMW; ++k) {
#pragma unroll
                    for (int h = 0; h < K::NR; ++h) {
                        if constexpr (KIND == kKindF32) {
                            const uint32_t col = (uint32_t)h * q32 + (uint32_t)(k * 32);
                            if (live && (!CHECKED || col < lim))
                                st_global_f32(reinterpret_cast<float*>(base + (size_t)col * 4u), accf[j][k][h]);
                        } else if constexpr (KIND == kKindU8) {   // (b0, b1, b2, b3) of the half word = segments 4h .. 4h+3
                            const uint32_t o = acc[j][k][h][1];
                            const uint32_t e = acc[j][k][h][0] - (o << 8);      // exact mod 2^32
                            acc[j][k][h][0] = 0u; acc[j][k][h][1] = 0u;
                            if (live) {
                                const uint32_t c0 = (uint32_t)(4 * h) * q32 + (uint32_t)(k * 32);
                                emit(base, c0, e & 0xffffu);
                                emit(base, c0 + q32, o & 0xffffu);
                                emit(base, c0 + 2u * q32, e >> 16);
                                emit(base, c0 + 3u * q32, o >> 16);
                            }
                        } else {                                   // two 16-bit bins = segments 2h, 2h+1
                            const uint32_t sum = acc[j][k][h][0];
                            acc[j][k][h][0] = 0u;
                            if (live) {
                                const uint32_t c0 = (uint32_t)(2 * h) * q32 + (uint32_t)(k * 32);
                                emit(base, c0, sum & 0xffffu);
                                emit(base, c0 + q32, sum >> 16);
                            }
                        }
                    }
                }
            }
        };
        // 16-bit lanes -> uint32 output rows (first flush of the item: store; later: reduction); fp32 accumulators ->
        // output rows, once.  Column offsets are 32-bit (W * Q < 2^31, checked at launch).  The common case -- every
        // column of this thread inside [0, nout) -- runs without a per-element test.
        auto flush = [&]() {
            const int64_t lim64 = a.nout - ((int64_t)tau * kTW + slab * (kMW * 32) + lane);
            const bool all_cols = (int64_t)(K::W - 1) * a.Q + (kMW - 1) * 32 < lim64;
            if (first_flush) {
                if (all_cols) flush_body(std::true_type{}, std::false_type{});
                else flush_body(std::true_type{}, std::true_type{});
            } else {
                if (all_cols) flush_body(std::false_type{}, std::false_type{});
                else flush_body(std::false_type{}, std::true_type{});
            }
            first_flush = false;
        };

        int since_flush = 0;
        for (int k_chunk = 0;; ++k_chunk) {
            const bool last = k_chunk == a.nchunk;
            // producer: refill the stage that every warp left two chunks ago (also while this warp flushes)
            if (!last && warp == 0 && p_issued < nchunks_my) {
                bool ok = true;
                if (p_issued >= a.NS) ok = mbar_wait(bar_empty + 8 * p_stage, p_phase ^ 1u, abort_flag, a.wait_budget);
                if (ok) issue();
                else { aborted = true; break; }
            }
            const int nrow = last ? 0 : min(kC, a.nlist - k_chunk * kC);
            if (last || (KIND != kKindF32 && since_flush + nrow > a.flush_rows)) { flush(); since_flush = 0; }   // the one call site
            if (last) break;
            since_flush += nrow;
            if (!mbar_wait(bar_full + 8 * c_stage, c_phase, abort_flag, a.wait_budget)) { aborted = true; break; }

            const uint32_t st = stages + (uint32_t)c_stage * (uint32_t)a.stage_bytes;
            const uint32_t tptr = st + (uint32_t)(kC * a.RS) + (uint32_t)(grp * (kDT * 4));
            const uint32_t rb = st + lane_off;
            int r = 0;
            for (; r + 2 <= nrow; r += 2) {            // two rows per iteration: they share the 3-input adds
                uint32_t o0[kDT], o1[kDT];
                lds128(tptr + (uint32_t)(r * kBDM * 4), o0);
                lds128(tptr + (uint32_t)((r + 1) * kBDM * 4), o1);
#pragma unroll
                for (int j = 0; j < kDT; ++j) {
                    const uint32_t a0 = rb + o0[j], a1 = rb + o1[j];
                    // loads of a batch of words first (kLB x 2 rows in flight per thread), then their adds: the
                    // shared-memory pipe stays full from 16 warps (Little's law), not from long dependency chains
#pragma unroll
                    for (int kb = 0; kb < kMW; kb += kLB) {
                        uint32_t w0[kLB][K::NR], w1[kLB][K::NR];
#pragma unroll
                        for (int q = 0; q < kLB; ++q) {
                            if constexpr (K::NR == 2) lds64(a0 + (kb + q) * 32 * K::WB, w0[q]);
                            else lds128(a0 + (kb + q) * 32 * K::WB, w0[q]);
                        }
#pragma unroll
                        for (int q = 0; q < kLB; ++q) {
                            if constexpr (K::NR == 2) lds64(a1 + (kb + q) * 32 * K::WB, w1[q]);
                            else lds128(a1 + (kb + q) * 32 * K::WB, w1[q]);
                        }
#pragma unroll
                        for (int q = 0; q < kLB; ++q) {
                            const int k = kb + q;
#pragma unroll
                            for (int h = 0; h < K::NR; ++h) {
                                if constexpr (KIND == kKindU8) {
                                    if constexpr (FMA_E != 0) {
                                        add_fma_pipe(acc[j][k][h][0], w0[q][h], one);
                                        add_fma_pipe(acc[j][k][h][0], w1[q][h], one);
                                    } else {
                                        acc[j][k][h][0] = acc[j][k][h][0] + w0[q][h] + w1[q][h];
                                    }
                                    acc[j][k][h][kNAcc - 1] = acc[j][k][h][kNAcc - 1] + odd_bytes(w0[q][h]) + odd_bytes(w1[q][h]);
                                } else if constexpr (KIND == kKindU16) {
                                    acc[j][k][h][0] = acc[j][k][h][0] + w0[q][h] + w1[q][h];
                                } else {                  // ascending channel order, one rounding per add
                                    accf[j][k][h] = __fadd_rn(__fadd_rn(accf[j][k][h], __uint_as_float(w0[q][h])),
                                                              __uint_as_float(w1[q][h]));
                                }
                            }
                        }
                    }
                }
            }
            if (r < nrow) {                              // odd row count (last chunk only)
                uint32_t o0[kDT];
                lds128(tptr + (uint32_t)(r * kBDM * 4), o0);
#pragma unroll
                for (int j = 0; j < kDT; ++j) {
                    const uint32_t a0 = rb + o0[j];
#pragma unroll
                    for (int k = 0; k < kMW; ++k) {
                        uint32_t w0[K::NR];
                        if constexpr (K::NR == 2) lds64(a0 + k * 32 * K::WB, w0);
                        else lds128(a0 + k * 32 * K::WB, w0);
#pragma unroll
                        for (int h = 0; h < K::NR; ++h) {
                            if constexpr (KIND == kKindU8) {
                                acc[j][k][h][0] += w0[h];
                                acc[j][k][h][kNAcc - 1] += odd_bytes(w0[h]);
                            } else if constexpr (KIND == kKindU16) {
                                acc[j][k][h][0] += w0[h];
                            } else {
                                accf[j][k][h] = __fadd_rn(accf[j][k][h], __uint_as_float(w0[h]));
                            }
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * c_stage);     // this warp is done with the stage
            if (++c_stage == a.NS) { c_stage = 0; c_phase ^= 1u; }
        }
    }
    if (aborted) report_status(a.status, kStatusTimeout);
}

typedef void (*PreKernel)(const PreArgs);
typedef void (*LanesKernel)(const LanesArgs);
const PreKernel kPreKernels[3] = {ddsp_interleave_kernel<kKindU8>, ddsp_interleave_kernel<kKindU16>,
                                  ddsp_interleave_kernel<kKindF32>};
const LanesKernel kLanesKernels[3] = {ddsp_lanes_kernel<kKindU8, DDSP_LANES_FMA_E>, ddsp_lanes_kernel<kKindU16, 0>,
                                      ddsp_lanes_kernel<kKindF32, 0>};
const int kWordBytes[3] = {Kind<kKindU8>::WB, Kind<kKindU16>::WB, Kind<kKindF32>::WB};
const int kLanesPerWord[3] = {Kind<kKindU8>::W, Kind<kKindU16>::W, Kind<kKindF32>::W};

template <typename T>
cudaError_t upload(T** dptr, const std::vector<T>& h) {
    cudaError_t e = cudaMalloc((void**)dptr, std::max<size_t>(h.size(), 1) * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side: A4 tile geometry
// ------------------------------------------------------------------------------------------------
// Segment geometry of a run of `nout` output columns: NT tiles of kTW words, Q = NT * kTW columns per segment,
// M words per interleaved row (the last tile's windows reach Q + d_max).
void ddsp_lanes_range(const ddsp_plan* p, int64_t nout, int64_t* NT, int64_t* Q, int64_t* M) {
    const int W = kLanesPerWord[p->lanes.kind];
    const int64_t qw = (nout + W - 1) / W;
    *NT = std::max<int64_t>(1, (qw + kTW - 1) / kTW);
    *Q = *NT * kTW;
    *M = (*Q + p->dmax + 2 + 1) & ~(int64_t)1;      // even: 8-byte words start every row on 16 bytes
}

int ddsp_lanes_plan(ddsp_plan* p) {
    ddsp_lanes& g = p->lanes;
    g.ok = false;
    const int nlist = (int)p->chan_list.size();
    if (p->in_dtype == DDSP_IN_F32) g.kind = kKindF32;
    else if (p->ds == 1) g.kind = kKindU8;
    else g.kind = kKindU16;
    g.flush_rows = g.kind == kKindU8 ? 256 : g.kind == kKindU16 ? 65535 / (255 * p->ds) : INT_MAX;
    if (g.flush_rows < kC) return DDSP_OK;            // ds > 64: the direct kernel
    const int WB = kWordBytes[g.kind];
    g.nblk = (p->ndm + kBDM - 1) / kBDM;
    g.nchunk = (nlist + kC - 1) / kC;
    const int lpad = g.nchunk * kC;
    if ((int64_t)g.nblk * std::max(lpad, 1) * kBDM > ((int64_t)1 << 31)) return DDSP_OK;

    // windows: per (block, listed channel) the delays of the block's trials span [lo, hi]
    g.h_win.assign((size_t)g.nblk * lpad, int2{0, 0});
    g.h_rows.assign((size_t)g.nblk * kBDM, -1);
    int64_t max_words = kTW;
    for (int b = 0; b < g.nblk; ++b) {
        for (int j = 0; j < kBDM; ++j) {
            const size_t s = (size_t)b * kBDM + j;
            if (s < (size_t)p->ndm) g.h_rows[s] = p->order[s];
        }
        for (int l = 0; l < nlist; ++l) {
            const int c = p->chan_list[l];
            int32_t lo = INT_MAX, hi = 0;
            for (int j = 0; j < kBDM; ++j) {
                const size_t s = std::min<size_t>((size_t)b * kBDM + j, (size_t)p->ndm - 1);
                const int32_t d = p->delays[(size_t)p->order[s] * p->nchan + c];
                lo = std::min(lo, d); hi = std::max(hi, d);
            }
            if (WB == 8) lo &= ~1;                       // 16-byte aligned source of the bulk copy
            int64_t words = (int64_t)kTW + (hi - lo);
            if (WB == 8) words = (words + 1) & ~(int64_t)1;
            if (words * WB > ((int64_t)1 << 20)) return DDSP_OK;      // absurd spread: the direct kernel
            g.h_win[(size_t)b * lpad + l] = int2{lo, (int)words};
            max_words = std::max(max_words, words);
        }
    }
    g.RS = (int)(max_words * WB);
    g.stage_bytes = kC * g.RS + kTblBytes;
    const int budget = (p->smem_optin > 0 ? p->smem_optin : 232448) - kBarBytes;
    g.NS = std::min(kMaxStages, budget / g.stage_bytes);
    if (g.NS < 3) return DDSP_OK;                      // windows too long for a ring: the direct kernel
    g.smem_bytes = kBarBytes + g.NS * g.stage_bytes;

    g.h_off.assign((size_t)g.nblk * std::max(g.nchunk, 1) * kTblWords, 0u);
    for (int b = 0; b < g.nblk; ++b)
        for (int l = 0; l < nlist; ++l) {
            const int c = p->chan_list[l];
            const int32_t lo = g.h_win[(size_t)b * lpad + l].x;
            for (int j = 0; j < kBDM; ++j) {
                const size_t s = std::min<size_t>((size_t)b * kBDM + j, (size_t)p->ndm - 1);
                const int32_t d = p->delays[(size_t)p->order[s] * p->nchan + c];
                g.h_off[((size_t)b * g.nchunk + l / kC) * kTblWords + (l % kC) * kBDM + j] =
                    (uint32_t)((l % kC) * g.RS + (d - lo) * WB);
            }
        }
    int64_t NT, Q, M;
    ddsp_lanes_range(p, p->nsamp_out, &NT, &Q, &M);
    if ((int64_t)g.nblk * NT * std::max(g.nchunk, 1) >= ((int64_t)1 << 31)) return DDSP_OK;   // 32-bit chunk counters
    if (Q * kLanesPerWord[g.kind] >= ((int64_t)1 << 31)) return DDSP_OK;                       // 32-bit column offsets
    g.ws_bytes = (size_t)std::max(nlist, 1) * (size_t)M * WB;
    g.ok = true;
    return DDSP_OK;
}

// Device tables, the status word and (unless the caller brings its own) the workspace.  Called when the lanes
// kernel becomes the plan's kernel -- never from ddsp_execute.
int ddsp_lanes_prepare(ddsp_plan* p) {
    ddsp_lanes& g = p->lanes;
    if (!g.ok || p->device < 0) return DDSP_OK;
    cudaError_t e = cudaSuccess;
    if (!g.d_win) {
        e = upload(&g.d_win, g.h_win);
        if (e == cudaSuccess) e = upload(&g.d_off, g.h_off);
        if (e == cudaSuccess) e = upload(&g.d_rows, g.h_rows);
        if (e == cudaSuccess) e = cudaMalloc((void**)&g.d_status, sizeof(int));
        if (e == cudaSuccess) e = cudaMemset(g.d_status, 0, sizeof(int));
        for (int k = 0; k < 3 && e == cudaSuccess; ++k)
            e = cudaFuncSetAttribute(kLanesKernels[k], cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_optin);
    }
    if (e == cudaSuccess && !g.d_ws) e = cudaMalloc((void**)&g.d_ws, g.ws_bytes);
    if (e != cudaSuccess) {
        p->last_cuda = (int)e;
        (void)cudaGetLastError();
        ddsp_lanes_free(p);
        return e == cudaErrorMemoryAllocation ? DDSP_ERR_ALLOC : DDSP_ERR_CUDA;
    }
    return DDSP_OK;
}

void ddsp_lanes_free(ddsp_plan* p) {
    ddsp_lanes& g = p->lanes;
    if (g.d_win) cudaFree(g.d_win);
    if (g.d_off) cudaFree(g.d_off);
    if (g.d_rows) cudaFree(g.d_rows);
    if (g.d_status) cudaFree(g.d_status);
    if (g.d_ws) cudaFree(g.d_ws);
    g.d_win = nullptr; g.d_off = nullptr; g.d_rows = nullptr; g.d_status = nullptr; g.d_ws = nullptr;
}

// Output columns [u_begin, u_begin + nout) of every trial (nout < 0: all from u_begin on).  `ws` = workspace of
// at least lanes.ws_bytes (NULL: the plan's own).
cudaError_t ddsp_launch_lanes(const ddsp_plan* p, const void* d_in, void* d_out, void* ws, cudaStream_t s,
                              int64_t u_begin, int64_t nout) {
    const ddsp_lanes& g = p->lanes;
    if (nout < 0) nout = p->nsamp_out - u_begin;
    if (!g.ok || !g.d_win || u_begin < 0 || nout < 1 || u_begin + nout > p->nsamp_out) return cudaErrorInvalidValue;
    uint8_t* y = ws ? (uint8_t*)ws : g.d_ws;
    if (!y) return cudaErrorInvalidValue;
    const int nlist = (int)p->chan_list.size();
    const int WB = kWordBytes[g.kind];
    int64_t NT, Q, M;
    ddsp_lanes_range(p, nout, &NT, &Q, &M);

    if (nlist > 0) {
        PreArgs pa;
        pa.in = d_in; pa.y = y; pa.chan_list = p->d_chan_list;
        pa.in_pitch = p->in_pitch; pa.nsamp = p->nsamp; pa.u_begin = u_begin; pa.Q = Q; pa.M = M;
        pa.nlist = nlist; pa.ds = p->ds;
        const int64_t gx = (M + kPreThreads - 1) / kPreThreads;
        if (gx > 2147483647LL) return cudaErrorInvalidConfiguration;
        const dim3 pgrid((unsigned)gx, (unsigned)std::min(nlist, 65535));
        kPreKernels[g.kind]<<<pgrid, kPreThreads, 0, s>>>(pa);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    LanesArgs a;
    a.y = y; a.out = d_out; a.win = g.d_win; a.off = g.d_off; a.rows = g.d_rows; a.status = g.d_status;
    a.out_pitch = p->out_pitch; a.u_begin = u_begin; a.nout = nout; a.Q = Q; a.M = M;
    a.y_bytes = (int64_t)std::max(nlist, 1) * M * WB;
    a.wait_budget = 4000000000LL;                        // ~2 s of SM clocks
    a.nlist = nlist; a.nchunk = g.nchunk; a.nblk = g.nblk; a.ndm = p->ndm; a.NT = (int)NT; a.RS = g.RS; a.NS = g.NS;
    a.stage_bytes = g.stage_bytes; a.flush_rows = g.flush_rows; a.one = 1u;
    const int64_t nitems = (int64_t)g.nblk * NT;
    if (nitems * std::max(g.nchunk, 1) >= ((int64_t)1 << 31)) return cudaErrorInvalidConfiguration;
    if (Q * kLanesPerWord[g.kind] >= ((int64_t)1 << 31)) return cudaErrorInvalidConfiguration;      // 32-bit column offsets
    const unsigned grid = (unsigned)std::min<int64_t>(nitems, p->sm_count > 0 ? p->sm_count : 148);
    kLanesKernels[g.kind]<<<grid, kThreads, g.smem_bytes, s>>>(a);
    return cudaGetLastError();
}

#ifdef DDSP_TESTING
// Introspection for the CPU tests (include/ddsp_testing.h); not part of the product library.
#include "../../include/ddsp_testing.h"
#include <cstring>

extern "C" int ddsp_testing_lanes_geometry(const ddsp_plan* p, int64_t* geom) {
    if (!p || !geom) return DDSP_ERR_INVALID_ARG;
    const ddsp_lanes& g = p->lanes;
    if (!g.ok) return DDSP_ERR_UNSUPPORTED;
    int64_t NT, Q, M;
    ddsp_lanes_range(p, p->nsamp_out, &NT, &Q, &M);
    const int64_t v[16] = {g.kind, kLanesPerWord[g.kind], kWordBytes[g.kind], kBDM, kTW, kC, g.nblk, g.nchunk, g.RS,
                           g.NS, g.stage_bytes, g.smem_bytes, g.flush_rows, NT, Q, M};
    std::memcpy(geom, v, sizeof(v));
    return DDSP_OK;
}

extern "C" int ddsp_testing_lanes_tables(const ddsp_plan* p, int32_t* win, uint32_t* off, int32_t* rows) {
    if (!p || !win || !off || !rows) return DDSP_ERR_INVALID_ARG;
    const ddsp_lanes& g = p->lanes;
    if (!g.ok) return DDSP_ERR_UNSUPPORTED;
    for (size_t i = 0; i < g.h_win.size(); ++i) { win[2 * i] = g.h_win[i].x; win[2 * i + 1] = g.h_win[i].y; }
    std::memcpy(off, g.h_off.data(), g.h_off.size() * sizeof(uint32_t));
    std::memcpy(rows, g.h_rows.data(), g.h_rows.size() * sizeof(int32_t));
    return DDSP_OK;
}
#endif  // DDSP_TESTING
