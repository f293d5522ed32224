// ddsp_tiled.cu -- DDSP_KERNEL_TILED: shared-memory tiled brute-force dedispersion, rows staged through registers
// (the round-1 kernel, the one with a hardware history).
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
// uint8 input with ds = 1 only; everything else runs on the lanes kernels (ddsp_lanes.cu) or the direct kernel.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "ddsp_internal.h"
#include "ddsp_dev.cuh"

using namespace ddsp_dev;

namespace {

// ------------------------------------------------------------------------------------------------
// compile-time geometry
// ------------------------------------------------------------------------------------------------
constexpr int kSlabs = 4;               // time slabs of 512 samples; warps = kSlabs x trial groups
constexpr int kWT = 4;                 // 32-bit words per thread per trial (strided by 32 lanes)
constexpr int kTileT = kSlabs * kWT * 128;   // 2048 output samples per CTA (uint8 path)
constexpr int kFlushEvery = 256;       // channels between flushes of the 16-bit lanes
constexpr int kUnitsPerRowMax = 256;   // 16-byte units of a row window that the staging threads can cover

struct TiledArgs {
    const uint8_t* in;
    uint32_t* out;
    const int64_t* meta;      // [nblk][nch_pad] bits 0..47: byte offset of the row window at t0 = 0
                              //                  (c * in_pitch + base); bits 48..63: 16-byte units needed
    const uint32_t* off;      // [nblk][nch_pad][bdm] byte offset inside a stage: (slot*4 + phase)*row_stride + (q>>2)*4
    const int32_t* rows;      // [nblk * bdm] output row of each sorted trial, -1 = padding
    int64_t out_pitch, nsamp_out, in_bytes;
    int nlist, nch_pad, nblk, chunk_shift, nchunk, row_stride, out_vec, in_vec;
};

// ------------------------------------------------------------------------------------------------
// uint8, ds = 1
// ------------------------------------------------------------------------------------------------
// BDM_T trials per thread, GROUPS trial groups (BDM = GROUPS * BDM_T trials per CTA, 128 * GROUPS threads).
// accE accumulates the WHOLE word (mod 2^32), accO the odd bytes (PRMT) in two 16-bit lanes.  At flush
// accE - (accO << 8) = B0 + 2^16 B2 exactly (mod 2^32), so the even bytes never need extracting.
template <int BDM_T, int GROUPS>
__global__ void __launch_bounds__(128 * GROUPS, 1) ddsp_tiled_u8_kernel(const TiledArgs a) {
    constexpr int BDM = GROUPS * BDM_T;
    constexpr int kThreads = 32 * kSlabs * GROUPS;
    constexpr int kThreadsLog2 = GROUPS == 8 ? 10 : 9;
    static_assert(GROUPS == 4 || GROUPS == 8, "4 or 8 trial groups");
    // 16-byte staging units per thread per chunk: chunk_c * kUnitsPerRowMax units over kThreads threads
    constexpr int kMaxUnits = GROUPS == 8 ? 2 : 4;
    extern __shared__ __align__(16) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slab = warp & (kSlabs - 1), grp = warp / kSlabs;
    const int blk = blockIdx.x % a.nblk;
    const int64_t tile = blockIdx.x / a.nblk;
    const int64_t t0 = tile * kTileT;

    const int chunk_c = 1 << a.chunk_shift;
    const int stage_rows_bytes = chunk_c * 4 * a.row_stride;
    const int stage_bytes = stage_rows_bytes + chunk_c * BDM * 4;
    const uint32_t smem_base = smem_addr(smem);

    const int64_t* __restrict__ meta_b = a.meta + (size_t)blk * a.nch_pad;
    const uint32_t* __restrict__ off_b = a.off + (size_t)blk * a.nch_pad * BDM;

    // packed accumulators of each owned word (4 consecutive samples s0..s3):
    //   accE = sum of whole words; accO = (s1, s3) in 16-bit lanes
    uint32_t accE[BDM_T][kWT];
    uint32_t accO[BDM_T][kWT];
#pragma unroll
    for (int k = 0; k < kWT; ++k) {
#pragma unroll
        for (int j = 0; j < BDM_T; ++j) { accE[j][k] = 0; accO[j][k] = 0; }
    }

    // Staging: 512 / chunk_c consecutive threads serve one row slot; a thread owns the 16-byte units
    // p0, p0 + tpr, p0 + 2 tpr, p0 + 3 tpr of that row in every chunk.
    const int tpr_shift = kThreadsLog2 - a.chunk_shift;
    const int srow = tid >> tpr_shift, p0 = tid & ((1 << tpr_shift) - 1), tpr = 1 << tpr_shift;
    uint4 pre[kMaxUnits];
    uint32_t nxt[kMaxUnits];
    uint32_t ptab = 0;
    int64_t meta_cur, meta_nxt;
    uint32_t live = 0;          // bit u: unit u of the chunk being prefetched is needed

    auto load_meta = [&](int chunk) -> int64_t {
        return chunk < a.nchunk ? __ldg(meta_b + (chunk << a.chunk_shift) + srow) : 0;
    };
    auto prefetch = [&](int chunk, int64_t m) {
        const int nunit = (int)(m >> 48);
        const int64_t so = (m & 0xffffffffffffLL) + t0 + p0 * 16;
        const uint8_t* src = a.in + so;
        const int64_t room = a.in_bytes - so;       // bytes that may be read from src on
        live = 0;
#pragma unroll
        for (int u = 0; u < kMaxUnits; ++u) {
            const int p = p0 + u * tpr;
            pre[u] = make_uint4(0, 0, 0, 0);
            nxt[u] = 0;
            if (p < nunit) {
                live |= 1u << u;
                const int64_t d = (int64_t)u * tpr * 16;
                if (a.in_vec) {
                    if (d + 16 <= room) pre[u] = __ldg(reinterpret_cast<const uint4*>(src + d));
                    if (d + 20 <= room) nxt[u] = __ldg(reinterpret_cast<const uint32_t*>(src + d + 16));
                } else {   // unaligned base pointer or row pitch: gather the 20 bytes one by one
                    uint32_t w[5];
#pragma unroll
                    for (int q = 0; q < 5; ++q) {
                        w[q] = 0;
#pragma unroll
                        for (int b = 0; b < 4; ++b)
                            if (d + q * 4 + b < room) w[q] |= (uint32_t)__ldg(src + d + q * 4 + b) << (8 * b);
                    }
                    pre[u] = make_uint4(w[0], w[1], w[2], w[3]);
                    nxt[u] = w[4];
                }
            }
        }
        if (tid < chunk_c * BDM) ptab = __ldg(off_b + (size_t)chunk * chunk_c * BDM + tid);
    };
    // Units that are not needed are not written either: whatever a stage holds there is never read
    // by a stored output.
    auto commit = [&](int stage) {
        uint8_t* sb = smem + (size_t)stage * stage_bytes;
        uint8_t* dst0 = sb + (size_t)(srow * 4) * a.row_stride + p0 * 16;
#pragma unroll
        for (int u = 0; u < kMaxUnits; ++u) {
            if (live & (1u << u)) {
                uint8_t* dst = dst0 + u * tpr * 16;
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
        if (tid < chunk_c * BDM) reinterpret_cast<uint32_t*>(sb + stage_rows_bytes)[tid] = ptab;
    };

    bool first_flush = true;
    auto flush = [&]() {
#pragma unroll 1
        for (int j = 0; j < BDM_T; ++j) {
            const int row = __ldg(a.rows + blk * BDM + grp * BDM_T + j);
#pragma unroll
            for (int k = 0; k < kWT; ++k) {
                const int64_t t = t0 + slab * (kWT * 128) + k * 128 + lane * 4;
                uint32_t e = 0, o = 0;
#pragma unroll
                for (int jj = 0; jj < BDM_T; ++jj)      // static register indexing under a rolled loop
                    if (jj == j) {
                        e = accE[jj][k]; accE[jj][k] = 0;
                        o = accO[jj][k]; accO[jj][k] = 0;
                    }
                if (row < 0 || t >= a.nsamp_out) continue;
                uint32_t* p = a.out + (size_t)row * (size_t)a.out_pitch + t;
                e -= o << 8;     // whole-word sum -> even bytes (exact mod 2^32)
                uint32_t v0 = e & 0xffffu, v2 = e >> 16, v1 = o & 0xffffu, v3 = o >> 16;
                if (a.out_vec && t + 3 < a.nsamp_out) {
                    if (!first_flush) {
                        const uint4 old = ld_global_v4(p);
                        v0 += old.x; v1 += old.y; v2 += old.z; v3 += old.w;
                    }
                    st_global_v4(p, v0, v1, v2, v3);
                } else {
                    const uint32_t v[4] = {v0, v1, v2, v3};
#pragma unroll
                    for (int s = 0; s < 4; ++s)
                        if (t + s < a.nsamp_out) st_global_u32(p + s, first_flush ? v[s] : ld_global_u32(p + s) + v[s]);
                }
            }
        }
        first_flush = false;
    };

    // byte offset of this thread's first word inside a phase copy (relative to the row window start)
    const uint32_t lane_off = (uint32_t)(slab * (kWT * 128) + lane * 4);

    meta_cur = load_meta(0);
    meta_nxt = load_meta(1);
    prefetch(0, meta_cur);
    commit(0);
    __syncthreads();
    int since_flush = 0;
    for (int chunk = 0; chunk < a.nchunk; ++chunk) {
        const int stage = chunk & 1;
        const bool more = chunk + 1 < a.nchunk;
        meta_cur = meta_nxt;                     // arrived during the previous chunk
        meta_nxt = load_meta(chunk + 2);
        if (more) prefetch(chunk + 1, meta_cur);
        const int nrow = min(chunk_c, a.nlist - (chunk << a.chunk_shift));
        if (since_flush + nrow > kFlushEvery) { flush(); since_flush = 0; }
        since_flush += nrow;

        const uint32_t sbase = smem_base + (uint32_t)stage * stage_bytes;
        uint32_t tptr = sbase + stage_rows_bytes + grp * (BDM_T * 4);
        const uint32_t rbase = sbase + lane_off;
        int r = 0;
        for (; r + 2 <= nrow; r += 2) {          // two rows per iteration: their even lanes share one IADD3
            uint32_t o0[BDM_T], o1[BDM_T];
#pragma unroll
            for (int j = 0; j < BDM_T; j += 4) {
                lds128(tptr + (uint32_t)(j * 4), &o0[j]);
                lds128(tptr + (uint32_t)(BDM * 4 + j * 4), &o1[j]);
            }
            tptr += 2 * BDM * 4;
#pragma unroll
            for (int j = 0; j < BDM_T; ++j) {
                const uint32_t a0 = rbase + o0[j], a1 = rbase + o1[j];
#pragma unroll
                for (int k = 0; k < kWT; ++k) {
                    const uint32_t w0 = lds32(a0 + k * 128), w1 = lds32(a1 + k * 128);
                    accE[j][k] = accE[j][k] + w0 + w1;                                              // IADD3
                    accO[j][k] = accO[j][k] + __byte_perm(w0, 0, 0x4341) + __byte_perm(w1, 0, 0x4341);    // 2 PRMT + IADD3
                }
            }
        }
        if (r < nrow) {                          // odd row count
            uint32_t o0[BDM_T];
#pragma unroll
            for (int j = 0; j < BDM_T; j += 4) lds128(tptr + (uint32_t)(j * 4), &o0[j]);
#pragma unroll
            for (int j = 0; j < BDM_T; ++j) {
                const uint32_t a0 = rbase + o0[j];
#pragma unroll
                for (int k = 0; k < kWT; ++k) {
                    const uint32_t w0 = lds32(a0 + k * 128);
                    accE[j][k] += w0;
                    accO[j][k] += __byte_perm(w0, 0, 0x4341);
                }
            }
        }
        if (more) commit(stage ^ 1);
        __syncthreads();
    }
    flush();
}

typedef void (*TiledKernel)(const TiledArgs);
struct Variant { int bdm_t; int groups; TiledKernel fn; };
const Variant kVariants[] = {
    {8, 4, ddsp_tiled_u8_kernel<8, 4>},     // 32 trials, 512 threads
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

}  // namespace

// Geometry of variant v for this plan; false if its staged rows do not fit.
static bool tiled_geometry(const ddsp_plan* p, int v, ddsp_tiled& g) {
    const int nlist = (int)p->chan_list.size();
    const int smem_budget = (p->smem_optin > 0 ? p->smem_optin : 232448) - 1024;
    const int bdm = kVariants[v].groups * kVariants[v].bdm_t;
    const int threads = 128 * kVariants[v].groups;
    const int nblk = (p->ndm + bdm - 1) / bdm;
    // longest row window over all (block, channel): from the 16-byte-aligned first delay to the last
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
    // bytes [0, max_len + T) are read; phase copy 3 of the last unit needs 3 more
    const int64_t units = (max_len + kTileT + 3 + 15) / 16;
    // chunk_c rows per stage, a power of two; the threads of a row slot must cover its units
    for (int shift = 4; shift >= 1; --shift) {
        const int chunk_c = 1 << shift;
        if (units * chunk_c > 8 * kUnitsPerRowMax) continue;
        if (chunk_c * bdm > threads) continue;
        const int row_stride = (int)units * 16;
        const int smem = 2 * (chunk_c * (4 * row_stride + bdm * 4));
        if (smem > smem_budget) continue;
        g.variant = v;
        g.bdm = bdm;
        g.threads = threads;
        g.tile_t = kTileT;
        g.nblk = nblk;
        g.ntile_t = (p->nsamp_out + kTileT - 1) / kTileT;
        g.chunk_c = chunk_c;
        g.chunk_shift = shift;
        g.nstage = 2;
        g.row_stride = row_stride;
        g.smem_bytes = smem;
        g.nchunk = (nlist + chunk_c - 1) / chunk_c;
        g.nch_pad = (g.nchunk + 2) * chunk_c;     // the metadata prefetch looks two chunks ahead
        return (int64_t)g.ntile_t * g.nblk <= 2147483647LL;
    }
    return false;
}

static int tiled_build_tables(ddsp_plan* p) {
    ddsp_tiled& g = p->tiled;
    const int nlist = (int)p->chan_list.size();
    const int bdm = g.bdm;
    std::vector<int32_t> rows((size_t)g.nblk * bdm, -1);
    std::vector<uint32_t> off((size_t)g.nblk * g.nch_pad * bdm);
    g.h_base.assign((size_t)g.nblk * g.nch_pad, 0);
    g.h_nunit.assign((size_t)g.nblk * g.nch_pad, 0);
    g.h_chan.assign((size_t)g.nch_pad, 0);
    for (int l = 0; l < g.nch_pad; ++l) g.h_chan[l] = p->chan_list[std::min(l, nlist - 1)];
    for (int b = 0; b < g.nblk; ++b) {
        for (int j = 0; j < bdm; ++j) {
            const size_t s = (size_t)b * bdm + j;
            if (s < (size_t)p->ndm) rows[s] = p->order[s];
        }
        const int i0 = p->order[(size_t)b * bdm];
        for (int l = 0; l < g.nch_pad; ++l) {
            const int c = g.h_chan[l];
            const int slot = l % g.chunk_c;
            const int32_t lo = p->delays[(size_t)i0 * p->nchan + c] & ~15;
            g.h_base[(size_t)b * g.nch_pad + l] = lo;
            int32_t qmax = 0;
            for (int j = 0; j < bdm; ++j) {
                const size_t s = std::min<size_t>((size_t)b * bdm + j, (size_t)p->ndm - 1);
                const int32_t q = p->delays[(size_t)p->order[s] * p->nchan + c] - lo;
                qmax = std::max(qmax, q);
                off[((size_t)b * g.nch_pad + l) * bdm + j] =
                    (uint32_t)((slot * 4 + (q & 3)) * g.row_stride + (q >> 2) * 4);
            }
            const int need = (qmax + kTileT + 3 + 15) / 16;
            g.h_nunit[(size_t)b * g.nch_pad + l] = (uint16_t)(l < nlist ? std::min(need, g.row_stride / 16) : 0);
        }
    }
#ifdef DDSP_TESTING
    g.h_off = off;
    g.h_rows = rows;
#endif
    if (p->device < 0) return DDSP_OK;   // host-only plan: geometry only
    cudaError_t e = upload(&g.d_off, off);
    if (e == cudaSuccess) e = upload(&g.d_rows, rows);
    if (e == cudaSuccess) e = cudaMalloc((void**)&g.d_meta, g.h_base.size() * sizeof(int64_t));
    // the attribute belongs to the function, not to a plan: always opt in to the device maximum
    for (int v = 0; v < kNumVariants && e == cudaSuccess; ++v)
        e = cudaFuncSetAttribute(kVariants[v].fn, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_optin);
    if (e != cudaSuccess) {
        p->last_cuda = (int)e;
        (void)cudaGetLastError();
        ddsp_tiled_free(p);
        g.ok = false;
        return e == cudaErrorMemoryAllocation ? DDSP_ERR_ALLOC : DDSP_ERR_CUDA;
    }
    return ddsp_tiled_set_pitch(p);
}

int ddsp_tiled_plan(ddsp_plan* p) {
    ddsp_tiled& g = p->tiled;
    g.ok = false;
    const int nlist = (int)p->chan_list.size();
    if (p->in_dtype != DDSP_IN_U8 || p->ds != 1 || nlist < 1) return DDSP_OK;   // other paths: direct kernel
    for (int v = 0; v < kNumVariants && !g.ok; ++v) g.ok = tiled_geometry(p, v, g);
    if (!g.ok) return DDSP_OK;
    return tiled_build_tables(p);
}

// Row-window metadata depends on the input pitch: offset = c * in_pitch + base, packed with the unit count.
int ddsp_tiled_set_pitch(ddsp_plan* p) {
    ddsp_tiled& g = p->tiled;
    if (!g.ok || p->device < 0) return DDSP_OK;
    if ((int64_t)p->nchan * p->in_pitch >= ((int64_t)1 << 47)) { g.ok = false; return DDSP_OK; }
    std::vector<int64_t> meta(g.h_base.size());
    for (int b = 0; b < g.nblk; ++b)
        for (int l = 0; l < g.nch_pad; ++l) {
            const size_t i = (size_t)b * g.nch_pad + l;
            meta[i] = ((int64_t)g.h_chan[l] * p->in_pitch + g.h_base[i]) | ((int64_t)g.h_nunit[i] << 48);
        }
    cudaError_t e = cudaMemcpy(g.d_meta, meta.data(), meta.size() * sizeof(int64_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { p->last_cuda = (int)e; (void)cudaGetLastError(); return DDSP_ERR_CUDA; }
    return DDSP_OK;
}

void ddsp_tiled_free(ddsp_plan* p) {
    ddsp_tiled& g = p->tiled;
    if (g.d_meta) cudaFree(g.d_meta);
    if (g.d_off) cudaFree(g.d_off);
    if (g.d_rows) cudaFree(g.d_rows);
    g.d_meta = nullptr; g.d_off = nullptr; g.d_rows = nullptr;
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
    a.meta = g.d_meta; a.off = g.d_off; a.rows = g.d_rows;
    a.out_pitch = p->out_pitch; a.nsamp_out = p->nsamp_out;
    a.in_bytes = (int64_t)p->nchan * p->in_pitch;
    a.nlist = (int)p->chan_list.size(); a.nch_pad = g.nch_pad; a.nblk = g.nblk;
    a.chunk_shift = g.chunk_shift; a.nchunk = g.nchunk; a.row_stride = g.row_stride;
    a.out_vec = ((uintptr_t)d_out % 16 == 0) && (p->out_pitch % 4 == 0);
    a.in_vec = ((uintptr_t)d_in % 16 == 0) && (p->in_pitch % 16 == 0);
    const unsigned grid = (unsigned)(g.ntile_t * g.nblk);
    kVariants[g.variant].fn<<<grid, g.threads, g.smem_bytes, s>>>(a);
    return cudaGetLastError();
}

#ifdef DDSP_TESTING
// Introspection for the CPU tests (include/ddsp_testing.h); not part of the product library.
#include "../../include/ddsp_testing.h"
#include <cstring>

extern "C" int ddsp_testing_tiled_geometry(const ddsp_plan* p, int64_t* geom) {
    if (!p || !geom) return DDSP_ERR_INVALID_ARG;
    const ddsp_tiled& g = p->tiled;
    if (!g.ok) return DDSP_ERR_UNSUPPORTED;
    const int64_t v[10] = {g.bdm, g.tile_t, g.nblk, g.ntile_t, g.chunk_c, g.nstage, g.row_stride, g.smem_bytes, g.nchunk,
                           g.nch_pad};
    std::memcpy(geom, v, sizeof(v));
    return DDSP_OK;
}

extern "C" int ddsp_testing_tiled_tables(const ddsp_plan* p, int32_t* base, int32_t* nunit, int32_t* chan, uint32_t* off,
                                         int32_t* rows) {
    if (!p || !base || !nunit || !chan || !off || !rows) return DDSP_ERR_INVALID_ARG;
    const ddsp_tiled& g = p->tiled;
    if (!g.ok) return DDSP_ERR_UNSUPPORTED;
    std::memcpy(base, g.h_base.data(), g.h_base.size() * sizeof(int32_t));
    for (size_t i = 0; i < g.h_nunit.size(); ++i) nunit[i] = g.h_nunit[i];
    std::memcpy(chan, g.h_chan.data(), g.h_chan.size() * sizeof(int32_t));
    std::memcpy(off, g.h_off.data(), g.h_off.size() * sizeof(uint32_t));
    std::memcpy(rows, g.h_rows.data(), g.h_rows.size() * sizeof(int32_t));
    return DDSP_OK;
}
#endif  // DDSP_TESTING
