// ddsp_internal.h -- plan object and kernel launchers shared by the translation units of libddsp.
// Product code: nothing under oracle/ is included or linked here.
#pragma once

#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <vector>

#include "../../include/ddsp.h"

// Geometry of the shared-memory tiled kernels for one plan.  Filled by
// ddsp_tiled_plan(); all device tables are owned by the plan.
struct ddsp_tiled {
    bool ok = false;       // the tiled kernel can run this plan
    int variant = 0;       // index into the compiled (B_dm, T) instantiations
    int bdm = 0;           // DM trials per CTA tile
    int threads = 0;       // threads per CTA
    int tile_t = 0;        // output samples per CTA tile (on the downsampled grid)
    int nblk = 0;          // number of DM blocks = ceil(ndm / bdm)
    int64_t ntile_t = 0;   // number of time tiles = ceil(nsamp_out / tile_t)
    int chunk_c = 0;       // channels staged per pipeline stage (a power of two)
    int chunk_shift = 0;   // log2(chunk_c)
    int nstage = 0;        // pipeline depth
    int row_stride = 0;    // bytes of shared memory per staged channel row (one phase copy)
    int smem_bytes = 0;    // dynamic shared memory per CTA
    int nchunk = 0;        // chunks per tile = ceil(nchan_unmasked / chunk_c)
    // device tables
    int64_t* d_meta = nullptr;    // [nblk][nch_pad] row-window byte offset at t0 = 0 (needs in_pitch) | units << 48
    uint32_t* d_off = nullptr;    // [nblk][nch_pad][bdm] shared-memory byte offsets per (channel, trial)
    int32_t* d_rows = nullptr;    // [ndm_pad] output row of each sorted trial (-1 = padding)
    std::vector<int32_t> h_base;  // [nblk][nch_pad] 16-byte-aligned first delay of the block per listed channel
    std::vector<uint16_t> h_nunit; // [nblk][nch_pad] 16-byte units of each row window that are needed
    std::vector<int32_t> h_chan;  // [nch_pad] channel index of each listed channel (padding repeats the last)
#ifdef DDSP_TESTING
    std::vector<uint32_t> h_off;  // host copies of d_off / d_rows for the table tests (include/ddsp_testing.h)
    std::vector<int32_t> h_rows;
#endif
    int nch_pad = 0;              // nchan_unmasked rounded up to chunk_c
};

// Geometry of the lanes kernels (ddsp_lanes.cu) for one plan.
enum { DDSP_LANES_U8 = 0, DDSP_LANES_U16 = 1, DDSP_LANES_F32 = 2 };
struct ddsp_lanes {
    bool ok = false;       // the lanes kernel can run this plan
    int kind = 0;          // DDSP_LANES_U8 (uint8, ds = 1), _U16 (uint8, ds > 1: 16-bit bins), _F32
    int nblk = 0;          // blocks of 16 DM-sorted trials
    int nchunk = 0;        // chunks of 4 listed channels
    int RS = 0;            // bytes of shared memory per staged row window (the longest window of the plan)
    int NS = 0;            // ring stages
    int stage_bytes = 0, smem_bytes = 0;
    int flush_rows = 0;    // channels between flushes of the 16-bit lanes
    size_t ws_bytes = 0;   // workspace (interleaved copy of the unmasked rows) for a full execute
    int2* d_win = nullptr;        // [nblk][nchunk * 4] {first word of the row window relative to the tile, words}
    uint32_t* d_off = nullptr;    // [nblk][nchunk][4 * 16] stage-relative byte offset of every (row, trial)
    int32_t* d_rows = nullptr;    // [nblk * 16] output row of each sorted trial (-1 = padding)
    int* d_status = nullptr;      // device status word (0 = ok) written by the kernels
    uint8_t* d_ws = nullptr;      // the plan's own workspace
    std::vector<int2> h_win;      // host copies (uploaded by ddsp_lanes_prepare; read by the table tests)
    std::vector<uint32_t> h_off;
    std::vector<int32_t> h_rows;
};

struct ddsp_plan {
    // problem
    int nchan = 0, ndm = 0, ds = 1, in_dtype = DDSP_IN_U8;
    double f_top = 0, chan_bw = 0, tsamp = 0;
    int64_t nsamp = 0, nsamp_ds = 0, nsamp_out = 0, dmax = 0;
    int64_t in_pitch = 0, out_pitch = 0;
    std::vector<double> dm;          // copy of dm_list
    std::vector<uint8_t> mask;       // copy of chan_mask (all zero if NULL)
    std::vector<int32_t> delays;     // host, [ndm][nchan], dm_list order
    std::vector<int32_t> chan_list;  // unmasked channels, ascending
    std::vector<int32_t> order;      // trial indices sorted by (DM, index)
    // device
    int device = 0;
    int sm_count = 0;
    int smem_optin = 0;
    int32_t* d_delays = nullptr;     // [ndm][nchan]
    int32_t* d_chan_list = nullptr;  // [nchan_unmasked]
    ddsp_tiled tiled;
    ddsp_lanes lanes;
    int kernel_req = DDSP_KERNEL_AUTO;
    int kernel = DDSP_KERNEL_DIRECT;
    mutable std::atomic<int> last_cuda{0};   // written by concurrent executes
    // staging buffers of ddsp_execute_host
    void* d_stage_in = nullptr;
    void* d_stage_out = nullptr;
    // streams of ddsp_execute_host_pipelined (created on first use)
    cudaStream_t hs_in = nullptr, hs_k = nullptr, hs_out = nullptr;
};

// ddsp_direct.cu
cudaError_t ddsp_launch_direct(const ddsp_plan* p, const void* d_in, void* d_out, cudaStream_t s);

// ddsp_tiled.cu
// Host-side geometry + tables; returns DDSP_OK (with p->tiled.ok possibly false = unsupported) or an error.
int ddsp_tiled_plan(ddsp_plan* p);
int ddsp_tiled_set_pitch(ddsp_plan* p);   // rebuilds the pitch-dependent table
void ddsp_tiled_free(ddsp_plan* p);
// true if this execute call meets the tiled kernel's alignment needs (16-byte base and row pitch)
bool ddsp_tiled_can_run(const ddsp_plan* p, const void* d_in, const void* d_out);
cudaError_t ddsp_launch_tiled(const ddsp_plan* p, const void* d_in, void* d_out, cudaStream_t s);

// ddsp_lanes.cu
int ddsp_lanes_plan(ddsp_plan* p);        // host geometry + tables (p->lanes.ok false = unsupported)
int ddsp_lanes_prepare(ddsp_plan* p);     // device tables, status word, the plan's workspace (idempotent)
void ddsp_lanes_free(ddsp_plan* p);
// segment geometry of a run of nout output columns: tiles, columns per segment, words per interleaved row
void ddsp_lanes_range(const ddsp_plan* p, int64_t nout, int64_t* NT, int64_t* Q, int64_t* M);
// output columns [u_begin, u_begin + nout) (nout < 0: to the end); ws = NULL: the plan's workspace
cudaError_t ddsp_launch_lanes(const ddsp_plan* p, const void* d_in, void* d_out, void* ws, cudaStream_t s,
                              int64_t u_begin = 0, int64_t nout = -1);
