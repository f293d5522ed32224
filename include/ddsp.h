/* ddsp.h -- C ABI of libddsp: brute-force incoherent dedispersion on one B200 (sm_100a).
 *
 * The operation (arxiv 2511.02328, "ASTROFLOW"; line numbers are those of PAPER.md):
 *
 *   f_c      = f_top + c * chan_bw                       channel centres, c = 0..nchan-1; the reference
 *                                                        frequency is the top of the band
 *   tsamp_ds = ds * tsamp,  N_ds = ceil(nsamp / ds)
 *   d(i,c)   = floor(K * DM_i * (f_c^-2 - f_top^-2) / tsamp_ds + 0.5),  K = 4.148808e3 s MHz^2 pc^-1 cm^3
 *                                                        (Eq. 4, Eq. 5), double
 *   x_ds[c][u] = sum_{k<ds} x[c][ds*u + k],  x[c][j] := 0 for j >= nsamp
 *   D[i][t]  = sum over unmasked c (ascending) of x_ds[c][t + d(i,c)]
 *   t = 0 .. nsamp_out-1,  nsamp_out = N_ds - d_max,  d_max = max_{i,c} d(i,c) over ALL channels
 *                                                        ("truncation by the DM delay")
 *
 * uint8 input -> uint32 output (exact); float32 input -> float32 output, one fp32 accumulator per
 * output element, channels added in ascending order, no FMA (bit-identical to a sequential fp32 sum).
 * Readings of the paper where it is silent or garbled: DESIGN.md section 3.
 *
 * Conventions for every entry point
 *   - returns an int status (DDSP_OK = 0) unless stated; nothing throws or aborts across the ABI;
 *   - "host" pointers are ordinary CPU memory, "device" pointers are CUDA device memory on the device
 *     that was current when the plan was created;
 *   - the plan copies dm_list and chan_mask at create; it owns its device tables and frees them in
 *     ddsp_plan_destroy; input/output buffers are always caller-owned;
 *   - ddsp_execute never changes the plan: after create / set_pitch / set_kernel, concurrent ddsp_execute
 *     calls on different streams with different buffers are legal for kernels without a workspace, and
 *     through ddsp_execute_ws (one workspace per concurrent call) for the others;
 *   - ddsp_plan_set_pitch, ddsp_plan_set_kernel and ddsp_execute_host DO change the plan (tables, workspace,
 *     staging buffers): they must not run concurrently with anything else on the same plan.
 */
#ifndef DDSP_H
#define DDSP_H

#include <stdint.h>

#if defined(__GNUC__)
#define DDSP_API __attribute__((visibility("default")))
#else
#define DDSP_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ddsp_plan ddsp_plan; /* opaque */

enum { DDSP_IN_U8 = 0, DDSP_IN_F32 = 1 }; /* output is uint32 for U8, float32 for F32 */

enum {
    DDSP_OK = 0,
    DDSP_ERR_INVALID_ARG = 1, /* bad argument; no side effects */
    DDSP_ERR_NO_OUTPUT = 2,   /* ceil(nsamp/ds) <= d_max: no valid output column */
    DDSP_ERR_UNSUPPORTED = 3, /* e.g. requested kernel cannot run this plan */
    DDSP_ERR_ALLOC = 4,       /* host or device allocation failed */
    DDSP_ERR_CUDA = 5         /* CUDA call failed; see ddsp_last_cuda_error */
};

/* Kernel selection (ddsp_plan_set_kernel).  AUTO picks the fastest kernel that supports the plan. */
enum {
    DDSP_KERNEL_AUTO = 0,
    DDSP_KERNEL_DIRECT = 1, /* one thread per output element, reads global memory directly (any plan) */
    DDSP_KERNEL_TILED = 2,  /* shared-memory tiled kernel, rows staged through registers (uint8, ds = 1) */
    DDSP_KERNEL_LANES = 3   /* segment-interleaved kernels: an interleave pass into a workspace,
                               then a persistent kernel fed by the copy engine; uint8 (ds <= 64) and float32 */
};

/* Create a plan (the delay table is precomputed once, in double).
 *   nchan >= 1; chan_bw_mhz < 0 (channel 0 is the top of the band); f_top + (nchan-1)*chan_bw > 0;
 *   tsamp_s > 0; nsamp >= 1; dm_list: host, ndm >= 1 finite values >= 0, any order (output rows follow
 *   the list order); downsample = ds >= 1; chan_mask: host, nchan bytes, nonzero = zapped channel that
 *   is skipped (never read), or NULL; in_dtype: DDSP_IN_U8 / DDSP_IN_F32.
 * Binds to the current CUDA device.  On failure *plan is set to NULL. */
DDSP_API int ddsp_plan_create(ddsp_plan** plan, int nchan, double f_top_mhz, double chan_bw_mhz, double tsamp_s,
                     int64_t nsamp, const double* dm_list, int ndm, int downsample,
                     const uint8_t* chan_mask, int in_dtype);

/* The same plan for a contiguous RANGE of the DM list: rows [row_begin, row_begin + row_count) of dm_list (ndm_all
 * entries).  d_max, and with it nsamp_out, is taken over the WHOLE list, so the outputs of plans that split one
 * list are row ranges of the output of the plan for the whole list (one observation, DM rows
 * sharded over GPUs, no reduction).  The output has row_count rows; ddsp_plan_get_delays returns them only. */
DDSP_API int ddsp_plan_create_rows(ddsp_plan** plan, int nchan, double f_top_mhz, double chan_bw_mhz, double tsamp_s,
                          int64_t nsamp, const double* dm_list, int ndm_all, int row_begin, int row_count,
                          int downsample, const uint8_t* chan_mask, int in_dtype);

/* Row pitches in ELEMENTS (not bytes).  Defaults: in_pitch = nsamp, out_pitch = nsamp_out.
 * Any pitch >= the row length is correct; the fast path wants 16-byte aligned base pointers and
 * (pitch * element size) % 16 == 0. */
DDSP_API int ddsp_plan_set_pitch(ddsp_plan* plan, int64_t in_pitch_elems, int64_t out_pitch_elems);

/* Force a kernel (tests / profiling).  DDSP_ERR_UNSUPPORTED if it cannot run this plan. */
DDSP_API int ddsp_plan_set_kernel(ddsp_plan* plan, int kernel);

DDSP_API int64_t ddsp_plan_nsamp_out(const ddsp_plan* plan);      /* ceil(nsamp/ds) - d_max; -1 if plan is NULL */
DDSP_API int64_t ddsp_plan_max_delay(const ddsp_plan* plan);      /* d_max on the downsampled grid */
DDSP_API int ddsp_plan_nchan_unmasked(const ddsp_plan* plan);     /* channels that enter the sum */
DDSP_API int ddsp_plan_kernel(const ddsp_plan* plan);             /* the kernel ddsp_execute will launch (resolved AUTO) */
DDSP_API int ddsp_plan_launches_per_execute(const ddsp_plan* plan); /* kernel launches one ddsp_execute enqueues */
/* Bytes of device workspace one execute of the plan's kernel needs (0: none).  The plan owns one workspace of
 * that size (allocated by ddsp_plan_create / ddsp_plan_set_kernel, never by ddsp_execute), which every
 * ddsp_execute of the plan uses; ddsp_execute_ws takes the caller's instead. */
DDSP_API int64_t ddsp_plan_workspace_bytes(const ddsp_plan* plan);
/* Device-side status of the plan's kernels: *status = 0 ok, 1 a bounded barrier wait ran out (the kernel ended
 * early instead of hanging; its output is invalid), 2 a plan table failed the kernel's own bounds check.
 * Copies one word from the device (synchronises with the work in flight). */
DDSP_API int ddsp_plan_device_status(ddsp_plan* plan, int* status);

/* Copy the plan's delay table d(i,c), row-major [ndm][nchan] in dm_list order, to host memory. */
DDSP_API int ddsp_plan_get_delays(const ddsp_plan* plan, int32_t* host_out);

/* Dedisperse.  d_in: device, x[c][t], nchan rows of in_pitch elements (first nsamp
 * valid), never written.  d_out: device, D[i][t], ndm rows (dm_list order) of out_pitch elements; the
 * first nsamp_out elements of every row are overwritten, pitch padding is left untouched.
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).  Asynchronous: enqueues kernels on the
 * stream and returns; never allocates, frees or synchronises.  Launch failures -> DDSP_ERR_CUDA;
 * asynchronous faults surface at the caller's next synchronisation. */
DDSP_API int ddsp_execute(const ddsp_plan* plan, const void* d_in, void* d_out, void* cuda_stream);

/* ddsp_execute with a caller-owned workspace: d_ws = device memory, 16-byte aligned, ws_bytes >=
 * ddsp_plan_workspace_bytes(plan) (d_ws = NULL: the plan's own).  Executes of ONE plan that may overlap in
 * time (different streams) must not share a workspace: give each its own through this call.  Kernels that
 * need no workspace ignore it. */
DDSP_API int ddsp_execute_ws(const ddsp_plan* plan, const void* d_in, void* d_out, void* d_ws, int64_t ws_bytes,
                             void* cuda_stream);

/* Same operation on HOST buffers (pinned memory recommended): copies h_in to a device staging buffer
 * owned by the plan (allocated on the first call after create / set_pitch, freed by set_pitch and destroy),
 * runs ddsp_execute, copies the result to h_out, all on cuda_stream, and synchronises that stream before
 * returning.  h_in: nchan rows of in_pitch elements;
 * h_out: ndm rows of out_pitch elements.  Not re-entrant for one plan (the staging buffers are shared). */
DDSP_API int ddsp_execute_host(ddsp_plan* plan, const void* h_in, void* h_out, void* cuda_stream);

/* ddsp_execute_host with the three phases overlapped (the paper names the copies, not the kernel, as its
 * bottleneck and leaves their overlap undone): the output columns are cut into
 * npieces runs; run j needs input columns < (end_j + d_max) * ds only, so the copy of the input for run j+1, the
 * kernels of run j and the copy of run j-1's result proceed at the same time on three internal streams.  Same
 * buffers, layout and result as ddsp_execute_host; synchronises cuda_stream first and returns when everything
 * is done.  Pinned host memory is needed for real overlap.  DDSP_ERR_UNSUPPORTED unless the plan's kernel is
 * DDSP_KERNEL_LANES (the kernels that can be launched on a run of output columns). */
DDSP_API int ddsp_execute_host_pipelined(ddsp_plan* plan, const void* h_in, void* h_out, void* cuda_stream,
                                         int npieces);

DDSP_API int ddsp_plan_destroy(ddsp_plan* plan); /* NULL is allowed */

DDSP_API const char* ddsp_strerror(int code);
DDSP_API int ddsp_last_cuda_error(const ddsp_plan* plan); /* last cudaError_t seen by this plan (0 = none) */
DDSP_API const char* ddsp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DDSP_H */
