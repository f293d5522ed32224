/* ddsp_testing.h -- introspection of plan-time tables, for the CPU tests only.
 *
 * These entry points exist only in builds made with -DDDSP_TESTING (the CPU emulation library of tests/emu);
 * the product library libddsp.so does not export them.  They let the host logic of SURVEY.md 8(a) A4 (tile
 * geometry) be checked at the FULL size of every BASELINE.json config without a GPU.
 */
#ifndef DDSP_TESTING_H
#define DDSP_TESTING_H

#include "ddsp.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Lanes kernels.  DDSP_ERR_UNSUPPORTED if they cannot run the plan.
 * geom: host int64[16] = {kind (0 uint8, 1 uint8 16-bit bins, 2 float32), lanes per word W, bytes per word WB,
 * trials per block, words per tile TW, rows per chunk C, DM blocks, chunks, row stride RS (bytes), stages NS,
 * stage bytes, shared memory bytes, channels between flushes, tiles NT, columns per segment Q, words per
 * interleaved row M} (the last three for a full execute). */
DDSP_API int ddsp_testing_lanes_geometry(const ddsp_plan* plan, int64_t* geom);
/* win: host int32[blocks * chunks * C * 2] = {first word of the row window relative to the tile, words};
 * off: host uint32[blocks * chunks * C * trials per block] stage-relative byte offset of every (row, trial);
 * rows: host int32[blocks * trials per block] output row of each DM-sorted trial, -1 = padding. */
DDSP_API int ddsp_testing_lanes_tables(const ddsp_plan* plan, int32_t* win, uint32_t* off, int32_t* rows);

/* Tiled kernel (uint8, ds = 1).  geom: host int64[10] = {trials per block, output samples
 * per tile T, DM blocks, time tiles, rows per chunk, stages, row stride (bytes of one phase copy), shared memory
 * bytes, chunks, padded channel count}.
 * base: int32[blocks * padded channels] 16-byte-aligned first delay of the block per listed channel;
 * nunit: int32[same] 16-byte units of the row window that are staged; chan: int32[padded channels] channel of
 * each listed entry (padding repeats the last); off: uint32[blocks * padded channels * trials per block]
 * stage-relative byte offset ((slot * 4 + phase) * row stride + word * 4); rows: int32[blocks * trials per block]. */
DDSP_API int ddsp_testing_tiled_geometry(const ddsp_plan* plan, int64_t* geom);
DDSP_API int ddsp_testing_tiled_tables(const ddsp_plan* plan, int32_t* base, int32_t* nunit, int32_t* chan, uint32_t* off,
                                       int32_t* rows);

#ifdef __cplusplus
}
#endif
#endif /* DDSP_TESTING_H */
