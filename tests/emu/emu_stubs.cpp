// Stubs for the kernels that the emulation harness does not run (verified on hardware instead): the direct
// and the register-staged tiled kernel.  Test infrastructure only.
#include "ddsp_internal.h"

cudaError_t ddsp_launch_direct(const ddsp_plan*, const void*, void*, cudaStream_t) { return cudaErrorInvalidConfiguration; }
int ddsp_tiled_plan(ddsp_plan* p) { p->tiled.ok = false; return DDSP_OK; }
int ddsp_tiled_set_pitch(ddsp_plan*) { return DDSP_OK; }
void ddsp_tiled_free(ddsp_plan*) {}
bool ddsp_tiled_can_run(const ddsp_plan*, const void*, const void*) { return false; }
cudaError_t ddsp_launch_tiled(const ddsp_plan*, const void*, void*, cudaStream_t) { return cudaErrorInvalidConfiguration; }
