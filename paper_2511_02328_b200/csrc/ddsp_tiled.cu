// ddsp_tiled.cu -- DDSP_KERNEL_TILED (placeholder until the tiled kernels land).
#include "ddsp_internal.h"

int ddsp_tiled_plan(ddsp_plan* p) { p->tiled.ok = false; return DDSP_OK; }
void ddsp_tiled_free(ddsp_plan*) {}
cudaError_t ddsp_launch_tiled(const ddsp_plan*, const void*, void*, cudaStream_t) {
    return cudaErrorNotSupported;
}
