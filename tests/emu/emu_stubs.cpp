// Stub for the one kernel that the emulation harness does not run: the direct kernel (2-D grid; verified on
// hardware).  Test infrastructure only.
#include "ddsp_internal.h"

cudaError_t ddsp_launch_direct(const ddsp_plan*, const void*, void*, cudaStream_t) { return cudaErrorInvalidConfiguration; }
