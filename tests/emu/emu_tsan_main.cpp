// Race check of the ring kernels' shared-memory protocol: the emulated kernels run under ThreadSanitizer.
// Every shared-memory access is a plain memory access of some std::thread; the mbarrier stand-ins give
// exactly the happens-before edges of the PTX model (arrive = release, successful wait = acquire, a bulk
// copy is ordered after its issue and before its complete_tx).  A stage that is overwritten while another
// warp may still read it, or read before its copy / expansion is complete, shows up as a data race.
// Usage: emu_tsan <case> ; cases: u8, bins2, bins4, f32.  Test infrastructure only.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "ddsp.h"

extern "C" long ddsp_emu_faults(void);

int main(int argc, char** argv) {
    const std::string which = argc > 1 ? argv[1] : "u8";
    setenv("DDSP_ENABLE_RING", "1", 1);
    int nchan = 120, ds = 1, dtype = DDSP_IN_U8;      // more chunks than ring stages: the ring wraps
    int64_t nsamp = 2200;
    if (which == "bins2") { ds = 2; nsamp = 2 * 2200 + 1; nchan = 60; }
    if (which == "bins4") { ds = 4; nsamp = 4 * 2200 + 3; nchan = 70; }
    if (which == "f32") { dtype = DDSP_IN_F32; nsamp = 1300; nchan = 60; }
    std::vector<double> dm;
    for (int i = 0; i < 36; ++i) dm.push_back(3.0 * i);
    std::vector<uint8_t> mask(nchan, 0);
    mask[3] = 1;
    ddsp_plan* p = nullptr;
    int rc = ddsp_plan_create(&p, nchan, 1400.0, -1.0, 2e-4, nsamp, dm.data(), (int)dm.size(), ds, mask.data(), dtype);
    if (rc) { std::printf("create rc=%d\n", rc); return 2; }
    const int64_t pitch = (nsamp + 15) / 16 * 16, nout = ddsp_plan_nsamp_out(p);
    rc = ddsp_plan_set_pitch(p, pitch, nout);
    if (!rc) rc = ddsp_plan_set_kernel(p, DDSP_KERNEL_RING);
    if (rc) { std::printf("setup rc=%d\n", rc); return 3; }
    const size_t esize = dtype == DDSP_IN_F32 ? 4 : 1;
    void* in = nullptr;
    void* out = nullptr;
    if (posix_memalign(&in, 64, (size_t)nchan * pitch * esize) || posix_memalign(&out, 64, dm.size() * nout * 4)) return 4;
    uint32_t s = 1;
    for (size_t i = 0; i < (size_t)nchan * pitch * esize; ++i) { s = s * 1664525u + 1013904223u; ((uint8_t*)in)[i] = (uint8_t)(s >> 24); }
    if (dtype == DDSP_IN_F32)
        for (size_t i = 0; i < (size_t)nchan * pitch; ++i) ((float*)in)[i] = (float)(((uint8_t*)in)[4 * i]) - 128.0f;
    rc = ddsp_execute(p, in, out, nullptr);
    std::printf("%s: execute rc=%d faults=%ld nsamp_out=%ld\n", which.c_str(), rc, ddsp_emu_faults(), (long)nout);
    ddsp_plan_destroy(p);
    return rc || ddsp_emu_faults() ? 1 : 0;
}
