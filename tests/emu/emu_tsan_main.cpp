// Race check of the lanes kernels' shared-memory protocol: the emulated kernels run under ThreadSanitizer.
// Every shared-memory access is a plain memory access of some std::thread; the mbarrier stand-ins give
// exactly the happens-before edges of the PTX model (arrive = release, successful wait = acquire, a bulk
// copy is ordered after its issue and before its complete_tx).  A stage that is overwritten while another
// warp may still read it, or read before its copy is complete, shows up as a data race.
// Usage: emu_tsan <case> ; cases: u8, bins2, bins4, f32.  Test infrastructure only.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "ddsp.h"

extern "C" long ddsp_emu_faults(void);
extern "C" void ddsp_emu_register(const void* p, size_t n);

int main(int argc, char** argv) {
    const std::string which = argc > 1 ? argv[1] : "u8";
    int nchan = 90, ds = 1, dtype = DDSP_IN_U8;       // 23 chunks of 4 rows: the ring of <= 8 stages wraps
    int64_t nsamp = 1100;
    if (which == "bins2") { ds = 2; nsamp = 2 * 1100 + 1; nchan = 70; }
    if (which == "bins4") { ds = 4; nsamp = 4 * 1100 + 3; nchan = 70; }
    if (which == "f32") { dtype = DDSP_IN_F32; nsamp = 900; nchan = 60; }
    std::vector<double> dm;
    for (int i = 0; i < 36; ++i) dm.push_back(3.0 * i);     // 3 DM blocks, the last one ragged
    std::vector<uint8_t> mask(nchan, 0);
    mask[3] = 1;
    ddsp_plan* p = nullptr;
    int rc = ddsp_plan_create(&p, nchan, 1400.0, -1.0, 2e-4, nsamp, dm.data(), (int)dm.size(), ds, mask.data(), dtype);
    if (rc) { std::printf("create rc=%d\n", rc); return 2; }
    const int64_t pitch = nsamp + 5, nout = ddsp_plan_nsamp_out(p);
    rc = ddsp_plan_set_pitch(p, pitch, nout);
    if (!rc) rc = ddsp_plan_set_kernel(p, DDSP_KERNEL_LANES);
    if (rc) { std::printf("setup rc=%d\n", rc); return 3; }
    const size_t esize = dtype == DDSP_IN_F32 ? 4 : 1;
    const size_t in_bytes = (size_t)nchan * pitch * esize, out_bytes = dm.size() * nout * 4;
    void* in = nullptr;
    void* out = nullptr;
    if (posix_memalign(&in, 64, in_bytes) || posix_memalign(&out, 64, out_bytes)) return 4;
    ddsp_emu_register(in, in_bytes);
    ddsp_emu_register(out, out_bytes);
    uint32_t s = 1;
    for (size_t i = 0; i < in_bytes; ++i) { s = s * 1664525u + 1013904223u; ((uint8_t*)in)[i] = (uint8_t)(s >> 24); }
    if (dtype == DDSP_IN_F32)
        for (size_t i = 0; i < (size_t)nchan * pitch; ++i) ((float*)in)[i] = (float)(((uint8_t*)in)[4 * i]) - 128.0f;
    rc = ddsp_execute(p, in, out, nullptr);
    int status = -1;
    ddsp_plan_device_status(p, &status);
    std::printf("%s: execute rc=%d status=%d faults=%ld nsamp_out=%ld\n", which.c_str(), rc, status, ddsp_emu_faults(), (long)nout);
    ddsp_plan_destroy(p);
    return rc || status || ddsp_emu_faults() ? 1 : 0;
}
