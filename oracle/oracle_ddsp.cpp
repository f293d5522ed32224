// oracle_ddsp.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded CPU statement of brute-force incoherent
// dedispersion, written from the paper (arxiv 2511.02328, PAPER.md) and the
// readings listed in DESIGN.md.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
// code with the CUDA path (paper_2511_02328_b200/csrc) and neither includes
// the other.
//
// What it computes (the plain definition; the method reaches exactly this):
//
//   f_c      = f_top + c * chan_bw                                (reference = top of band)
//   d(i,c)   = floor( ((K*DM_i) * (1/(f_c*f_c) - 1/(f_top*f_top))) / tsamp_ds + 0.5 )
//                                                                  (Eq. 4; Eq. 5)
//   tsamp_ds = ds * tsamp
//   N_ds     = ceil(nsamp / ds)
//   x_ds[c][u] = sum_{k<ds} x[c][ds*u + k],  x[c][j] := 0 for j >= nsamp   ("zero outside bounds")
//   D[i][t]  = sum over unmasked c, ascending, of x_ds[c][t + d(i,c)]
//
// K = 4.148808e3 with f in MHz and tsamp in seconds (PAPER.md:97 prints "ms";
// DESIGN.md reading R1).  All of it is three nested loops: for i / for c / for t.
//
// Parity status: pinned (tests/test_oracle_pins.py): exact-rational delay
// values, hand-checked golden example, invariants I1-I12, per-output gather
// brute force.  Nothing here is "parity unpinned".
//
// Build: g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/oracle.py).

#include <cmath>
#include <cstdint>
#include <cstddef>

namespace {

const double K_DM = 4.148808e3;  // s MHz^2 pc^-1 cm^3   (R1)

// x_ds[c][u] for uint8 input, computed from the definition (no materialised copy).
inline uint32_t bin_u8(const uint8_t* row, int64_t nsamp, int ds, int64_t u) {
    uint32_t s = 0;
    for (int k = 0; k < ds; ++k) {
        int64_t j = (int64_t)ds * u + k;
        if (j < nsamp) s += row[j];
    }
    return s;
}

// x_ds[c][u] for float32 input: ((x0 + x1) + x2) + ... in fp32, zero beyond nsamp.
inline float bin_f32(const float* row, int64_t nsamp, int ds, int64_t u) {
    int64_t j0 = (int64_t)ds * u;
    float s = (j0 < nsamp) ? row[j0] : 0.0f;
    for (int k = 1; k < ds; ++k) {
        int64_t j = j0 + k;
        float v = (j < nsamp) ? row[j] : 0.0f;
        s = s + v;
    }
    return s;
}

}  // namespace

extern "C" {

// N_ds = ceil(nsamp / ds)
int64_t oracle_nsamp_ds(int64_t nsamp, int ds) { return (nsamp + ds - 1) / ds; }

// Delay table, row-major [ndm][nchan], Eq. 4/5 in double in the literal order above.
// Returns d_max over ALL channels (masked or not; R6), or -1 on bad args.
int64_t oracle_delay_table(int nchan, double f_top, double chan_bw, double tsamp, int ds,
                           const double* dm, int ndm, int32_t* out) {
    if (nchan < 1 || ndm < 1 || ds < 1 || !(tsamp > 0.0) || !dm || !out) return -1;
    const double tsamp_ds = (double)ds * tsamp;
    int64_t dmax = 0;
    for (int i = 0; i < ndm; ++i) {
        for (int c = 0; c < nchan; ++c) {
            double f = f_top + (double)c * chan_bw;
            double a = 1.0 / (f * f);
            double b = 1.0 / (f_top * f_top);
            double delay_s = (K_DM * dm[i]) * (a - b);
            double v = std::floor(delay_s / tsamp_ds + 0.5);
            int32_t d = (int32_t)v;
            out[(size_t)i * nchan + c] = d;
            if (d > dmax) dmax = d;
        }
    }
    return dmax;
}

// uint8 in, uint32 out.  Computes columns t in [t_lo, t_hi) of rows 0..ndm-1 of the
// given delay table; out[i*out_pitch + (t - t_lo)].  mask may be NULL; nonzero = zapped
// (skipped, never read: DESIGN.md R6).  The caller guarantees t_hi + max delay <= N_ds
// (the "truncate" reading R5); reads beyond nsamp inside the last partial bin are zero.
int oracle_dedisperse_u8(const uint8_t* x, int nchan, int64_t nsamp, int64_t in_pitch, int ds,
                         const uint8_t* mask, const int32_t* delays, int ndm,
                         int64_t t_lo, int64_t t_hi, uint32_t* out, int64_t out_pitch) {
    if (!x || !delays || !out || nchan < 1 || ndm < 1 || ds < 1 || t_lo < 0 || t_hi < t_lo) return 1;
    const int64_t n = t_hi - t_lo;
    for (int i = 0; i < ndm; ++i) {
        uint32_t* o = out + (size_t)i * out_pitch;
        for (int64_t t = 0; t < n; ++t) o[t] = 0u;
        for (int c = 0; c < nchan; ++c) {
            if (mask && mask[c]) continue;
            const uint8_t* row = x + (size_t)c * in_pitch;
            const int64_t d = delays[(size_t)i * nchan + c];
            if (ds == 1) {
                const uint8_t* p = row + t_lo + d;
                for (int64_t t = 0; t < n; ++t) o[t] += p[t];
            } else {
                for (int64_t t = 0; t < n; ++t) o[t] += bin_u8(row, nsamp, ds, t_lo + t + d);
            }
        }
    }
    return 0;
}

// float32 in, float32 out: one fp32 accumulator per output starting at +0.0f, channels
// added in ascending order, no FMA, no reassociation (R9).
int oracle_dedisperse_f32(const float* x, int nchan, int64_t nsamp, int64_t in_pitch, int ds,
                          const uint8_t* mask, const int32_t* delays, int ndm,
                          int64_t t_lo, int64_t t_hi, float* out, int64_t out_pitch) {
    if (!x || !delays || !out || nchan < 1 || ndm < 1 || ds < 1 || t_lo < 0 || t_hi < t_lo) return 1;
    const int64_t n = t_hi - t_lo;
    for (int i = 0; i < ndm; ++i) {
        float* o = out + (size_t)i * out_pitch;
        for (int64_t t = 0; t < n; ++t) o[t] = 0.0f;
        for (int c = 0; c < nchan; ++c) {
            if (mask && mask[c]) continue;
            const float* row = x + (size_t)c * in_pitch;
            const int64_t d = delays[(size_t)i * nchan + c];
            if (ds == 1) {
                const float* p = row + t_lo + d;
                for (int64_t t = 0; t < n; ++t) o[t] = o[t] + p[t];
            } else {
                for (int64_t t = 0; t < n; ++t) o[t] = o[t] + bin_f32(row, nsamp, ds, t_lo + t + d);
            }
        }
    }
    return 0;
}

// float32 in, float64 out: the same sum accumulated in double (bins still formed in fp32,
// as the input to the sum is x_ds, an fp32 quantity).  The order-independent truth used
// for the second fp32 check (R9).
int oracle_dedisperse_f32_acc64(const float* x, int nchan, int64_t nsamp, int64_t in_pitch, int ds,
                                const uint8_t* mask, const int32_t* delays, int ndm,
                                int64_t t_lo, int64_t t_hi, double* out, int64_t out_pitch) {
    if (!x || !delays || !out || nchan < 1 || ndm < 1 || ds < 1 || t_lo < 0 || t_hi < t_lo) return 1;
    const int64_t n = t_hi - t_lo;
    for (int i = 0; i < ndm; ++i) {
        double* o = out + (size_t)i * out_pitch;
        for (int64_t t = 0; t < n; ++t) o[t] = 0.0;
        for (int c = 0; c < nchan; ++c) {
            if (mask && mask[c]) continue;
            const float* row = x + (size_t)c * in_pitch;
            const int64_t d = delays[(size_t)i * nchan + c];
            for (int64_t t = 0; t < n; ++t) o[t] += (double)bin_f32(row, nsamp, ds, t_lo + t + d);
        }
    }
    return 0;
}

}  // extern "C"
