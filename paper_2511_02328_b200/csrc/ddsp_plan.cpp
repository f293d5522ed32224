// ddsp_plan.cpp -- C ABI of libddsp (include/ddsp.h): plan creation (delay table in double, mask
// compaction, DM ordering), execute dispatch, host-buffer execute, destroy.
//
// The delay table follows PAPER.md:95-97 (Eq. 4) and PAPER.md:121 (Eq. 5) with the readings of
// K = 4.148808e3 s MHz^2, reference = centre of channel 0 (top of band),
// floor(x + 0.5) rounding, tsamp_ds = ds * tsamp, all in IEEE double on the host.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <numeric>

#include "ddsp_internal.h"

namespace {

const double kDispersionConstant = 4.148808e3;  // s MHz^2 pc^-1 cm^3 (units: DESIGN.md R1)

int note_cuda(const ddsp_plan* p, cudaError_t e) {
    if (e == cudaSuccess) return DDSP_OK;
    if (p) p->last_cuda = (int)e;
    (void)cudaGetLastError();  // clear the sticky-less error state of this thread
    return e == cudaErrorMemoryAllocation ? DDSP_ERR_ALLOC : DDSP_ERR_CUDA;
}

size_t elem_size_in(const ddsp_plan* p) { return p->in_dtype == DDSP_IN_U8 ? 1 : 4; }

// AUTO takes the lanes kernels only after they have passed their parity tests on a B200 (DESIGN.md section 8
// records the log); until then they run on request (ddsp_plan_set_kernel) and AUTO stays with the kernels that
// have a hardware history.  Flipped in code, by a commit that cites the log -- never by the environment.
constexpr bool kAutoTakesLanes = false;

void resolve_kernel(ddsp_plan* p) {
    if (p->kernel_req == DDSP_KERNEL_AUTO)
        p->kernel = (kAutoTakesLanes && p->lanes.ok) ? DDSP_KERNEL_LANES
                    : p->tiled.ok                    ? DDSP_KERNEL_TILED
                                                     : DDSP_KERNEL_DIRECT;
    else
        p->kernel = p->kernel_req;
}

}  // namespace

extern "C" {

const char* ddsp_version(void) { return "ddsp 0.1 (sm_100a)"; }

const char* ddsp_strerror(int code) {
    switch (code) {
        case DDSP_OK: return "ok";
        case DDSP_ERR_INVALID_ARG: return "invalid argument";
        case DDSP_ERR_NO_OUTPUT: return "no output: ceil(nsamp/downsample) <= maximum delay";
        case DDSP_ERR_UNSUPPORTED: return "unsupported";
        case DDSP_ERR_ALLOC: return "allocation failed";
        case DDSP_ERR_CUDA: return "CUDA error";
        default: return "unknown error code";
    }
}

int ddsp_plan_create(ddsp_plan** plan, int nchan, double f_top, double chan_bw, double tsamp,
                     int64_t nsamp, const double* dm_list, int ndm, int downsample,
                     const uint8_t* chan_mask, int in_dtype) {
    return ddsp_plan_create_rows(plan, nchan, f_top, chan_bw, tsamp, nsamp, dm_list, ndm, 0, ndm, downsample,
                                 chan_mask, in_dtype);
}

int ddsp_plan_create_rows(ddsp_plan** plan, int nchan, double f_top, double chan_bw, double tsamp,
                          int64_t nsamp, const double* dm_list, int ndm_all, int row_begin, int row_count,
                          int downsample, const uint8_t* chan_mask, int in_dtype) {
    if (!plan) return DDSP_ERR_INVALID_ARG;
    *plan = nullptr;
    if (ndm_all < 1 || row_begin < 0 || row_count < 1 || row_begin > ndm_all - row_count) return DDSP_ERR_INVALID_ARG;
    const int ndm = row_count;
    if (nchan < 1 || downsample < 1 || nsamp < 1 || !dm_list) return DDSP_ERR_INVALID_ARG;
    if (!(chan_bw < 0.0) || !(tsamp > 0.0) || !std::isfinite(f_top) || !std::isfinite(chan_bw) ||
        !std::isfinite(tsamp))
        return DDSP_ERR_INVALID_ARG;
    if (!(f_top + (double)(nchan - 1) * chan_bw > 0.0)) return DDSP_ERR_INVALID_ARG;
    if (in_dtype != DDSP_IN_U8 && in_dtype != DDSP_IN_F32) return DDSP_ERR_INVALID_ARG;
    for (int i = 0; i < ndm_all; ++i)
        if (!std::isfinite(dm_list[i]) || dm_list[i] < 0.0) return DDSP_ERR_INVALID_ARG;
    if ((int64_t)ndm * nchan > ((int64_t)1 << 31) - 1) return DDSP_ERR_UNSUPPORTED;

    ddsp_plan* p = new (std::nothrow) ddsp_plan;
    if (!p) return DDSP_ERR_ALLOC;
    int rc = DDSP_OK;
    try {
        p->nchan = nchan; p->ndm = ndm; p->ds = downsample; p->in_dtype = in_dtype;
        p->f_top = f_top; p->chan_bw = chan_bw; p->tsamp = tsamp; p->nsamp = nsamp;
        p->nsamp_ds = (nsamp + downsample - 1) / downsample;
        p->dm.assign(dm_list + row_begin, dm_list + row_begin + ndm);
        p->mask.assign((size_t)nchan, 0);
        if (chan_mask)
            for (int c = 0; c < nchan; ++c) p->mask[c] = chan_mask[c] ? 1 : 0;
        for (int c = 0; c < nchan; ++c)
            if (!p->mask[c]) p->chan_list.push_back(c);

        // A1/A2: channel frequencies and the delay table, in double, in this literal order.
        const double tsamp_ds = (double)downsample * tsamp;
        std::vector<double> chan_term((size_t)nchan);
        const double inv_top = 1.0 / (f_top * f_top);
        for (int c = 0; c < nchan; ++c) {
            const double f = f_top + (double)c * chan_bw;
            chan_term[c] = 1.0 / (f * f) - inv_top;
        }
        // d_max is the maximum over the WHOLE list (all trials, all channels), so that every shard of a list
        // has the same nsamp_out (invariant I7); only the plan's own rows are kept.
        p->delays.resize((size_t)ndm * nchan);
        std::vector<int32_t> scratch((size_t)nchan);
        int64_t dmax = 0;
        bool overflow = false;
        for (int i = 0; i < ndm_all; ++i) {
            const double kdm = kDispersionConstant * dm_list[i];
            const bool mine = i >= row_begin && i < row_begin + ndm;
            int32_t* row = mine ? &p->delays[(size_t)(i - row_begin) * nchan] : scratch.data();
            for (int c = 0; c < nchan; ++c) {
                const double v = std::floor((kdm * chan_term[c]) / tsamp_ds + 0.5);
                if (!(v < 2147483647.0)) { overflow = true; break; }
                row[c] = (int32_t)v;
                if (row[c] > dmax) dmax = row[c];
            }
            if (overflow) break;
        }
        if (overflow) {
            rc = DDSP_ERR_NO_OUTPUT;
        } else {
            p->dmax = dmax;
            p->nsamp_out = p->nsamp_ds - dmax;  // PAPER.md:228 (truncate; R5)
            if (p->nsamp_out <= 0) rc = DDSP_ERR_NO_OUTPUT;
        }
        if (rc == DDSP_OK) {
            p->in_pitch = nsamp;
            p->out_pitch = p->nsamp_out;
            p->order.resize((size_t)ndm);
            std::iota(p->order.begin(), p->order.end(), 0);
            std::stable_sort(p->order.begin(), p->order.end(),
                             [&](int a, int b) { return p->dm[a] < p->dm[b]; });   // p->dm: the plan's own rows
        }
    } catch (const std::bad_alloc&) {
        rc = DDSP_ERR_ALLOC;
    }
    if (rc != DDSP_OK) { delete p; return rc; }

    // device side.  Without a usable CUDA device the plan is host-only (device = -1): the getters and
    // ddsp_plan_get_delays work, ddsp_execute fails with DDSP_ERR_CUDA.  There is no CPU fallback.
    cudaError_t e = cudaGetDevice(&p->device);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        p->device = -1;
        p->last_cuda = (int)e;
    } else {
        cudaDeviceProp prop;
        e = cudaGetDeviceProperties(&prop, p->device);
        if (e == cudaSuccess) {
            p->sm_count = prop.multiProcessorCount;
            p->smem_optin = (int)prop.sharedMemPerBlockOptin;
            e = cudaMalloc((void**)&p->d_delays, p->delays.size() * sizeof(int32_t));
        }
        if (e == cudaSuccess)
            e = cudaMemcpy(p->d_delays, p->delays.data(), p->delays.size() * sizeof(int32_t),
                           cudaMemcpyHostToDevice);
        if (e == cudaSuccess && !p->chan_list.empty()) {
            e = cudaMalloc((void**)&p->d_chan_list, p->chan_list.size() * sizeof(int32_t));
            if (e == cudaSuccess)
                e = cudaMemcpy(p->d_chan_list, p->chan_list.data(),
                               p->chan_list.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
        }
        if (e != cudaSuccess) {
            rc = note_cuda(nullptr, e);
            ddsp_plan_destroy(p);
            return rc;
        }
    }
    rc = ddsp_tiled_plan(p);
    if (rc == DDSP_OK) rc = ddsp_lanes_plan(p);
    if (rc == DDSP_OK) {
        resolve_kernel(p);
        if (p->kernel == DDSP_KERNEL_LANES) rc = ddsp_lanes_prepare(p);
    }
    if (rc != DDSP_OK) { ddsp_plan_destroy(p); return rc; }
    *plan = p;
    return DDSP_OK;
}

int ddsp_plan_set_pitch(ddsp_plan* p, int64_t in_pitch, int64_t out_pitch) {
    if (!p || in_pitch < p->nsamp || out_pitch < p->nsamp_out) return DDSP_ERR_INVALID_ARG;
    p->in_pitch = in_pitch;
    p->out_pitch = out_pitch;
    if (p->d_stage_in) { cudaFree(p->d_stage_in); p->d_stage_in = nullptr; }
    if (p->d_stage_out) { cudaFree(p->d_stage_out); p->d_stage_out = nullptr; }
    int rc = ddsp_tiled_set_pitch(p);
    resolve_kernel(p);     // a pitch can disable a kernel that AUTO had chosen (16-byte row alignment)
    return rc;
}

int ddsp_plan_set_kernel(ddsp_plan* p, int kernel) {
    if (!p) return DDSP_ERR_INVALID_ARG;
    if (kernel != DDSP_KERNEL_AUTO && kernel != DDSP_KERNEL_DIRECT && kernel != DDSP_KERNEL_TILED &&
        kernel != DDSP_KERNEL_LANES)
        return DDSP_ERR_INVALID_ARG;
    if (kernel == DDSP_KERNEL_TILED && !p->tiled.ok) return DDSP_ERR_UNSUPPORTED;
    if (kernel == DDSP_KERNEL_LANES && !p->lanes.ok) return DDSP_ERR_UNSUPPORTED;
    p->kernel_req = kernel;
    resolve_kernel(p);
    return p->kernel == DDSP_KERNEL_LANES ? ddsp_lanes_prepare(p) : DDSP_OK;
}

int64_t ddsp_plan_nsamp_out(const ddsp_plan* p) { return p ? p->nsamp_out : -1; }
int64_t ddsp_plan_max_delay(const ddsp_plan* p) { return p ? p->dmax : -1; }
int ddsp_plan_nchan_unmasked(const ddsp_plan* p) { return p ? (int)p->chan_list.size() : -1; }
int ddsp_plan_kernel(const ddsp_plan* p) { return p ? p->kernel : -1; }
int ddsp_plan_launches_per_execute(const ddsp_plan* p) {
    if (!p) return -1;
    return p->kernel == DDSP_KERNEL_LANES ? (p->chan_list.empty() ? 1 : 2) : 1;   // interleave + accumulate
}
int64_t ddsp_plan_workspace_bytes(const ddsp_plan* p) {
    if (!p) return -1;
    return p->kernel == DDSP_KERNEL_LANES ? (int64_t)p->lanes.ws_bytes : 0;
}
int ddsp_plan_device_status(ddsp_plan* p, int* status) {
    if (!p || !status) return DDSP_ERR_INVALID_ARG;
    *status = 0;
    if (p->device < 0 || !p->lanes.d_status) return DDSP_OK;
    return note_cuda(p, cudaMemcpy(status, p->lanes.d_status, sizeof(int), cudaMemcpyDeviceToHost));
}
int ddsp_last_cuda_error(const ddsp_plan* p) { return p ? p->last_cuda.load() : 0; }

int ddsp_plan_get_delays(const ddsp_plan* p, int32_t* host_out) {
    if (!p || !host_out) return DDSP_ERR_INVALID_ARG;
    std::memcpy(host_out, p->delays.data(), p->delays.size() * sizeof(int32_t));
    return DDSP_OK;
}

int ddsp_execute(const ddsp_plan* p, const void* d_in, void* d_out, void* cuda_stream) {
    return ddsp_execute_ws(p, d_in, d_out, nullptr, 0, cuda_stream);
}

int ddsp_execute_ws(const ddsp_plan* p, const void* d_in, void* d_out, void* d_ws, int64_t ws_bytes,
                    void* cuda_stream) {
    if (!p || !d_in || !d_out) return DDSP_ERR_INVALID_ARG;
    if (p->device < 0) return DDSP_ERR_CUDA;  // host-only plan: no device, no fallback
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (p->kernel == DDSP_KERNEL_LANES) {
        if (d_ws && (ws_bytes < (int64_t)p->lanes.ws_bytes || ((uintptr_t)d_ws & 15u))) return DDSP_ERR_INVALID_ARG;
        e = ddsp_launch_lanes(p, d_in, d_out, d_ws, s);
    } else if (p->kernel == DDSP_KERNEL_TILED && !ddsp_tiled_can_run(p, d_in, d_out)) {
        // unaligned buffers: correct through the direct kernel unless the tiled one was forced
        if (p->kernel_req == DDSP_KERNEL_TILED) return DDSP_ERR_UNSUPPORTED;
        e = ddsp_launch_direct(p, d_in, d_out, s);
    } else if (p->kernel == DDSP_KERNEL_TILED)
        e = ddsp_launch_tiled(p, d_in, d_out, s);
    else
        e = ddsp_launch_direct(p, d_in, d_out, s);
    return note_cuda(p, e);
}

int ddsp_execute_host(ddsp_plan* p, const void* h_in, void* h_out, void* cuda_stream) {
    if (!p || !h_in || !h_out) return DDSP_ERR_INVALID_ARG;
    if (p->device < 0) return DDSP_ERR_CUDA;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t in_bytes = (size_t)p->nchan * (size_t)p->in_pitch * elem_size_in(p);
    const size_t out_bytes = (size_t)p->ndm * (size_t)p->out_pitch * 4;
    cudaError_t e = cudaSuccess;
    if (!p->d_stage_in) e = cudaMalloc(&p->d_stage_in, in_bytes);
    if (e == cudaSuccess && !p->d_stage_out) e = cudaMalloc(&p->d_stage_out, out_bytes);
    if (e != cudaSuccess) return note_cuda(p, e);
    e = cudaMemcpyAsync(p->d_stage_in, h_in, in_bytes, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return note_cuda(p, e);
    int rc = ddsp_execute(p, p->d_stage_in, p->d_stage_out, cuda_stream);
    if (rc != DDSP_OK) return rc;
    // Only the valid columns need to come back, but rows are pitch-strided on both sides.
    e = cudaMemcpy2DAsync(h_out, (size_t)p->out_pitch * 4, p->d_stage_out, (size_t)p->out_pitch * 4,
                          (size_t)p->nsamp_out * 4, (size_t)p->ndm, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    return note_cuda(p, e);
}

int ddsp_execute_host_pipelined(ddsp_plan* p, const void* h_in, void* h_out, void* cuda_stream, int npieces) {
    if (!p || !h_in || !h_out || npieces < 1) return DDSP_ERR_INVALID_ARG;
    if (p->device < 0) return DDSP_ERR_CUDA;
    // only the lanes kernels can be launched on a range of output columns
    if (p->kernel != DDSP_KERNEL_LANES || !p->lanes.ok) return DDSP_ERR_UNSUPPORTED;
    const size_t esize = elem_size_in(p);
    const size_t in_bytes = (size_t)p->nchan * (size_t)p->in_pitch * esize;
    const size_t out_bytes = (size_t)p->ndm * (size_t)p->out_pitch * 4;
    cudaError_t e = cudaSuccess;
    if (!p->d_stage_in) e = cudaMalloc(&p->d_stage_in, in_bytes);
    if (e == cudaSuccess && !p->d_stage_out) e = cudaMalloc(&p->d_stage_out, out_bytes);
    if (e == cudaSuccess && !p->hs_in) e = cudaStreamCreateWithFlags(&p->hs_in, cudaStreamNonBlocking);
    if (e == cudaSuccess && !p->hs_k) e = cudaStreamCreateWithFlags(&p->hs_k, cudaStreamNonBlocking);
    if (e == cudaSuccess && !p->hs_out) e = cudaStreamCreateWithFlags(&p->hs_out, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)cuda_stream);   // work queued before this call
    if (e != cudaSuccess) return note_cuda(p, e);

    const int64_t nout = p->nsamp_out;
    const int64_t piece = (nout + npieces - 1) / npieces;
    const size_t in_pitch_b = (size_t)p->in_pitch * esize, out_pitch_b = (size_t)p->out_pitch * 4;
    std::vector<cudaEvent_t> events;
    int64_t in_done = 0;      // native input columns [0, in_done) are on the device (or on their way, in order)
    for (int64_t a = 0; a < nout && e == cudaSuccess; a += piece) {
        const int64_t b = std::min(a + piece, nout);
        // outputs [a, b) read downsampled samples < b + d_max, i.e. native columns < (b + d_max) * ds
        const int64_t need = std::min<int64_t>(p->nsamp, (b + p->dmax) * p->ds);
        cudaEvent_t ev_in = nullptr, ev_k = nullptr;
        e = cudaEventCreateWithFlags(&ev_in, cudaEventDisableTiming);
        if (e == cudaSuccess) { events.push_back(ev_in); e = cudaEventCreateWithFlags(&ev_k, cudaEventDisableTiming); }
        if (e == cudaSuccess) events.push_back(ev_k);
        if (e == cudaSuccess && need > in_done) {
            e = cudaMemcpy2DAsync((char*)p->d_stage_in + (size_t)in_done * esize, in_pitch_b,
                                  (const char*)h_in + (size_t)in_done * esize, in_pitch_b,
                                  (size_t)(need - in_done) * esize, (size_t)p->nchan, cudaMemcpyHostToDevice, p->hs_in);
            in_done = need;
        }
        if (e == cudaSuccess) e = cudaEventRecord(ev_in, p->hs_in);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->hs_k, ev_in, 0);
        // the pieces share the plan's workspace: they are ordered on one stream
        if (e == cudaSuccess) e = ddsp_launch_lanes(p, p->d_stage_in, p->d_stage_out, nullptr, p->hs_k, a, b - a);
        if (e == cudaSuccess) e = cudaEventRecord(ev_k, p->hs_k);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->hs_out, ev_k, 0);
        if (e == cudaSuccess)
            e = cudaMemcpy2DAsync((char*)h_out + (size_t)a * 4, out_pitch_b, (const char*)p->d_stage_out + (size_t)a * 4,
                                  out_pitch_b, (size_t)(b - a) * 4, (size_t)p->ndm, cudaMemcpyDeviceToHost, p->hs_out);
    }
    // drain everything that was enqueued, also after an error
    cudaError_t e1 = cudaStreamSynchronize(p->hs_in), e2 = cudaStreamSynchronize(p->hs_k), e3 = cudaStreamSynchronize(p->hs_out);
    for (cudaEvent_t ev : events) cudaEventDestroy(ev);
    if (e == cudaSuccess) e = e1 != cudaSuccess ? e1 : (e2 != cudaSuccess ? e2 : e3);
    return note_cuda(p, e);
}

int ddsp_plan_destroy(ddsp_plan* p) {
    if (!p) return DDSP_OK;
    ddsp_tiled_free(p);
    ddsp_lanes_free(p);
    if (p->d_delays) cudaFree(p->d_delays);
    if (p->d_chan_list) cudaFree(p->d_chan_list);
    if (p->d_stage_in) cudaFree(p->d_stage_in);
    if (p->d_stage_out) cudaFree(p->d_stage_out);
    if (p->hs_in) cudaStreamDestroy(p->hs_in);
    if (p->hs_k) cudaStreamDestroy(p->hs_k);
    if (p->hs_out) cudaStreamDestroy(p->hs_out);
    delete p;
    return DDSP_OK;
}

}  // extern "C"
