// api.cu -- the extern "C" boundary declared in include/mred.h: argument validation, workspace
// carving and kernel launches.  No allocation, no synchronisation, no global state except the last
// CUDA error code.
#include "common.cuh"
#include <atomic>
#include <math.h>

namespace mred {

static std::atomic<int> g_last_cuda_error{0};
void set_cuda_error(cudaError_t e) { g_last_cuda_error.store((int)e); }

int sm_count()
{
    static std::atomic<int> cached[64];
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    n = cached[dev].load(std::memory_order_relaxed);
    if (n > 0) return n;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) return 148;
    cached[dev].store(n, std::memory_order_relaxed);
    return n;
}

static bool opts_ok(const mred_comb_opts* o, bool allow_minmax = false)
{
    if (!o) return false;
    if (o->mode != MRED_MEDIAN && o->mode != MRED_MEAN && o->mode != MRED_SIGCLIP && !(allow_minmax && (o->mode == MRED_MINMAX || o->mode == MRED_MEDCLIP)))
        return false;
    if ((o->mode == MRED_SIGCLIP || o->mode == MRED_MEDCLIP) && (!(o->ksigma >= 0.f) || o->max_iter < 0)) return false;
    return true;
}

struct ReduceWs {
    float* cal;               // [n][h][w]
    float* reg;               // [n][h][w]
    unsigned long long* os;   // [n][frame_sums_parts] block partials of the overscan sums
    int32_t* ishift;          // [n][2]
    double* shift;            // [n][2]
    int32_t* fp;              // [n][4]
    void* est;                // estimate workspace
    void* rs;                 // resample workspace (x-shifted stack, small stacks only)
    size_t rs_bytes;
    void* fill;               // list of the bad-pixel fill (mred_reduce_filled)
    size_t bytes;
};

static ReduceWs carve_reduce(void* ws, const Geom& g, int n)
{
    ReduceWs r;
    char* p = static_cast<char*>(ws);
    auto take = [&](size_t b) { char* q = p; p += align_up(b, 256); return q; };
    const size_t np = (size_t)g.w * g.h;
    r.cal = reinterpret_cast<float*>(take(4 * np * n));
    r.reg = reinterpret_cast<float*>(take(4 * np * n));
    r.os = reinterpret_cast<unsigned long long*>(take(8 * (size_t)n * frame_sums_parts(g)));
    r.ishift = reinterpret_cast<int32_t*>(take(8 * (size_t)n));
    r.shift = reinterpret_cast<double*>(take(16 * (size_t)n));
    r.fp = reinterpret_cast<int32_t*>(take(16 * (size_t)n));
    r.est = take(estimate_ws_bytes(g.w, g.h, n));
    r.rs_bytes = resample_ws_bytes(g.w, g.h, n);
    r.rs = take(r.rs_bytes);
    r.fill = take(fill_ws_bytes(g.w, g.h));
    r.bytes = (size_t)(p - static_cast<char*>(ws));
    return r;
}

struct HostWs {
    uint16_t* raw;   // [n][H][W]
    float* out;      // [h][w]
    uint16_t* count; // [h][w]
    void* reduce;
    size_t bytes;
};

static HostWs carve_host(void* ws, const Geom& g, int n)
{
    HostWs r;
    char* p = static_cast<char*>(ws);
    auto take = [&](size_t b) { char* q = p; p += align_up(b, 256); return q; };
    const size_t np = (size_t)g.w * g.h;
    r.raw = reinterpret_cast<uint16_t*>(take(2 * (size_t)g.W * g.H * n));
    r.out = reinterpret_cast<float*>(take(4 * np));
    r.count = reinterpret_cast<uint16_t*>(take(2 * np));
    r.reduce = take(carve_reduce(nullptr, g, n).bytes);
    r.bytes = (size_t)(p - static_cast<char*>(ws));
    return r;
}

// Everything mred_reduce* checks apart from the raw / out pointers (device for mred_reduce, host for
// mred_reduce_host) and the workspace: shared so that mred_reduce_host can refuse a call before it enqueues anything.
static int reduce_args_ok(const mred_geom* geom, int n, const float* MB, const float* MD, const float* MF, int ref_index,
                          int max_lag, const uint8_t* badmask, const mred_comb_opts* opts, const uint16_t* count,
                          const uint32_t* rejmask, const double* shift_out, const int32_t* footprint_out)
{
    if (!geom_ok(geom) || !MB || !MD || !MF || !opts_ok(opts, true)) return MRED_EINVAL;
    if (n < 1 || n > MRED_MAX_STACK || geom->w < 4 || geom->h < 4 || geom->w > MRED_MAX_PROFILE || geom->h > MRED_MAX_PROFILE)
        return MRED_EINVAL;
    if (ref_index < 0 || ref_index >= n || max_lag < 0 || max_lag > MRED_MAX_LAG || max_lag >= geom->w || max_lag >= geom->h)
        return MRED_EINVAL;
    if (!aligned16(MB) || !aligned16(MD) || !aligned16(MF) || (count && !aligned16(count)) || (rejmask && !aligned16(rejmask)) ||
        (badmask && !aligned16(badmask)) || (shift_out && !aligned16(shift_out)) || (footprint_out && !aligned16(footprint_out)))
        return MRED_EALIGN;
    return MRED_OK;
}

}  // namespace mred

using namespace mred;

extern "C" {
#pragma GCC visibility push(default)

const char* mred_version(void) { return "mred 0.1 (sm_100a)"; }

int mred_last_cuda_error(void) { return g_last_cuda_error.load(); }

const char* mred_strerror(int status)
{
    switch (status) {
        case MRED_OK: return "ok";
        case MRED_EINVAL: return "invalid argument (null pointer, shape, geometry, count or option)";
        case MRED_EALIGN: return "device pointer not 16-byte aligned";
        case MRED_EWORKSPACE: return "workspace missing or too small";
        case MRED_ECUDA: return "CUDA runtime error (see mred_last_cuda_error)";
        case MRED_ELIMIT: return "problem exceeds the static scratch of the no-allocation entry point (MRED_STATIC_SCRATCH_BYTES)";
        default: return "unknown status";
    }
}

size_t mred_workspace_bytes(int call, const mred_geom* geom, int n)
{
    if (!geom || n < 1) return 0;
    const Geom g = to_geom(geom);
    switch (call) {
        case MRED_CALL_BUILD_MASTERS: return masters_ws_bytes(g, n);
        case MRED_CALL_CALIBRATE: return align_up(8 * (size_t)n * frame_sums_parts(g), 16);
        case MRED_CALL_ESTIMATE_SHIFTS: return estimate_ws_bytes(g.w, g.h, n);
        case MRED_CALL_RESAMPLE: return resample_ws_bytes(g.w, g.h, n);   /* optional: without it the one-kernel route runs */
        case MRED_CALL_COADD: return 0;
        case MRED_CALL_REDUCE: return carve_reduce(nullptr, g, n).bytes;
        case MRED_CALL_FILL_BAD: return fill_ws_bytes(g.w, g.h);
        default: return 0;
    }
}

size_t mred_reduce_host_workspace_bytes(const mred_geom* geom, int n)
{
    if (!geom || n < 1) return 0;
    return carve_host(nullptr, to_geom(geom), n).bytes;
}

int mred_build_masters(const mred_geom* geom, const uint16_t* bias, int nb, const uint16_t* dark, int nd,
                       float t_dark, const uint16_t* flat, int nf, float t_flat, const mred_comb_opts* opts,
                       float* MB, float* MD, float* MF, void* ws, size_t ws_bytes, void* stream)
{
    if (!geom_ok(geom) || !bias || !dark || !flat || !MB || !MD || !MF || !opts_ok(opts)) return MRED_EINVAL;
    if (nb < 1 || nd < 1 || nf < 1 || nb > MRED_MAX_STACK || nd > MRED_MAX_STACK || nf > MRED_MAX_STACK) return MRED_EINVAL;
    if (!(t_dark > 0.f) || !(t_flat >= 0.f)) return MRED_EINVAL;
    if (!aligned16(bias) || !aligned16(dark) || !aligned16(flat) || !aligned16(MB) || !aligned16(MD) || !aligned16(MF))
        return MRED_EALIGN;
    const Geom g = to_geom(geom);
    int nmax = nb > nd ? nb : nd;
    nmax = nmax > nf ? nmax : nf;
    if (!ws || !aligned16(ws) || ws_bytes < masters_ws_bytes(g, nmax)) return MRED_EWORKSPACE;
    return launch_build_masters(g, bias, nb, dark, nd, t_dark, flat, nf, t_flat, *opts, MB, MD, MF, ws,
                                static_cast<cudaStream_t>(stream));
}

int mred_calibrate(const mred_geom* geom, const uint16_t* raw, int n, float dark_scale, const float* MB,
                   const float* MD, const float* MF, float* out, double* level_out, void* ws, size_t ws_bytes,
                   void* stream)
{
    if (!geom_ok(geom) || !raw || !MB || !MD || !MF || !out || n < 1 || n > 65535 * 8) return MRED_EINVAL;
    if (!aligned16(raw) || !aligned16(MB) || !aligned16(MD) || !aligned16(MF) || !aligned16(out)) return MRED_EALIGN;
    const Geom g = to_geom(geom);
    if (!ws || !aligned16(ws) || ws_bytes < 8 * (size_t)n * frame_sums_parts(g)) return MRED_EWORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned long long* os = static_cast<unsigned long long*>(ws);
    int rc = launch_frame_sums(raw, g, n, os, nullptr, 0, st);
    if (rc) return rc;
    return launch_calibrate(raw, g, n, dark_scale, MB, MD, MF, out, level_out, os, st);
}

int mred_fill_bad(float* frames, int n, int w, int h, const uint8_t* badmask, void* ws, size_t ws_bytes, void* stream)
{
    if (!frames || !badmask || n < 1 || n > 65535 || w < 1 || h < 1) return MRED_EINVAL;
    if ((int64_t)w * h >= (int64_t)1 << 31) return MRED_EINVAL;
    if (!aligned16(frames) || !aligned16(badmask)) return MRED_EALIGN;
    if (!ws || !aligned16(ws) || ws_bytes < fill_ws_bytes(w, h)) return MRED_EWORKSPACE;
    return launch_fill_bad(frames, n, w, h, badmask, ws, static_cast<cudaStream_t>(stream));
}

int mred_estimate_shifts_peak(const float* frames, int n, int w, int h, int ref_index, int max_lag,
                              const uint8_t* badmask, int peak, int32_t* ishift, double* shift, void* ws, size_t ws_bytes,
                              void* stream)
{
    if (!frames || !ishift || !shift || n < 1 || n > MRED_MAX_STACK || w < 1 || h < 1) return MRED_EINVAL;
    if (w > MRED_MAX_PROFILE || h > MRED_MAX_PROFILE) return MRED_EINVAL;   // a whole profile is sorted in shared memory
    if (ref_index < 0 || ref_index >= n || max_lag < 0 || max_lag > MRED_MAX_LAG || max_lag >= w || max_lag >= h)
        return MRED_EINVAL;
    if (peak != MRED_PEAK_PARABOLA && peak != MRED_PEAK_GAUSSIAN) return MRED_EINVAL;
    if (!aligned16(frames) || !aligned16(ishift) || !aligned16(shift) || (badmask && !aligned16(badmask)))
        return MRED_EALIGN;
    if (!ws || !aligned16(ws) || ws_bytes < estimate_ws_bytes(w, h, n)) return MRED_EWORKSPACE;
    return launch_estimate(frames, n, w, h, ref_index, max_lag, badmask, ishift, shift, ws, 0, peak,
                           static_cast<cudaStream_t>(stream));
}

int mred_estimate_shifts(const float* frames, int n, int w, int h, int ref_index, int max_lag,
                         const uint8_t* badmask, int32_t* ishift, double* shift, void* ws, size_t ws_bytes,
                         void* stream)
{
    return mred_estimate_shifts_peak(frames, n, w, h, ref_index, max_lag, badmask, MRED_PEAK_PARABOLA, ishift, shift, ws,
                                     ws_bytes, stream);
}

int mred_estimate_shifts_static(const float* frames, int n, int w, int h, int ref_index, int max_lag,
                                const uint8_t* badmask, int peak, int32_t* ishift, double* shift, void* stream)
{
    if (!frames || !ishift || !shift || n < 1 || n > MRED_MAX_STACK || w < 1 || h < 1) return MRED_EINVAL;
    if (w > MRED_MAX_PROFILE || h > MRED_MAX_PROFILE) return MRED_EINVAL;
    if (ref_index < 0 || ref_index >= n || max_lag < 0 || max_lag > MRED_MAX_LAG || max_lag >= w || max_lag >= h)
        return MRED_EINVAL;
    if (peak != MRED_PEAK_PARABOLA && peak != MRED_PEAK_GAUSSIAN) return MRED_EINVAL;
    if (!aligned16(frames) || !aligned16(ishift) || !aligned16(shift) || (badmask && !aligned16(badmask)))
        return MRED_EALIGN;
    return launch_estimate_static(frames, n, w, h, ref_index, max_lag, badmask, ishift, shift, peak,
                                  static_cast<cudaStream_t>(stream));
}

int mred_resample(const float* in, int n, int w, int h, const double* sx, const double* sy, float fill,
                  float* out, int32_t* footprint, void* ws, size_t ws_bytes, void* stream)
{
    if (ws && !aligned16(ws)) return MRED_EALIGN;
    if (!in || !out || !sx || !sy || n < 1 || n > MRED_MAX_STACK || w < 4 || h < 4 || in == out) return MRED_EINVAL;
    for (int k = 0; k < n; ++k)
        if (!isfinite(sx[k]) || !isfinite(sy[k]) || fabs(sx[k]) > 1.0e6 || fabs(sy[k]) > 1.0e6) return MRED_EINVAL;
    if (!aligned16(in) || !aligned16(out)) return MRED_EALIGN;
    if (footprint)
        for (int k = 0; k < n; ++k) {
            int lo, hi;
            axis_footprint(w, sx[k], lo, hi);
            footprint[4 * k] = lo; footprint[4 * k + 1] = hi;
            axis_footprint(h, sy[k], lo, hi);
            footprint[4 * k + 2] = lo; footprint[4 * k + 3] = hi;
        }
    return launch_resample(in, n, w, h, sx, sy, nullptr, fill, out, nullptr, ws, ws_bytes, static_cast<cudaStream_t>(stream));
}

int mred_resample_interp(const float* in, int n, int w, int h, const double* sx, const double* sy, float fill,
                         int interp, float* out, int32_t* footprint, void* stream)
{
    if (interp == MRED_INTERP_SPLINE) return mred_resample(in, n, w, h, sx, sy, fill, out, footprint, nullptr, 0, stream);
    if (interp != MRED_INTERP_BILINEAR && interp != MRED_INTERP_NEAREST) return MRED_EINVAL;
    if (!in || !out || !sx || !sy || n < 1 || n > MRED_MAX_STACK || w < 2 || h < 2 || in == out) return MRED_EINVAL;
    if ((int64_t)w * h >= (int64_t)1 << 31) return MRED_EINVAL;
    for (int k = 0; k < n; ++k)
        if (!isfinite(sx[k]) || !isfinite(sy[k]) || fabs(sx[k]) > 1.0e6 || fabs(sy[k]) > 1.0e6) return MRED_EINVAL;
    if (!aligned16(in) || !aligned16(out)) return MRED_EALIGN;
    if (footprint)
        for (int k = 0; k < n; ++k) {
            int lo, hi;
            axis_footprint(w, sx[k], lo, hi);
            footprint[4 * k] = lo; footprint[4 * k + 1] = hi;
            axis_footprint(h, sy[k], lo, hi);
            footprint[4 * k + 2] = lo; footprint[4 * k + 3] = hi;
        }
    return launch_resample_lin(in, n, w, h, sx, sy, interp, fill, out, static_cast<cudaStream_t>(stream));
}

int mred_coadd(const float* stack, int n, int w, int h, const int32_t* footprint, const mred_comb_opts* opts,
               float* out, uint16_t* count, uint32_t* rejmask, void* stream)
{
    if (!stack || !out || n < 1 || n > MRED_MAX_STACK || w < 1 || h < 1 || !opts_ok(opts, true)) return MRED_EINVAL;
    if ((int64_t)w * h >= (int64_t)1 << 31) return MRED_EINVAL;
    if (!aligned16(stack) || !aligned16(out) || (count && !aligned16(count)) || (rejmask && !aligned16(rejmask)))
        return MRED_EALIGN;
    return launch_coadd(stack, n, w, h, footprint, nullptr, *opts, out, count, rejmask,
                        static_cast<cudaStream_t>(stream));
}

int mred_reduce_workspace_views(const mred_geom* geom, int n, size_t* calibrated_offset, size_t* registered_offset)
{
    if (!geom_ok(geom) || n < 1 || n > MRED_MAX_STACK || !calibrated_offset || !registered_offset) return MRED_EINVAL;
    char* base = nullptr;
    const ReduceWs r = carve_reduce(base, to_geom(geom), n);
    *calibrated_offset = (size_t)(reinterpret_cast<char*>(r.cal) - base);
    *registered_offset = (size_t)(reinterpret_cast<char*>(r.reg) - base);
    return MRED_OK;
}

// The science path in two parts, so that mred_reduce_host_overlapped can run the first one chunk by chunk while the rest
// of the stack is still on its way to the device.
//   reduce_calibrate: frames [c0, c0 + nc) of the raw stack: overscan levels, calibration, and the marginal profile sums
//   of O4 (left in the accumulators of the estimate workspace).  The call for c0 == 0 also clears those accumulators and
//   takes the valid-pixel counts of the bad-pixel mask, so it has to be enqueued first.
//   reduce_finish: estimate_shifts from the sums, (fill,) resample, coadd.
static int reduce_calibrate(const Geom& g, const uint16_t* raw, int n, int c0, int nc, float dark_scale, const float* MB,
                            const float* MD, const float* MF, const uint8_t* badmask, const ReduceWs& r, cudaStream_t st)
{
    // The level kernel also clears the accumulators of estimate_shifts (no memset node between the stages); the
    // calibrate kernel sums the marginal profiles itself (leaving out masked pixels), so estimate_shifts starts at
    // its finalize step and the calibrated stack is not re-read.
    void* zero;
    size_t zero_bytes;
    long long *colsum, *rowsum;
    estimate_accumulators(r.est, g.w, g.h, n, &zero, &zero_bytes, &colsum, &rowsum);
    const int nos = frame_sums_parts(g);
    const uint16_t* rawc = raw + (size_t)c0 * g.W * g.H;
    unsigned long long* osc = r.os + (size_t)c0 * nos;
    int rc;
    if ((rc = launch_frame_sums(rawc, g, nc, osc, c0 == 0 ? zero : nullptr, c0 == 0 ? zero_bytes : 0, st))) return rc;
    if (c0 == 0 && badmask)      // the mask is the same for every frame: its valid-pixel counts are taken once
        if ((rc = launch_mask_counts(badmask, g.w, g.h, n, r.est, st))) return rc;
    return launch_calibrate_prof(rawc, g, nc, dark_scale, MB, MD, MF, r.cal + (size_t)c0 * g.w * g.h, osc, badmask,
                                 colsum + (size_t)c0 * g.w, rowsum + (size_t)c0 * g.h, st);
}

#define MRED_STAGE_EVENT(i) \
    do { if (events && events[i]) MRED_CUDA_TRY(cudaEventRecord(static_cast<cudaEvent_t>(events[i]), st)); } while (0)

static int reduce_finish(const Geom& g, int n, int ref_index, int max_lag, const uint8_t* badmask, float fill,
                         const mred_comb_opts* opts, float* out, uint16_t* count, uint32_t* rejmask, double* shift_out,
                         int32_t* footprint_out, const ReduceWs& r, cudaStream_t st, void* const* events, bool fill_bad)
{
    int rc;
    const int est_flags = EST_ZEROED | EST_HAVE_SUMS | (badmask ? EST_SHARED_COUNTS : 0);
    double* shift = shift_out ? shift_out : r.shift;
    int32_t* fp = footprint_out ? footprint_out : r.fp;
    if ((rc = launch_estimate(r.cal, n, g.w, g.h, ref_index, max_lag, badmask, r.ishift, shift, r.est, est_flags, MRED_PEAK_PARABOLA, st))) return rc;
    MRED_STAGE_EVENT(2);
    // bad-pixel fill (O7) between the calibrated stack and its resampling: a hot pixel would otherwise ring through the
    // spline prefilter; the profile sums above were taken without the masked pixels, so the shifts do not depend on it
    if (fill_bad && (rc = launch_fill_bad(r.cal, n, g.w, g.h, badmask, r.fill, st))) return rc;
    if ((rc = launch_resample(r.cal, n, g.w, g.h, nullptr, nullptr, shift, fill, r.reg, fp, r.rs, r.rs_bytes, st))) return rc;
    MRED_STAGE_EVENT(3);
    if ((rc = launch_coadd(r.reg, n, g.w, g.h, nullptr, fp, *opts, out, count, rejmask, st))) return rc;
    MRED_STAGE_EVENT(4);
    return MRED_OK;
}

static int reduce_impl(const mred_geom* geom, const uint16_t* raw, int n, float dark_scale, const float* MB,
                       const float* MD, const float* MF, int ref_index, int max_lag, const uint8_t* badmask, float fill,
                       const mred_comb_opts* opts, float* out, uint16_t* count, uint32_t* rejmask, double* shift_out,
                       int32_t* footprint_out, void* ws, size_t ws_bytes, void* stream, void* const* events, bool fill_bad)
{
    if (!raw || !out || (fill_bad && !badmask)) return MRED_EINVAL;
    if (!aligned16(raw) || !aligned16(out)) return MRED_EALIGN;
    int rc = reduce_args_ok(geom, n, MB, MD, MF, ref_index, max_lag, badmask, opts, count, rejmask, shift_out, footprint_out);
    if (rc) return rc;
    const Geom g = to_geom(geom);
    if (!ws || !aligned16(ws) || ws_bytes < carve_reduce(nullptr, g, n).bytes) return MRED_EWORKSPACE;
    const ReduceWs r = carve_reduce(ws, g, n);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    MRED_STAGE_EVENT(0);
    if ((rc = reduce_calibrate(g, raw, n, 0, n, dark_scale, MB, MD, MF, badmask, r, st))) return rc;
    MRED_STAGE_EVENT(1);
    return reduce_finish(g, n, ref_index, max_lag, badmask, fill, opts, out, count, rejmask, shift_out, footprint_out, r, st,
                         events, fill_bad);
}
#undef MRED_STAGE_EVENT

int mred_reduce_staged(const mred_geom* geom, const uint16_t* raw, int n, float dark_scale, const float* MB,
                       const float* MD, const float* MF, int ref_index, int max_lag, const uint8_t* badmask, float fill,
                       const mred_comb_opts* opts, float* out, uint16_t* count, uint32_t* rejmask, double* shift_out,
                       int32_t* footprint_out, void* ws, size_t ws_bytes, void* stream, void* const* events)
{
    return reduce_impl(geom, raw, n, dark_scale, MB, MD, MF, ref_index, max_lag, badmask, fill, opts, out, count, rejmask,
                       shift_out, footprint_out, ws, ws_bytes, stream, events, false);
}

int mred_reduce_filled(const mred_geom* geom, const uint16_t* raw, int n, float dark_scale, const float* MB,
                       const float* MD, const float* MF, int ref_index, int max_lag, const uint8_t* badmask, float fill,
                       const mred_comb_opts* opts, float* out, uint16_t* count, uint32_t* rejmask, double* shift_out,
                       int32_t* footprint_out, void* ws, size_t ws_bytes, void* stream)
{
    return reduce_impl(geom, raw, n, dark_scale, MB, MD, MF, ref_index, max_lag, badmask, fill, opts, out, count, rejmask,
                       shift_out, footprint_out, ws, ws_bytes, stream, nullptr, true);
}

int mred_reduce(const mred_geom* geom, const uint16_t* raw, int n, float dark_scale, const float* MB,
                const float* MD, const float* MF, int ref_index, int max_lag, const uint8_t* badmask, float fill,
                const mred_comb_opts* opts, float* out, uint16_t* count, uint32_t* rejmask, double* shift_out,
                int32_t* footprint_out, void* ws, size_t ws_bytes, void* stream)
{
    return mred_reduce_staged(geom, raw, n, dark_scale, MB, MD, MF, ref_index, max_lag, badmask, fill, opts, out, count,
                              rejmask, shift_out, footprint_out, ws, ws_bytes, stream, nullptr);
}

int mred_reduce_host(const mred_geom* geom, const uint16_t* raw_host, int n, float dark_scale, const float* MB,
                     const float* MD, const float* MF, int ref_index, int max_lag, const uint8_t* badmask, float fill,
                     const mred_comb_opts* opts, float* out_host, uint16_t* count_host, double* shift_host, void* ws,
                     size_t ws_bytes, void* stream)
{
    if (!raw_host || !out_host) return MRED_EINVAL;
    // every argument is checked before the first copy is enqueued (header: nothing is enqueued on EINVAL / EALIGN / EWORKSPACE)
    int rc = reduce_args_ok(geom, n, MB, MD, MF, ref_index, max_lag, badmask, opts, nullptr, nullptr, nullptr, nullptr);
    if (rc) return rc;
    const Geom g = to_geom(geom);
    if (!ws || !aligned16(ws) || ws_bytes < carve_host(nullptr, g, n).bytes) return MRED_EWORKSPACE;
    const HostWs hw = carve_host(ws, g, n);
    const ReduceWs r = carve_reduce(hw.reduce, g, n);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t np = (size_t)g.w * g.h;
    MRED_CUDA_TRY(cudaMemcpyAsync(hw.raw, raw_host, 2 * (size_t)g.W * g.H * n, cudaMemcpyHostToDevice, st));
    rc = mred_reduce(geom, hw.raw, n, dark_scale, MB, MD, MF, ref_index, max_lag, badmask, fill, opts, hw.out,
                     count_host ? hw.count : nullptr, nullptr, r.shift, nullptr, hw.reduce,
                     carve_reduce(nullptr, g, n).bytes, stream);
    if (rc) return rc;
    MRED_CUDA_TRY(cudaMemcpyAsync(out_host, hw.out, 4 * np, cudaMemcpyDeviceToHost, st));
    if (count_host) MRED_CUDA_TRY(cudaMemcpyAsync(count_host, hw.count, 2 * np, cudaMemcpyDeviceToHost, st));
    if (shift_host) MRED_CUDA_TRY(cudaMemcpyAsync(shift_host, r.shift, 16 * (size_t)n, cudaMemcpyDeviceToHost, st));
    return MRED_OK;
}

int mred_reduce_host_overlapped(const mred_geom* geom, const uint16_t* raw_host, int n, float dark_scale, const float* MB,
                                const float* MD, const float* MF, int ref_index, int max_lag, const uint8_t* badmask,
                                float fill, const mred_comb_opts* opts, float* out_host, uint16_t* count_host,
                                double* shift_host, void* ws, size_t ws_bytes, void* stream, void* copy_stream,
                                void* const* events)
{
    if (!raw_host || !out_host || !events || !copy_stream || copy_stream == stream) return MRED_EINVAL;
    for (int i = 0; i <= MRED_HOST_CHUNKS; ++i)
        if (!events[i]) return MRED_EINVAL;
    int rc = reduce_args_ok(geom, n, MB, MD, MF, ref_index, max_lag, badmask, opts, nullptr, nullptr, nullptr, nullptr);
    if (rc) return rc;
    const Geom g = to_geom(geom);
    if (!ws || !aligned16(ws) || ws_bytes < carve_host(nullptr, g, n).bytes) return MRED_EWORKSPACE;
    const HostWs hw = carve_host(ws, g, n);
    const ReduceWs r = carve_reduce(hw.reduce, g, n);
    cudaStream_t st = static_cast<cudaStream_t>(stream), cs = static_cast<cudaStream_t>(copy_stream);
    const size_t np = (size_t)g.w * g.h, fb = 2 * (size_t)g.W * g.H;
    // chunks of whole calibrate blocks (4 frames), at most MRED_HOST_CHUNKS of them
    int per = (n + MRED_HOST_CHUNKS - 1) / MRED_HOST_CHUNKS;
    per = (per + 3) / 4 * 4;
    // the copies may not start before what `stream` still does with the workspace has finished
    MRED_CUDA_TRY(cudaEventRecord(static_cast<cudaEvent_t>(events[0]), st));
    MRED_CUDA_TRY(cudaStreamWaitEvent(cs, static_cast<cudaEvent_t>(events[0]), 0));
    int ci = 0;
    for (int c0 = 0; c0 < n; c0 += per, ++ci) {
        const int nc = n - c0 < per ? n - c0 : per;
        MRED_CUDA_TRY(cudaMemcpyAsync(reinterpret_cast<char*>(hw.raw) + (size_t)c0 * fb, reinterpret_cast<const char*>(raw_host) + (size_t)c0 * fb,
                                      (size_t)nc * fb, cudaMemcpyHostToDevice, cs));
        cudaEvent_t ev = static_cast<cudaEvent_t>(events[1 + ci]);
        MRED_CUDA_TRY(cudaEventRecord(ev, cs));
        MRED_CUDA_TRY(cudaStreamWaitEvent(st, ev, 0));
        if ((rc = reduce_calibrate(g, hw.raw, n, c0, nc, dark_scale, MB, MD, MF, badmask, r, st))) return rc;
    }
    if ((rc = reduce_finish(g, n, ref_index, max_lag, badmask, fill, opts, hw.out, count_host ? hw.count : nullptr, nullptr,
                            r.shift, nullptr, r, st, nullptr, false)))
        return rc;
    MRED_CUDA_TRY(cudaMemcpyAsync(out_host, hw.out, 4 * np, cudaMemcpyDeviceToHost, st));
    if (count_host) MRED_CUDA_TRY(cudaMemcpyAsync(count_host, hw.count, 2 * np, cudaMemcpyDeviceToHost, st));
    if (shift_host) MRED_CUDA_TRY(cudaMemcpyAsync(shift_host, r.shift, 16 * (size_t)n, cudaMemcpyDeviceToHost, st));
    return MRED_OK;
}

#pragma GCC visibility pop
}  // extern "C"
