/*
 * mred.h -- C ABI of the B200 (sm_100a) image-reduction hot path of arXiv 2008.11486
 *           ("GPU-accelerated Image Reduction Pipeline", PAPER.md).
 *
 * The calls follow the paper's problem statement: overscan cutout, bias subtraction, dark
 * subtraction, flat fielding, alignment by bicubic-spline sub-pixel shift and sigma-clipped-mean
 * co-adding, plus the two steps the north star adds around them (master
 * frame construction, image-based offset estimation).  The paper prints no formulas; the exact
 * definition of every result is DESIGN.md section 3 (readings O1-O6, Q1-Q24).
 *
 * Conventions (all calls):
 *  - Every array pointer is DEVICE memory owned by the caller unless the comment says "host".
 *    The library never allocates, frees or retains a pointer and keeps no global mutable state
 *    (apart from the last CUDA error code, see mred_last_cuda_error, and the static device scratch of
 *    mred_estimate_shifts_static, which only that call touches); calls on different streams are
 *    independent.
 *  - Work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *    stream) and the call returns WITHOUT synchronising, except mred_reduce_host which
 *    returns after its device->host copies are enqueued (also not synchronised).
 *  - Device array pointers must be 16-byte aligned (MRED_EALIGN otherwise).
 *  - Layout: raw frames uint16 [n][H][W], x fastest; image planes [h][w], x fastest; stacks
 *    [n][h][w].  Origin lower-left, X horizontal, Y vertical; row y=0 is first
 *    in memory.
 *  - Return value: MRED_OK (0) or a negative mred_status; never throws, never aborts.  On error
 *    nothing has been enqueued unless the status is MRED_ECUDA.
 *  - `ws` is caller-owned device scratch of at least mred_workspace_bytes(call, geom, n) bytes,
 *    16-byte aligned; its contents are undefined afterwards and it must not be shared by calls
 *    that may run concurrently.
 *  - Frame counts: 1 <= n <= MRED_MAX_STACK (255) for every per-pixel-column call.
 *  - One plane (W x H raw, w x h image) must hold fewer than 2^31 pixels (MRED_EINVAL otherwise).
 */
#ifndef MRED_H
#define MRED_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MRED_MAX_STACK 255
#define MRED_MAX_LAG 256
#define MRED_MAX_PROFILE 4096 /* longest row / column mred_estimate_shifts and mred_reduce* accept */
#define MRED_HOST_CHUNKS 4 /* pieces mred_reduce_host_overlapped copies the raw stack in */
#define MRED_STATIC_SCRATCH_BYTES (4u << 20) /* the built-in scratch of mred_estimate_shifts_static, per device */

typedef struct {
    int32_t W, H;         /* raw frame size, x fastest (1074 x 1024 incl. overscan)   */
    int32_t os_x0, os_x1; /* overscan columns [os_x0, os_x1) over all H rows; equal -> level = 0     */
    int32_t x0, y0, w, h; /* image rectangle kept by the overscan cutout               */
} mred_geom;

typedef enum { MRED_MEDIAN = 0, MRED_MEAN = 1, MRED_SIGCLIP = 2,
               MRED_MINMAX = 3, MRED_MEDCLIP = 4 /* 3, 4: mred_coadd and mred_reduce* only */ } mred_combine;
typedef enum { MRED_PEAK_PARABOLA = 0, MRED_PEAK_GAUSSIAN = 1 } mred_peak;
typedef enum { MRED_INTERP_SPLINE = 0, MRED_INTERP_BILINEAR = 1, MRED_INTERP_NEAREST = 2 } mred_interp;

typedef struct {
    int32_t mode;     /* mred_combine                                                             */
    float ksigma;     /* clip threshold in sigma (SIGCLIP only), e.g. 3.0                          */
    int32_t max_iter; /* maximum number of clip passes (SIGCLIP only), e.g. 3; 0 = plain mean      */
} mred_comb_opts;

typedef enum {
    MRED_OK = 0,
    MRED_EINVAL = -1,     /* null pointer, bad shape/geometry/count/option                          */
    MRED_EALIGN = -2,     /* a device pointer is not 16-byte aligned                                */
    MRED_EWORKSPACE = -3, /* ws is null or smaller than mred_workspace_bytes()                      */
    MRED_ECUDA = -4,      /* a CUDA runtime call failed; see mred_last_cuda_error()                 */
    MRED_ELIMIT = -5      /* the problem needs more scratch than a no-allocation entry point holds  */
} mred_status;

typedef enum {
    MRED_CALL_BUILD_MASTERS = 0,
    MRED_CALL_CALIBRATE = 1,
    MRED_CALL_ESTIMATE_SHIFTS = 2,
    MRED_CALL_RESAMPLE = 3,
    MRED_CALL_COADD = 4,
    MRED_CALL_REDUCE = 5,
    MRED_CALL_FILL_BAD = 6
} mred_call;

/*
 * Master bias / dark / flat (O2; the paper uses masters but does not describe their
 * construction).  With L_k the overscan level of each input frame (O1: exact
 * integer mean of its overscan pixels) and comb = per-pixel median / mean / sigma-clipped mean:
 *     MB = comb_k(B_k - L_k)
 *     MD = comb_k(D_k - L_k - MB)                                   [ADU at t_dark]
 *     G_k = F_k - L_k - MB - (t_flat/t_dark) MD ,  MF = comb_k(G_k/<G_k>) / <comb_k(..)>,  <MF> = 1
 * bias/dark/flat: uint16 [nb|nd|nf][H][W].  MB, MD, MF: float32 [h][w] outputs.
 */
int mred_build_masters(const mred_geom *geom, const uint16_t *bias, int nb, const uint16_t *dark, int nd,
                       float t_dark, const uint16_t *flat, int nf, float t_flat, const mred_comb_opts *opts,
                       float *MB, float *MD, float *MF, void *ws, size_t ws_bytes, void *stream);

/*
 * Overscan cutout + level subtraction + bias/dark subtraction + flat fielding in one pass over
 * the uint16 input (O1, O3):
 *     out_k = (raw_k - L_k - MB - dark_scale * MD) / MF   on the image rectangle;  MF <= 0 or
 *     non-finite -> 0.   dark_scale = t_sci / t_dark.
 * raw: uint16 [n][H][W]; out: float32 [n][h][w]; level_out: float64 [n] (device, nullable)
 * receives L_k.  1 <= n <= 524 280 (8 x 65535; MRED_EINVAL beyond).  ws holds ceil(H/256)
 * partial overscan sums per frame (mred_workspace_bytes).
 */
int mred_calibrate(const mred_geom *geom, const uint16_t *raw, int n, float dark_scale, const float *MB,
                   const float *MD, const float *MF, float *out, double *level_out, void *ws, size_t ws_bytes,
                   void *stream);

/*
 * Bad-pixel fill ("bad pixel masking", Table 6; O7, reading Q25), in place on a float32
 * stack, e.g. between mred_calibrate and mred_resample: every pixel with badmask != 0 becomes the linear interpolation
 * between the nearest good pixels of the same frame along the axis with the shorter gap (ties: x), else the nearest
 * one-sided good neighbour (order left, right, below, above), else 0.  Good pixels are never changed and filled values
 * are never used as sources.  frames: float32 [n][h][w]; badmask: uint8 [h][w] (the same for every frame).
 * 1 <= n <= 65535; ws: mred_workspace_bytes(MRED_CALL_FILL_BAD, ..) bytes (a list entry per pixel of the plane).
 */
int mred_fill_bad(float *frames, int n, int w, int h, const uint8_t *badmask, void *ws, size_t ws_bytes, void *stream);

/*
 * Per-frame offset relative to frame `ref_index` from marginal profiles (O4; replaces
 * the WCS-header path of PAPER.md L69/L99): mean row/column profiles over pixels with
 * badmask == 0, median-subtracted, 1-D cross-correlation over lags -max_lag..max_lag, integer
 * argmax + 3-point parabola.  (dx, dy) is the displacement of frame k's CONTENT relative to the
 * reference: a source at (x, y) in the reference sits at (x+dx, y+dy) in frame k.
 * frames: float32 [n][h][w]; badmask: uint8 [h][w], nullable; ishift: int32 [n][2] (ix, iy);
 * shift: float64 [n][2] (dx, dy); both device.  0 <= max_lag <= MRED_MAX_LAG, max_lag < min(w,h).
 * w, h <= MRED_MAX_PROFILE (a whole profile is sorted in shared memory); MRED_EINVAL beyond.
 */
int mred_estimate_shifts(const float *frames, int n, int w, int h, int ref_index, int max_lag,
                         const uint8_t *badmask, int32_t *ishift, double *shift, void *ws, size_t ws_bytes,
                         void *stream);

/*
 * mred_estimate_shifts with a choice of the sub-pixel estimator (Q27): peak =
 * MRED_PEAK_PARABOLA is mred_estimate_shifts; MRED_PEAK_GAUSSIAN fits the parabola to the LOGARITHMS of the three
 * correlation samples around the maximum (exact for a Gaussian peak), and falls back to the plain parabola where one of
 * them is not positive.  Integer part, tie rule and everything else are unchanged.
 */
int mred_estimate_shifts_peak(const float *frames, int n, int w, int h, int ref_index, int max_lag,
                              const uint8_t *badmask, int peak, int32_t *ishift, double *shift, void *ws,
                              size_t ws_bytes, void *stream);

/*
 * mred_estimate_shifts_peak for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no workspace argument.  The scratch is a static device array of
 * MRED_STATIC_SCRATCH_BYTES (4 MiB) inside the library, held by every device that loads the library until the process
 * exits; the call itself calls no cudaMalloc / cudaFree and no allocating library routine.  Results are those of
 * mred_estimate_shifts_peak, bit for bit (same kernels, O4).
 * Limit: mred_workspace_bytes(MRED_CALL_ESTIMATE_SHIFTS, {w, h}, n) <= MRED_STATIC_SCRATCH_BYTES, else MRED_ELIMIT and
 * nothing is enqueued (64 frames of 1024 x 1024 need 3.1 MiB; 100 frames of 4096 x 4096 do not fit).
 * Every call on a device shares the one array, which keeps the previous call's contents: the call clears what has to
 * start at zero (on `stream`, before its kernels), and calls that may OVERLAP on the GPU (different streams, or graph
 * branches) race on it -- serialise them.  The first call on a device looks up the array's device address
 * (cudaGetSymbolAddress, kept per device); make that first call outside a stream capture.
 */
int mred_estimate_shifts_static(const float *frames, int n, int w, int h, int ref_index, int max_lag,
                                const uint8_t *badmask, int peak, int32_t *ishift, double *shift, void *stream);

/*
 * Sub-pixel shift by bicubic (tensor-product natural cubic) spline interpolation (PAPER.md L63,
 * L107, L164, L266; O5):  out_k(x, y) = spline_k(x - sx[k], y - sy[k]); pixels whose
 * source lies outside the frame get `fill`.  An axis whose shift has zero fractional part is a
 * pure integer translation, so (0, 0) is the bit-exact identity.  To align frame k onto the
 * reference use (sx, sy) = (-dx, -dy) of mred_estimate_shifts.
 * in/out: float32 [n][h][w] (must not overlap); sx, sy: HOST float64 [n];
 * footprint: HOST int32 [n][4] output {x_lo, x_hi, y_lo, y_hi} inclusive (nullable) --
 * written before the call returns.  w, h >= 4.  ws is optional: with at least
 * mred_workspace_bytes(MRED_CALL_RESAMPLE, ..) bytes (non-zero only for planes up to 16 MB and stacks up to 4 GB) the
 * shift runs as an x kernel and a y kernel with the intermediate held in ws; without it, as one fused kernel.
 * Both routes give the same result to float32 rounding.
 */
int mred_resample(const float *in, int n, int w, int h, const double *sx, const double *sy, float fill,
                  float *out, int32_t *footprint, void *ws, size_t ws_bytes, void *stream);

/*
 * mred_resample with a choice of the interpolator (PAPER.md L239 suggests cheaper ones; Q28):
 * MRED_INTERP_SPLINE is mred_resample (without workspace); MRED_INTERP_BILINEAR takes the two nearest source samples per axis
 * with weights (1 - t, t), MRED_INTERP_NEAREST the sample floor(u + 1/2), u = x - sx; no prefilter.  Shift sense, validity
 * (0 <= u <= n - 1 on both axes, else `fill`), footprint and the bit-exact copy for integer shifts are those of the spline.
 * sx, sy, footprint: HOST.  w, h >= 2.
 */
int mred_resample_interp(const float *in, int n, int w, int h, const double *sx, const double *sy, float fill,
                         int interp, float *out, int32_t *footprint, void *stream);

/*
 * Per-pixel combine along the stack axis (O6) over the
 * frames whose footprint contains the pixel: median, mean, or ksigma-clipped mean (mean-centred,
 * population sigma, keep |v-mu| <= k sigma, <= max_iter passes, early stop).
 * stack: float32 [n][h][w]; footprint: HOST int32 [n][4] (nullable = every frame covers every
 * pixel); out: float32 [h][w]; count: uint16 [h][w] number of frames used (nullable);
 * rejmask: uint32 [ceil(n/32)][h][w], bit k%32 of word k/32 set iff frame k was NOT used
 * (nullable).  No covering frame -> value 0, count 0.  mode MRED_MINMAX (Q26; mred_coadd and
 * mred_reduce* only): the mean without one minimum and one maximum (first occurrences in frame order; fewer than 3 values:
 * the plain mean).  mode MRED_MEDCLIP (NEXT-2, Q29): the k-sigma clip centred on the MEDIAN of the survivors, sigma = their
 * r.m.s. about it (clips from N = 10 at k = 3, where the mean-centred clip cannot); result = mean of the survivors.
 */
int mred_coadd(const float *stack, int n, int w, int h, const int32_t *footprint, const mred_comb_opts *opts,
               float *out, uint16_t *count, uint32_t *rejmask, void *stream);

/*
 * The whole science path for one group, device-resident and chained without host round trips:
 * calibrate -> estimate_shifts (vs ref_index) -> resample by (-dx, -dy) -> coadd.
 * The marginal profiles of estimate_shifts are summed inside the calibrate kernel (same definition,
 * DESIGN.md O4, masked pixels left out; the calibrated stack is not read a second time).
 * raw: uint16 [n][H][W].  shift_out: float64 [n][2] device (nullable) receives (dx, dy);
 * footprint_out: int32 [n][4] device (nullable).  Other arguments as in the single calls; in particular
 * 4 <= w, h <= MRED_MAX_PROFILE and n <= MRED_MAX_STACK.
 */
int mred_reduce(const mred_geom *geom, const uint16_t *raw, int n, float dark_scale, const float *MB,
                const float *MD, const float *MF, int ref_index, int max_lag, const uint8_t *badmask,
                float fill, const mred_comb_opts *opts, float *out, uint16_t *count, uint32_t *rejmask,
                double *shift_out, int32_t *footprint_out, void *ws, size_t ws_bytes, void *stream);

/*
 * mred_reduce with stage markers: events is a HOST array of 5 cudaEvent_t (as void*, entries nullable)
 * recorded on `stream` before calibrate and after calibrate, estimate_shifts, resample and coadd, so a
 * caller can time each stage of the chained pass on the device.  events == NULL is mred_reduce.
 */
int mred_reduce_staged(const mred_geom *geom, const uint16_t *raw, int n, float dark_scale, const float *MB,
                       const float *MD, const float *MF, int ref_index, int max_lag, const uint8_t *badmask,
                       float fill, const mred_comb_opts *opts, float *out, uint16_t *count, uint32_t *rejmask,
                       double *shift_out, int32_t *footprint_out, void *ws, size_t ws_bytes, void *stream,
                       void *const *events);

/*
 * mred_reduce with the bad-pixel fill (mred_fill_bad, O7) applied to the calibrated stack before it is
 * resampled: calibrate -> estimate_shifts (masked pixels left out of the profiles) -> fill -> resample -> coadd.
 * badmask must not be NULL.  Same workspace as mred_reduce.
 */
int mred_reduce_filled(const mred_geom *geom, const uint16_t *raw, int n, float dark_scale, const float *MB,
                       const float *MD, const float *MF, int ref_index, int max_lag, const uint8_t *badmask,
                       float fill, const mred_comb_opts *opts, float *out, uint16_t *count, uint32_t *rejmask,
                       double *shift_out, int32_t *footprint_out, void *ws, size_t ws_bytes, void *stream);

/*
 * Same as mred_reduce with HOST input and output buffers: raw_host (uint16 [n][H][W], ideally
 * pinned) is copied to the device inside the call, out_host (float32 [h][w]), count_host
 * (uint16 [h][w], nullable) and shift_host (float64 [n][2], nullable) are copied back; all on
 * `stream`, nothing synchronised.  Masters and badmask stay device pointers.  ws needs
 * mred_workspace_bytes(MRED_CALL_REDUCE, geom, n) + the staging the call adds itself, i.e. use
 * mred_reduce_host_workspace_bytes().
 */
int mred_reduce_host(const mred_geom *geom, const uint16_t *raw_host, int n, float dark_scale, const float *MB,
                     const float *MD, const float *MF, int ref_index, int max_lag, const uint8_t *badmask,
                     float fill, const mred_comb_opts *opts, float *out_host, uint16_t *count_host,
                     double *shift_host, void *ws, size_t ws_bytes, void *stream);

/*
 * mred_reduce_host with the host->device copy OVERLAPPED with the calibration inside the call (PAPER.md
 * Table 6: transfers and I/O are 64 % of the paper's run): the raw stack is copied in up to MRED_HOST_CHUNKS pieces of
 * whole frames on `copy_stream`, and the overscan levels, the calibration and the profile sums of each piece are enqueued
 * on `stream` behind an event of its copy, so piece c is calibrated while piece c + 1 is still on the bus; estimate_shifts,
 * resample and coadd follow on `stream` as in mred_reduce.  Results are bit-identical to mred_reduce_host.
 * The library creates nothing: copy_stream (a second cudaStream_t, != stream) and events (HOST array of MRED_HOST_CHUNKS + 1
 * cudaEvent_t, timing may be disabled) come from the caller and may be reused by the next call.  On return everything is
 * enqueued; `stream` has been made to wait for every copy, so synchronising `stream` also covers copy_stream's work.
 * raw_host should be pinned memory (pageable memory makes the copies synchronous).  Same workspace as mred_reduce_host.
 */
int mred_reduce_host_overlapped(const mred_geom *geom, const uint16_t *raw_host, int n, float dark_scale, const float *MB,
                                const float *MD, const float *MF, int ref_index, int max_lag, const uint8_t *badmask,
                                float fill, const mred_comb_opts *opts, float *out_host, uint16_t *count_host,
                                double *shift_host, void *ws, size_t ws_bytes, void *stream, void *copy_stream,
                                void *const *events);

/*
 * Where mred_reduce / mred_reduce_staged leave their two intermediate stacks inside `ws` (byte offsets from ws):
 * the calibrated stack (O3) and the registered stack (O5), both float32 [n][h][w].  They stay valid
 * until ws is used again.  For inspection and stage-by-stage checks; MRED_EINVAL on a null pointer or bad geometry.
 */
int mred_reduce_workspace_views(const mred_geom *geom, int n, size_t *calibrated_offset, size_t *registered_offset);

/* Scratch size for one call (call = mred_call).  geom may be NULL for the calls that take w, h
 * directly, in which case pass them through a mred_geom with only w, h set. */
size_t mred_workspace_bytes(int call, const mred_geom *geom, int n);
size_t mred_reduce_host_workspace_bytes(const mred_geom *geom, int n);

const char *mred_strerror(int status);
int mred_last_cuda_error(void); /* cudaError_t of the most recent failing runtime call, else 0 */
const char *mred_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MRED_H */
