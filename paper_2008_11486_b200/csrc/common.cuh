// common.cuh -- shared device helpers and host-side checks for libmred (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <stdint.h>
#include <stddef.h>
#include "../../include/mred.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libmred is written for sm_100a (B200) only"
#endif

namespace mred {

struct Geom {
    int W, H, os_x0, os_x1, x0, y0, w, h;
};

inline Geom to_geom(const mred_geom* g) { return Geom{g->W, g->H, g->os_x0, g->os_x1, g->x0, g->y0, g->w, g->h}; }

inline bool geom_ok(const mred_geom* g)
{
    if (!g) return false;
    if (g->W < 1 || g->H < 1 || g->w < 1 || g->h < 1) return false;
    if (g->x0 < 0 || g->y0 < 0 || (int64_t)g->x0 + g->w > g->W || (int64_t)g->y0 + g->h > g->H) return false;
    if (g->os_x0 < 0 || g->os_x1 < g->os_x0 || g->os_x1 > g->W) return false;
    if ((int64_t)g->W * g->H >= (int64_t)1 << 31) return false;   // kernels index one plane with 32 bits
    return true;
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

void set_cuda_error(cudaError_t e);   // api.cu
int sm_count();                       // api.cu: multiprocessors of the current device (cached per device)

// One-time, per-DEVICE setup (function attributes such as the dynamic shared-memory opt-in belong to the device's
// context, not to the process): done[dev] is set once the attributes have been applied on that device.
struct PerDeviceOnce {
    std::atomic<unsigned char> done[64];
    bool pending(int& dev)
    {
        if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { dev = -1; return true; }   // unknown: set every time
        return done[dev].load(std::memory_order_acquire) == 0;
    }
    void mark(int dev) { if (dev >= 0) done[dev].store(1, std::memory_order_release); }
};

#define MRED_CUDA_TRY(expr)                                   \
    do {                                                      \
        cudaError_t _e = (expr);                              \
        if (_e != cudaSuccess) { ::mred::set_cuda_error(_e); return MRED_ECUDA; } \
    } while (0)

#define MRED_LAUNCH_CHECK() MRED_CUDA_TRY(cudaPeekAtLastError())

// Per-frame shifts / footprints handed over from the host by value (no allocation, no copy):
// 255 frames x 16 B = 4080 B of kernel parameter space (sm_70+ allows 32 KB with CUDA >= 12.1).
constexpr float PROF_FIX = 16384.0f;   // fixed-point scale of the profile sums of O4 (2^14: 6e-5 ADU per partial)

struct HostShifts { double s[MRED_MAX_STACK][2]; };       // (sx, sy) as passed to mred_resample
struct HostFootprints { int4 fp[MRED_MAX_STACK]; };       // {x_lo, x_hi, y_lo, y_hi}

#ifdef __CUDACC__
__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ int warp_sum(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum of the overscan pixels of row r of frame f (one THREAD per row: its ~50 loads are independent, so a warp
// keeps 32 rows x 4 sectors in flight; rows are 2W bytes apart, so lanes never share a sector anyway).
__device__ __forceinline__ unsigned int overscan_row_sum(const uint16_t* __restrict__ f, int W, int os_x0, int os_x1, int r)
{
    const uint16_t* row = f + (size_t)r * W;
    unsigned int a = 0;
    int x = os_x0;
    if (((reinterpret_cast<uintptr_t>(row + x)) & 3u) && x < os_x1) a += __ldg(row + x++);     // align to 4 bytes
    const unsigned int* row2 = reinterpret_cast<const unsigned int*>(row + x);
    const int n2 = (os_x1 - x) >> 1;
#pragma unroll 8
    for (int i = 0; i < n2; ++i) { const unsigned int v = __ldg(row2 + i); a += (v & 0xffffu) + (v >> 16); }
    if (x + 2 * n2 < os_x1) a += __ldg(row + x + 2 * n2);
    return a;
}

// footprint of a shift along one axis of length n: [max(0, ceil(s)), min(n-1, floor(n-1+s))]
// (O5).  Same IEEE double operations on host and device.
__host__ __device__ inline void axis_footprint(int n, double s, int& lo, int& hi)
{
    double a = ceil(s), b = floor((double)(n - 1) + s);
    lo = a > 0.0 ? (a > (double)n ? n : (int)a) : 0;
    hi = b < (double)(n - 1) ? (b < -1.0 ? -1 : (int)b) : n - 1;
}
#endif

// launchers implemented in the .cu files (all enqueue on `st`, return mred_status)
int frame_sums_parts(const Geom& g);      // partial sums per frame that launch_frame_sums writes (8 bytes each)
int launch_frame_sums(const uint16_t* raw, const Geom& g, int n, unsigned long long* os_part, void* zero /* nullable */,
                      size_t zero_bytes, cudaStream_t st);
int launch_calibrate(const uint16_t* raw, const Geom& g, int n, float dark_scale, const float* MB, const float* MD,
                     const float* MF, float* out, double* level_out, const unsigned long long* os_part, cudaStream_t st);
int launch_calibrate_prof(const uint16_t* raw, const Geom& g, int n, float dark_scale, const float* MB, const float* MD,
                          const float* MF, float* out, const unsigned long long* os_part, const uint8_t* bad /* nullable */,
                          long long* colsum, long long* rowsum, cudaStream_t st);
int launch_build_masters(const Geom& g, const uint16_t* bias, int nb, const uint16_t* dark, int nd, float t_dark,
                         const uint16_t* flat, int nf, float t_flat, const mred_comb_opts& o, float* MB, float* MD,
                         float* MF, void* ws, cudaStream_t st);
size_t masters_ws_bytes(const Geom& g, int n);
int launch_coadd(const float* stack, int n, int w, int h, const int32_t* fp_host, const int32_t* fp_dev,
                 const mred_comb_opts& o, float* out, uint16_t* count, uint32_t* rejmask, cudaStream_t st);
// stage flags of launch_estimate (chained path): accumulators already cleared / profile sums already accumulated
enum { EST_ZEROED = 1, EST_HAVE_SUMS = 2, EST_SHARED_COUNTS = 4 };   // 4: valid-pixel counts of the mask in frame 0's arrays (launch_mask_counts)
int launch_mask_counts(const uint8_t* bad, int w, int h, int n, void* ws, cudaStream_t st);
int launch_estimate(const float* frames, int n, int w, int h, int ref, int max_lag, const uint8_t* bad,
                    int32_t* ishift, double* shift, void* ws, int flags, int peak /* 0 parabola, 1 log-parabola */, cudaStream_t st);
size_t estimate_ws_bytes(int w, int h, int n);
// launch_estimate on the library's own static device scratch (estimate.cu); MRED_ELIMIT when it is too small
int launch_estimate_static(const float* frames, int n, int w, int h, int ref, int max_lag, const uint8_t* bad,
                           int32_t* ishift, double* shift, int peak, cudaStream_t st);
// the accumulators inside an estimate workspace: what has to be zero before the sums start, and where they are
void estimate_accumulators(void* ws, int w, int h, int n, void** zero, size_t* zero_bytes, long long** colsum, long long** rowsum);
int launch_resample(const float* in, int n, int w, int h, const double* sx_host, const double* sy_host,
                    const double* dshift_dev /* [n][2] (dx,dy): shift = -d */, float fill, float* out,
                    int32_t* fp_dev /* nullable */, void* ws /* nullable */, size_t ws_bytes, cudaStream_t st);
size_t resample_ws_bytes(int w, int h, int n);
int launch_resample_lin(const float* in, int n, int w, int h, const double* sx_host, const double* sy_host, int interp,
                        float fill, float* out, cudaStream_t st);
int launch_fill_bad(float* frames, int n, int w, int h, const uint8_t* bad, void* ws, cudaStream_t st);
size_t fill_ws_bytes(int w, int h);

}  // namespace mred
