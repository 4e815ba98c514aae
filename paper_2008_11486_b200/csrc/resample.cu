// resample.cu -- sub-pixel shift by bicubic (tensor-product natural cubic) spline interpolation
// (O5).
//
// Mathematics.  Along one axis with samples f_0..f_{n-1} the natural-spline coefficients solve
//     c_0 = f_0,  c_{n-1} = f_{n-1},  c_{i-1} + 4 c_i + c_{i+1} = 6 f_i,
// with virtual c_{-1} = 2c_0 - c_1, c_n = 2c_{n-1} - c_{n-2} for the two border intervals.  That is
// exactly the shift-invariant cubic-spline prefilter applied to the samples extended by point
// reflection about both ends, f_{-i} = 2f_0 - f_i, f_{n-1+i} = 2f_{n-1} - f_{n-1-i} (an odd
// sequence about an end has an odd solution, so c_0 = f_0 and c_{-1} = 2c_0 - c_1 come out by
// themselves).  So the kernel extends the image on load and then runs, everywhere, the constant
// recursions   g_i = f_i - a g_{i-1},   c'_i = g_i - a c'_{i+1},   c_i = 6a c'_i,   a = 2 - sqrt(3)
// (the factor 6a is folded into the interpolation weights).  A pure translation evaluates every
// pixel with the same four B-spline weights: m = floor(-s), t = -s - m,
// out(x) = sum_i w_i(t) c_{x+m-1+i}.  Both recursions forget their start like a^d (7e-10 after 16
// steps), so they are restarted from truncated sums >= 16 samples away wherever the data is cut.
// An axis with zero fractional shift uses a = 0 and weights (0, 1, 0, 0): a bit-exact copy.
//
// Kernel design (B200).  One WARP owns one work item = (frame, strip of 208 output columns, band
// of output rows) and needs no barrier and no other warp:
//   * lane l holds the 8 consecutive source samples of one row that lie under its 8 output columns
//     (two aligned 128-bit loads + a register realignment by (x0+m) mod 4 through shuffles);
//   * x pass entirely in registers: 8-step recursions inside the lane, the carry between lanes by
//     two shuffles (lane-to-lane factor a^8, so two lanes = 16 samples of history suffice);
//     3 lanes on either side of the warp are halo, 26 x 8 = 208 columns are kept;
//   * y pass streaming down the rows: causal recursion in registers (one FMA per row), its result
//     kept in a per-lane shared-memory ring of 3 blocks x 8 rows; the anti-causal start value of a
//     block is accumulated on the fly from the 16 rows that follow it (A += (-a)^d g), then the
//     block is swept backwards out of the ring, evaluated with the 4 y weights and stored with
//     128-bit stores.
//   * the hot loop is kept small (one code path, rolled over groups of 4 rows): with 8 warps per SM
//     instruction fetch, not arithmetic, was the first bottleneck (profiles/r1c_resample.md).
// HBM traffic: every input sample read once per strip (halo re-reads hit L2), every output written
// once: 8 B/px algorithmic.
#include "common.cuh"
#include <math.h>

namespace mred {
namespace rs {

constexpr int V = 8;          // samples per lane per row
constexpr int WARPCOLS = 256; // 32 lanes x 8
constexpr int HALO_L = 3;     // halo lanes on the left  (2 for the recursion history, 1 for c_{k-1})
constexpr int HALO_R = 3;     // halo lanes on the right (2 for the look-ahead, 1 for c_{k+1}, c_{k+2})
constexpr int OUTCOLS = (32 - HALO_L - HALO_R) * V;   // 208 output columns per strip
constexpr int RB = 8;         // rows per block of the y pass
constexpr int NRING = 3;      // blocks in the ring: the block being swept trails the loads by 16 rows
constexpr int WARM = 17;      // rows of forward warm-up before the first interval of a band
constexpr int EXT = 40;       // samples beyond an image edge that are given their reflected value (the rest: 0, never used)
constexpr size_t RESAMPLE_TWO_PASS_MAX = (size_t)4 << 30;        // two-kernel route: stacks up to this size ...
constexpr size_t RESAMPLE_TWO_PASS_PLANE = (size_t)16 << 20;     // ... of planes up to this size (measured: 200 x 1024^2 0.83 ms in two kernels; 100 x 4096^2 5.4 ms fused, 6.5 ms in two)
constexpr int Y4_MIN_ROWS = 32;   // shortest band of the 4-column y pass
constexpr float U_INF = 0.26794919243112270647f;   // 2 - sqrt(3)

// One axis of one frame: integer part, weights, identity flag, footprint.
struct Axis {
    int n;        // samples along the axis
    int m;        // floor(-s): source index k = x + m
    int ident;    // 1: zero fractional part -> pure translation (no prefilter, weights 0,1,0,0)
    int lo, hi;   // footprint along this axis, inclusive
    float w[4];   // weights on c_{k-1}, c_k, c_{k+1}, c_{k+2}
};

__device__ __forceinline__ Axis make_axis(int n, double s)
{
    Axis a;
    a.n = n;
    const double ms = -s;
    const double fl = floor(ms);
    const double t = ms - fl;
    a.m = (int)fl;
    a.ident = (t == 0.0) ? 1 : 0;
    if (a.ident) {
        a.w[0] = 0.f; a.w[1] = 1.f; a.w[2] = 0.f; a.w[3] = 0.f;
    } else {
        const double t2 = t * t, t3 = t2 * t, o = 1.0 - t;
        a.w[0] = (float)(o * o * o / 6.0);
        a.w[1] = (float)((3.0 * t3 - 6.0 * t2 + 4.0) / 6.0);
        a.w[2] = (float)((-3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0) / 6.0);
        a.w[3] = (float)(t3 / 6.0);
    }
    axis_footprint(n, s, a.lo, a.hi);
    return a;
}

}  // namespace rs
}  // namespace mred

#include "resample_warp.cuh"
#include "resample_ypass.cuh"
#include "resample_tile.cuh"
#include "resample_pipe.cuh"
#include "resample_lin.cuh"

namespace mred {

// band height for the kernels that carry y state: enough warps for every SM x 8, no band under 64 rows
static int band_rows(long long cols, int h, int min_rows = 64, int warps_per_sm = 8)
{
    long long bands = ((long long)sm_count() * warps_per_sm + cols - 1) / cols;
    const long long maxb = (h + min_rows - 1) / min_rows;
    if (bands > maxb) bands = maxb;
    if (bands < 1) bands = 1;
    int BH = (int)((h + bands - 1) / bands);
    return (BH + 7) / 8 * 8;
}

size_t resample_ws_bytes(int w, int h, int n)
{
    if (rt::tile_route(w, h)) return 0;          // the tiled kernel needs no scratch
    const size_t plane = (size_t)w * h * sizeof(float), b = plane * (size_t)n;
    return (b <= RESAMPLE_TWO_PASS_MAX && plane <= RESAMPLE_TWO_PASS_PLANE) ? b : 0;
}

int launch_resample(const float* in, int n, int w, int h, const double* sx_host, const double* sy_host,
                    const double* dshift_dev, float fill, float* out, int32_t* fp_dev, void* ws, size_t ws_bytes,
                    cudaStream_t st)
{
    HostShifts hs;
    if (!dshift_dev)
        for (int k = 0; k < n; ++k) { hs.s[k][0] = sx_host[k]; hs.s[k][1] = sy_host[k]; }
    int4* fpd = reinterpret_cast<int4*>(fp_dev);
    // planes with 16-byte-aligned rows, at least 256 x 64: the CTA-tiled, TMA-staged pipeline (resample_pipe.cuh, with the
    // row / column code of resample_tile.cuh); smaller or unaligned planes: the warp kernels below
    if (rt::tile_route(w, h)) return rp::launch_resample_pipe(in, n, w, h, hs, dshift_dev, fill, out, fpd, st);
    const int vec = (w % 4 == 0) ? 1 : 0;
    const size_t smem = (size_t)NRING * RB * WARPCOLS * sizeof(float);
    static PerDeviceOnce once;
    int dev;
    if (once.pending(dev)) {
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample<0>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample<2>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        once.mark(dev);
    }
    const size_t need = resample_ws_bytes(w, h, n);
    if (need && ws && ws_bytes >= need) {
        // small stack: x pass and y pass as two kernels, the x-shifted rows stay in the 126 MB L2 in between;
        // neither kernel carries the other's state, so both run with far more parallel work items
        float* tmp = static_cast<float*>(ws);
        const int sx1 = (w + ModeGeom<1>::OUTC - 1) / ModeGeom<1>::OUTC;
        const int slots1 = sm_count() * 16;
        int BH1 = (int)(((long long)h * sx1 * n + slots1 - 1) / slots1);     // one wave of 16 warps per SM
        BH1 = (BH1 + 3) / 4 * 4;
        if (BH1 < 8) BH1 = 8;
        k_resample<1><<<dim3(sx1, (h + BH1 - 1) / BH1, n), 32, 0, st>>>(in, n, w, h, hs, dshift_dev, fill, tmp, nullptr, BH1, vec);
        MRED_LAUNCH_CHECK();
        if (vec) {
            const int bx = (w + 511) / 512;
            const int BH2 = band_rows((long long)bx * 4 * n, h, Y4_MIN_ROWS, 16);
            k_ypass4<<<dim3(bx, (h + BH2 - 1) / BH2, n), 128, 0, st>>>(tmp, n, w, h, hs, dshift_dev, fill, out, fpd, BH2);
        } else {
            const int sx2 = (w + ModeGeom<2>::OUTC - 1) / ModeGeom<2>::OUTC;
            const int BH2 = band_rows((long long)sx2 * n, h, 48);
            k_resample<2><<<dim3(sx2, (h + BH2 - 1) / BH2, n), 32, smem, st>>>(tmp, n, w, h, hs, dshift_dev, fill, out, fpd, BH2, vec);
        }
        MRED_LAUNCH_CHECK();
        return MRED_OK;
    }
    const int strips = (w + OUTCOLS - 1) / OUTCOLS;
    const int BH = band_rows((long long)strips * n, h);
    k_resample<0><<<dim3(strips, (h + BH - 1) / BH, n), 32, smem, st>>>(in, n, w, h, hs, dshift_dev, fill, out, fpd, BH, vec);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

int launch_resample_lin(const float* in, int n, int w, int h, const double* sx_host, const double* sy_host, int interp,
                        float fill, float* out, cudaStream_t st)
{
    rl::LinAxes axes;
    for (int k = 0; k < n; ++k) {
        axes.a[k][0] = rl::make_lin_axis(w, sx_host[k], interp);
        axes.a[k][1] = rl::make_lin_axis(h, sy_host[k], interp);
    }
    if ((h + RL_ROWS - 1) / RL_ROWS > 65535) return MRED_EINVAL;
    k_resample_lin<<<dim3((unsigned)((w + 255) / 256), (unsigned)((h + RL_ROWS - 1) / RL_ROWS), (unsigned)n), 256, 0, st>>>(in, w, h, axes, fill, out);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
