// resample_lin.cuh -- the cheaper interpolators of SURVEY 8(f) NEXT-2 (PAPER.md L239 suggests them to save time):
// bilinear and nearest-neighbour shifts, same shift sense, validity rule and footprint as the spline (O5, Q28).
// No prefilter, so this is a plain gather: two (one) source samples per axis, rows then columns.  HBM traffic 4 + 4 B per pixel.
#pragma once

namespace mred {
namespace rl {

// one axis of one frame: source index of output i is i + m (and i + m + 1 with weight t); identity axes have t = 0
struct LinAxis { int m; float w0, w1; int lo, hi; };

__host__ __device__ inline LinAxis make_lin_axis(int n, double s, int interp)
{
    LinAxis a;
    axis_footprint(n, s, a.lo, a.hi);
    const double ms = -s, fl = floor(ms), t = ms - fl;
    if (t == 0.0) { a.m = (int)fl; a.w0 = 1.f; a.w1 = 0.f; }                                    // integer shift: a copy
    else if (interp == MRED_INTERP_BILINEAR) { a.m = (int)fl; a.w0 = (float)(1.0 - t); a.w1 = (float)t; }
    else { a.m = (int)floor(ms + 0.5); a.w0 = 1.f; a.w1 = 0.f; }                                 // nearest: floor(u + 1/2)
    return a;
}

// the axes of every frame, set up on the host (the shifts of mred_resample_interp are host arrays) and handed over by
// value: 10 KB of kernel parameter space
struct LinAxes { LinAxis a[MRED_MAX_STACK][2]; };

}  // namespace rl

// grid (ceil(w / 256), ceil(h / 8), n), block 256: thread = one output column of a strip of 8 rows.  A warp reads 32
// consecutive source samples of a row (one coalesced 128-byte request), the second x tap is the neighbouring lane's sample
// (one shuffle; lane 31 loads it), and the 9 source rows of the strip serve its 8 output rows: 9 loads per 8 pixels, where
// a thread per pixel issued 4 per pixel.  The frames' axes (float64 floor and weights) come ready from the host: computed by
// every thread for its own pixel they were most of the first version of this kernel (398 us per 60 x 1024^2 against the
// spline kernel's 137 us), and set up per block behind a barrier they still cost every block a microsecond.
constexpr int RL_ROWS = 8;

__global__ void __launch_bounds__(256) k_resample_lin(const float* __restrict__ in, int w, int h,
                                                      const __grid_constant__ rl::LinAxes axes, float fill,
                                                      float* __restrict__ out)
{
    using namespace rl;
    const int k = blockIdx.z;
    const LinAxis ax = axes.a[k][0], ay = axes.a[k][1];
    const size_t np = (size_t)w * h;
    const int lane = threadIdx.x & 31;
    const int x = blockIdx.x * blockDim.x + threadIdx.x, yb = blockIdx.y * RL_ROWS;
    const float* f = in + (size_t)k * np;
    // inside the footprint 0 <= x + m <= w - 1; outside it the clamped samples are never used
    const int x0 = min(max(x + ax.m, 0), w - 1), x1 = min(x0 + 1, w - 1);
    const bool xtap = ax.w1 != 0.f, ytap = ay.w1 != 0.f;
    // every load of the thread first (the fifth / ninth row only feeds the second y tap; lane 31's second x tap is a
    // predicated load, not a branch, so that nothing separates the loads), then the shuffles and the arithmetic
    float hrow[RL_ROWS + 1], edge[RL_ROWS + 1];
#pragma unroll
    for (int r = 0; r < RL_ROWS + 1; ++r) {
        hrow[r] = 0.f;
        edge[r] = 0.f;
        if (r == RL_ROWS && !ytap) continue;                      // block-uniform
        const int ys = min(max(yb + r + ay.m, 0), h - 1);
        const float* row = f + (size_t)ys * w;
        hrow[r] = __ldg(row + x0);
        if (xtap && lane == 31) edge[r] = __ldg(row + x1);
    }
    if (xtap) {                                                   // block-uniform
#pragma unroll
        for (int r = 0; r < RL_ROWS + 1; ++r) {
            float b = __shfl_down_sync(0xffffffffu, hrow[r], 1);
            b = lane == 31 ? edge[r] : b;
            hrow[r] = fmaf(ax.w1, b, ax.w0 * hrow[r]);
        }
    }
    if (x >= w) return;
    const bool xin = x >= ax.lo && x <= ax.hi;
    float* o = out + (size_t)k * np + (size_t)yb * w + x;
#pragma unroll
    for (int r = 0; r < RL_ROWS; ++r) {
        const int y = yb + r;
        if (y >= h) break;
        float v = ytap ? fmaf(ay.w1, hrow[r + 1], ay.w0 * hrow[r]) : hrow[r];
        if (!(xin && y >= ay.lo && y <= ay.hi)) v = fill;
        __stcs(o + (size_t)r * w, v);
    }
}

}  // namespace mred
