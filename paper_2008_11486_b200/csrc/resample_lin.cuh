// resample_lin.cuh -- the cheaper interpolators of SURVEY 8(f) NEXT-2 (PAPER.md L239 suggests them to save time):
// bilinear and nearest-neighbour shifts, same shift sense, validity rule and footprint as the spline (O5, Q28).
// No prefilter, so this is a plain gather: thread = one output pixel, two (one) source samples per axis, rows then columns;
// consecutive threads read consecutive source columns.  HBM traffic 4 + 4 B per pixel; the kernel is bound by it.
#pragma once

namespace mred {
namespace rl {

// one axis of one frame: source index of output i is i + m (and i + m + 1 with weight t); identity axes have t = 0
struct LinAxis { int m; float w0, w1; int lo, hi; };

__device__ __forceinline__ LinAxis make_lin_axis(int n, double s, int interp)
{
    LinAxis a;
    axis_footprint(n, s, a.lo, a.hi);
    const double ms = -s, fl = floor(ms), t = ms - fl;
    if (t == 0.0) { a.m = (int)fl; a.w0 = 1.f; a.w1 = 0.f; }                                    // integer shift: a copy
    else if (interp == MRED_INTERP_BILINEAR) { a.m = (int)fl; a.w0 = (float)(1.0 - t); a.w1 = (float)t; }
    else { a.m = (int)floor(ms + 0.5); a.w0 = 1.f; a.w1 = 0.f; }                                 // nearest: floor(u + 1/2)
    return a;
}

}  // namespace rl

// grid (ceil(w * h / 256), n), block 256
__global__ void __launch_bounds__(256) k_resample_lin(const float* __restrict__ in, int w, int h,
                                                      const __grid_constant__ HostShifts hs, int interp, float fill,
                                                      float* __restrict__ out)
{
    using namespace rl;
    const int k = blockIdx.y;
    const size_t np = (size_t)w * h;
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const LinAxis ax = make_lin_axis(w, hs.s[k][0], interp), ay = make_lin_axis(h, hs.s[k][1], interp);
    const int y = (int)((unsigned)p / (unsigned)w), x = (int)((unsigned)p - (unsigned)y * (unsigned)w);
    float v = fill;
    if (x >= ax.lo && x <= ax.hi && y >= ay.lo && y <= ay.hi) {
        // inside the footprint 0 <= x + m <= w - 1; the second tap is clamped where its weight is 0 anyway
        const int x0 = min(max(x + ax.m, 0), w - 1), x1 = min(x0 + 1, w - 1);
        const int y0 = min(max(y + ay.m, 0), h - 1), y1 = min(y0 + 1, h - 1);
        const float* f = in + (size_t)k * np;
        const float* r0 = f + (size_t)y0 * w;
        const float r0v = ax.w1 != 0.f ? fmaf(ax.w1, __ldg(r0 + x1), ax.w0 * __ldg(r0 + x0)) : __ldg(r0 + x0);
        if (ay.w1 != 0.f) {
            const float* r1 = f + (size_t)y1 * w;
            const float r1v = ax.w1 != 0.f ? fmaf(ax.w1, __ldg(r1 + x1), ax.w0 * __ldg(r1 + x0)) : __ldg(r1 + x0);
            v = fmaf(ay.w1, r1v, ay.w0 * r0v);
        } else {
            v = r0v;
        }
    }
    out[(size_t)k * np + p] = v;
}

}  // namespace mred
