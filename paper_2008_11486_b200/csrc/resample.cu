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
