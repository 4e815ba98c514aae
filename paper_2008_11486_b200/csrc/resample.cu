// resample.cu -- sub-pixel shift by bicubic (tensor-product natural cubic) spline interpolation
// (O5).
//
// Mathematics.  Along one axis with samples f_0..f_{n-1} the natural-spline coefficients solve
//     c_0 = f_0,  c_{n-1} = f_{n-1},  c_{i-1} + 4 c_i + c_{i+1} = 6 f_i.
// Thomas:  g_i = P_i f_i - Q_i g_{i-1},  c_i = g_i - U_i c_{i+1},  u_0 = 0, u_i = 1/(4 - u_{i-1})
// -> 2 - sqrt(3);  (P, Q, U)_i = (6u_i, u_i, u_i) inside, (1, 0, 0) on rows 0 and n-1 and (0, 0, 0)
// outside [0, n), so c_{-1} = c_n = 0 there and the virtual coefficients 2c_0 - c_1,
// 2c_{n-1} - c_{n-2} are put in by hand.  A pure translation evaluates every pixel with the same
// four B-spline weights: m = floor(-s), t = -s - m, out(x) = sum_i w_i(t) c_{x+m-1+i}.
// Both recursions forget their start like 0.268^d (7e-10 after 16 steps), so they are restarted
// from truncated sums 16 samples away wherever the data is cut into pieces.
//
// Kernel design (B200).  One WARP owns one work item = (frame, strip of 208 output columns, band
// of output rows) and needs no barrier and no other warp:
//   * lane l holds the 8 consecutive source samples of one row that lie under its 8 output columns
//     (two aligned 128-bit loads + a register realignment by (x0+m) mod 4 through shuffles);
//   * x pass entirely in registers: 8-step recursions inside the lane, the carry between lanes by
//     two shuffles (lane-to-lane factor 0.268^8, so two lanes = 16 samples of history suffice);
//     3 lanes on either side of the warp are halo, 26 x 8 = 208 columns are kept;
//   * y pass streaming down the rows: causal recursion in registers (one FMA per row), its result
//     kept in a per-lane shared-memory ring of 3 blocks x 8 rows; the anti-causal start value of a
//     block is accumulated on the fly from the 16 rows that follow it (A += prod(-U) g), then the
//     block is swept backwards out of the ring, evaluated with the 4 y weights and stored with
//     128-bit stores.
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
constexpr float U_INF = 0.26794919243112270647f;   // 2 - sqrt(3)

__host__ __device__ __forceinline__ float u_table(int i)
{
    // u_0 = 0, u_i = 1/(4 - u_{i-1}), rounded to float32; equal to the limit from i = 10 on
    switch (i) {
        case 0: return 0.0f;
        case 1: return 2.5000000000e-01f;
        case 2: return 2.6666666667e-01f;
        case 3: return 2.6785714286e-01f;
        case 4: return 2.6794258373e-01f;
        case 5: return 2.6794871795e-01f;
        case 6: return 2.6794915836e-01f;
        case 7: return 2.6794918999e-01f;
        case 8: return 2.6794919226e-01f;
        case 9: return 2.6794919242e-01f;
        default: return U_INF;
    }
}

struct Coef { float P, nQ, nU; };   // g = P f + nQ g_prev ;  c = g + nU c_next

__device__ __forceinline__ Coef coef(int i, int n, int ident)
{
    Coef c;
    c.P = 0.f; c.nQ = 0.f; c.nU = 0.f;
    if (i < 0 || i >= n) return c;
    if (ident || i == 0 || i == n - 1) { c.P = 1.f; return c; }
    const float u = u_table(i);
    c.P = 6.0f * u; c.nQ = -u; c.nU = -u;
    return c;
}

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
