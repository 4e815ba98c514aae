// resample_core.cuh -- per-thread building blocks of the bicubic-spline shift kernel (O5;
// PAPER.md L63, L107, L164, L266).  Plain C++ apart from the MRED_HD decoration, so the same code
// runs inside the CUDA kernel (resample.cu) and, thread by thread, in a host harness.
//
// Mathematics.  Along one axis with samples f_0..f_{n-1} the natural-spline coefficients solve
//     c_0 = f_0,  c_{n-1} = f_{n-1},  c_{i-1} + 4 c_i + c_{i+1} = 6 f_i,
// i.e. (Thomas) g_i = p_i f_i - q_i g_{i-1},  c_i = g_i - u_i c_{i+1}  with
//     u_0 = 0, u_i = 1/(4 - u_{i-1}) -> 2 - sqrt(3);  p_i = 6 u_i, q_i = u_i  (interior rows),
//     p = 1, q = u = 0 on rows 0 and n-1, and p = q = u = 0 outside [0, n) (so c_{-1} = c_n = 0 and
//     the virtual coefficients 2c_0 - c_1, 2c_{n-1} - c_{n-2} are folded into the weights of the
//     two border intervals).
// A pure translation evaluates every pixel with the same four weights: with m = floor(-s),
// t = -s - m:  out(x) = w0 c_{k-1} + w1 c_k + w2 c_{k+1} + w3 c_{k+2},  k = x + m.
// Both recursions forget their start geometrically (|u| = 0.268: 7e-10 after 16 steps), so a line
// is cut into pieces that start from a steady-state guess L = 16 samples early; u_i equals its
// limit to float32 from i = 12 on, so only pieces touching the first 16 samples, the last sample or
// the outside of the line need the per-index coefficients (EDGE path).
#pragma once
#include <math.h>

#ifdef __CUDACC__
#define MRED_HD __host__ __device__ __forceinline__
#else
#define MRED_HD inline
#endif

namespace mred {
namespace rs {

constexpr int R = 32;   // source rows per block of the streaming (y) pass
constexpr int L = 16;   // warm-up / look-ahead length of a truncated recursion
constexpr int S = 32;   // outputs per x-pass task
constexpr int NU = 16;  // indices with their own Thomas multiplier

constexpr float U_INF = 0.26794919243112270647f;     // 2 - sqrt(3)
constexpr float P_INF = 6.0f * 0.26794919243112270647f;
constexpr float G_GUESS = 1.2679491924311227f;        // steady state g/f = 6u/(1+u)
constexpr float C_GUESS = 0.7886751345948129f;        // steady state c/g = 1/(1+u)

MRED_HD float u_table(int i)
{
    // u_0 = 0, u_i = 1/(4 - u_{i-1}), rounded to float32
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

struct Coef { float p, q, u; };

MRED_HD Coef coef(int i, int n, bool ident)
{
    Coef c;
    c.p = 0.f; c.q = 0.f; c.u = 0.f;
    if (i < 0 || i >= n) return c;
    if (ident || i == 0 || i == n - 1) { c.p = 1.f; return c; }
    const float u = i < NU ? u_table(i) : U_INF;
    c.p = 6.0f * u; c.q = u; c.u = u;
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

MRED_HD Axis make_axis(int n, double s)
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
    const double lo = ceil(s), hi = floor((double)(n - 1) + s);
    a.lo = lo > 0.0 ? (lo > (double)n ? n : (int)lo) : 0;
    a.hi = hi < (double)(n - 1) ? (hi < -1.0 ? -1 : (int)hi) : n - 1;
    return a;
}

// value of interval k from the window (c_{k-1}, c_k, c_{k+1}, c_{k+2}); c_{-1} and c_n arrive as 0
// and their virtual values are folded into the neighbours' weights (EDGE only).
template <bool EDGE>
MRED_HD float interp(const Axis& a, int k, float c0, float c1, float c2, float c3)
{
    float w0 = a.w[0], w1 = a.w[1], w2 = a.w[2], w3 = a.w[3];
    if (EDGE) {
        if (k == 0) { w1 = w1 + 2.0f * w0; w2 = w2 - w0; }
        if (k == a.n - 2) { w1 = w1 - w3; w2 = w2 + 2.0f * w3; }
    }
    return fmaf(w3, c3, fmaf(w2, c2, fmaf(w1, c1, w0 * c0)));
}

MRED_HD bool range_is_edge(const Axis& a, int first, int last)
{
    return a.ident || first < NU || last >= a.n - 1;
}

// ---------------------------------------------------------------------------------------------
// x pass, one task = S consecutive outputs of one tile row.
//   trow   : the tile row, trow[j] = source sample (tile_x0 + j), zero outside the image
//   ka     : source index k of the first output; outputs k = ka .. ka+S-1 go to dst[0..S)
// Forward over [ka-1-L, ka+S+1+L], g kept for [ka-1, ka+S+1+L]; backward from the far end.
// ---------------------------------------------------------------------------------------------
template <bool EDGE>
MRED_HD void x_task(const Axis& a, const float* trow, int tile_x0, int ka, float* dst)
{
    constexpr int NG = S + L + 3;
    const int fa = ka - 1 - L;
    const float* f = trow + (fa - tile_x0);
    float g[NG];
    float gp;
    if (EDGE) {
        gp = (fa > 0 && !a.ident) ? G_GUESS * f[0] : 0.f;
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const Coef c = coef(fa + i, a.n, a.ident != 0);
            gp = fmaf(c.p, f[i], -c.q * gp);
        }
#pragma unroll
        for (int i = 0; i < NG; ++i) {
            const Coef c = coef(ka - 1 + i, a.n, a.ident != 0);
            gp = fmaf(c.p, f[L + i], -c.q * gp);
            g[i] = gp;
        }
    } else {
        gp = G_GUESS * f[0];
#pragma unroll
        for (int i = 0; i < L; ++i) gp = fmaf(P_INF, f[i], -U_INF * gp);
#pragma unroll
        for (int i = 0; i < NG; ++i) {
            gp = fmaf(P_INF, f[L + i], -U_INF * gp);
            g[i] = gp;
        }
    }
    float cn = C_GUESS * g[NG - 1];
    float c1 = 0.f, c2 = 0.f, c3 = 0.f;
#pragma unroll
    for (int i = NG - 1; i >= 0; --i) {
        const float u = EDGE ? coef(ka - 1 + i, a.n, a.ident != 0).u : U_INF;
        const float c0 = fmaf(-u, cn, g[i]);
        cn = c0;
        if (i < S) dst[i] = interp<EDGE>(a, ka + i, c0, c1, c2, c3);
        c3 = c2; c2 = c1; c1 = c0;
    }
}

}  // namespace rs
}  // namespace mred
