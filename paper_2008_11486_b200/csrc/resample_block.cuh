// resample_block.cuh -- the per-CTA program of the spline-shift kernel, written as per-thread
// phase functions (load / x pass / y pass) over a block context, so that resample.cu runs them
// with __syncthreads() in between and a host harness can run them thread by thread.
//
// CTA = (frame, strip of TW output columns, band of output rows).  It streams the source rows of
// its band top to bottom in blocks of R rows:
//   load  : R x (TW + 2L + 3) source samples -> shared tile (zero outside the image)
//   x pass: per (row, S-column segment) task: truncated Thomas recursion along x in registers,
//           4-tap evaluation -> shared T[R][TW] (x-shifted rows)
//   y pass: one thread per column: the forward recursion runs continuously down the band; the
//           backward recursion restarts every block from L rows of look-ahead, so outputs trail the
//           loads by L + 2 rows; 4-tap evaluation; coalesced store of R output rows.
// HBM traffic: each input sample read once per strip (+ (2L+3)/TW halo, L2 hits) and each output
// written once: 8 B/px algorithmic.
#pragma once
#include "resample_core.cuh"

namespace mred {
namespace rs {

struct YState {
    float gw[R + L];   // g of source rows [rb - L, rb + R)
    float gp;          // g of the last row processed by the forward recursion
    float s1, s2, s3;  // c of rows rb-L-1, rb-L-2, rb-L-3 (finalised by the previous block)
};

MRED_HD void y_state_init(YState& st)
{
#pragma unroll
    for (int i = 0; i < R + L; ++i) st.gw[i] = 0.f;
    st.gp = 0.f; st.s1 = 0.f; st.s2 = 0.f; st.s3 = 0.f;
}

// One block of the y pass for one column.  tcol[i * tpitch] = x-shifted sample of source row rb + i.
// emit(k, value) is called for the R intervals k = rb-L-2 .. rb+R-L-3.
template <bool EDGE, class Emit>
MRED_HD void y_block(const Axis& a, YState& st, const float* tcol, int tpitch, int rb, bool first, Emit& emit)
{
#pragma unroll
    for (int i = 0; i < L; ++i) st.gw[i] = st.gw[R + i];
    float gp = st.gp;
    if (first) gp = (rb > 0 && !a.ident) ? G_GUESS * tcol[0] : 0.f;
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const float f = tcol[i * tpitch];
        if (EDGE) {
            const Coef c = coef(rb + i, a.n, a.ident != 0);
            gp = fmaf(c.p, f, -c.q * gp);
        } else {
            gp = fmaf(P_INF, f, -U_INF * gp);
        }
        st.gw[L + i] = gp;
    }
    st.gp = gp;
    float cn = C_GUESS * gp;
    float c1 = 0.f, c2 = 0.f, c3 = 0.f, n1 = 0.f, n2 = 0.f, n3 = 0.f;
#pragma unroll
    for (int i = R + L - 1; i >= 0; --i) {
        const int row = rb - L + i;
        const float u = EDGE ? coef(row, a.n, a.ident != 0).u : U_INF;
        const float c0 = fmaf(-u, cn, st.gw[i]);
        cn = c0;
        if (i <= R - 4) emit(row + 1, interp<EDGE>(a, row + 1, c0, c1, c2, c3));
        if (i == R - 1) n1 = c0;
        if (i == R - 2) n2 = c0;
        if (i == R - 3) n3 = c0;
        c3 = c2; c2 = c1; c1 = c0;
    }
    // c1, c2, c3 now hold rows rb-L, rb-L+1, rb-L+2; finish the three intervals that straddle blocks
    emit(rb - L, interp<EDGE>(a, rb - L, st.s1, c1, c2, c3));
    emit(rb - L - 1, interp<EDGE>(a, rb - L - 1, st.s2, st.s1, c1, c2));
    emit(rb - L - 2, interp<EDGE>(a, rb - L - 2, st.s3, st.s2, st.s1, c1));
    st.s1 = n1; st.s2 = n2; st.s3 = n3;
}

// ---------------------------------------------------------------------------------------------
template <int TW>
struct BlockCfg {
    static constexpr int NSEG = TW / S;
    static constexpr int TWIN = TW + 2 * L + 3;
    static constexpr int PITCH_IN = (TWIN % 2 == 0) ? TWIN + 1 : TWIN;   // odd: row-per-lane reads are conflict-free
    static constexpr int PITCH_T = TW + 1;
    static constexpr int TILE_FLOATS = R * PITCH_IN;
    static constexpr int T_FLOATS = R * PITCH_T;
};

struct BlockCtx {
    const float* in;   // frame k input plane
    float* out;        // frame k output plane
    int w, h;
    Axis ax, ay;
    int X0;            // first output column of the strip
    int ya, yb;        // output rows [ya, yb) of the band
    int tile_x0;       // source column of tile column 0
    int r_begin;       // first source row of block 0
    int nblocks;
    float fill;
    float* tile;       // shared [R][PITCH_IN]
    float* T;          // shared [R][PITCH_T]
};

template <int TW>
MRED_HD void block_setup(BlockCtx& c, const float* in, float* out, int w, int h, double sx, double sy, int strip,
                         int band, int BH, float fill, float* tile, float* T)
{
    c.in = in; c.out = out; c.w = w; c.h = h; c.fill = fill; c.tile = tile; c.T = T;
    c.ax = make_axis(w, sx);
    c.ay = make_axis(h, sy);
    c.X0 = strip * TW;
    c.ya = band * BH;
    c.yb = c.ya + BH < h ? c.ya + BH : h;
    c.tile_x0 = c.X0 + c.ax.m - 1 - L;
    const int kA = c.ya + c.ay.m, kB = c.yb + c.ay.m;
    c.r_begin = kA - R + L + 2;
    c.nblocks = 1 + (kB - kA + R - 1) / R;
}

template <int TW>
MRED_HD void load_phase(const BlockCtx& c, int tid, int nthreads, int rb)
{
    typedef BlockCfg<TW> Cfg;
    for (int idx = tid; idx < R * Cfg::TWIN; idx += nthreads) {
        const int r = idx / Cfg::TWIN, cc = idx - r * Cfg::TWIN;
        const int row = rb + r, col = c.tile_x0 + cc;
        float v = 0.f;
        if (row >= 0 && row < c.h && col >= 0 && col < c.w) v = c.in[(size_t)row * c.w + col];
        c.tile[r * Cfg::PITCH_IN + cc] = v;
    }
}

template <int TW>
MRED_HD void x_phase(const BlockCtx& c, int tid, int nthreads)
{
    typedef BlockCfg<TW> Cfg;
    for (int t = tid; t < Cfg::NSEG * R; t += nthreads) {
        const int seg = t / R, row = t - seg * R;
        const int ka = c.X0 + c.ax.m + seg * S;
        const float* trow = c.tile + row * Cfg::PITCH_IN;
        float* dst = c.T + row * Cfg::PITCH_T + seg * S;
        if (range_is_edge(c.ax, ka - 1 - L, ka + S + 1 + L)) x_task<true>(c.ax, trow, c.tile_x0, ka, dst);
        else x_task<false>(c.ax, trow, c.tile_x0, ka, dst);
    }
}

struct EmitStore {
    float* out;
    int w, x, my, ya, yb, ylo, yhi;
    bool xok;
    float fill;
    MRED_HD void operator()(int k, float v) const
    {
        const int y = k - my;
        if (y >= ya && y < yb) out[(size_t)y * w + x] = (xok && y >= ylo && y <= yhi) ? v : fill;
    }
};

template <int TW>
MRED_HD void y_phase(const BlockCtx& c, YState& st, int tid, int rb, bool first)
{
    typedef BlockCfg<TW> Cfg;
    const int x = c.X0 + tid;
    EmitStore emit;
    emit.out = c.out; emit.w = c.w; emit.x = x; emit.my = c.ay.m; emit.ya = c.ya;
    emit.yb = x < c.w ? c.yb : c.ya;          // columns beyond the image store nothing
    emit.ylo = c.ay.lo; emit.yhi = c.ay.hi; emit.xok = (x >= c.ax.lo && x <= c.ax.hi); emit.fill = c.fill;
    const float* tcol = c.T + tid;
    if (range_is_edge(c.ay, rb - L, rb + R - 1)) y_block<true>(c.ay, st, tcol, Cfg::PITCH_T, rb, first, emit);
    else y_block<false>(c.ay, st, tcol, Cfg::PITCH_T, rb, first, emit);
}

}  // namespace rs
}  // namespace mred
