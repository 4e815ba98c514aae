// resample_warp.cuh -- the per-warp program of the spline-shift kernel (see resample.cu for the
// mathematics and the design), the kernel shell and the launcher.
#pragma once

namespace mred {
namespace rs {

constexpr unsigned FULL = 0xffffffffu;

struct Item {
    const float* in;   // frame k input plane
    float* out;        // frame k output plane
    int w, h;
    Axis ax, ay;
    int XA;            // output column of lane 0, element 0 (multiple of 4; first kept column is XA + 24)
    int ya, yb;        // output rows [ya, yb) of the band
    float fill;
};

// Point-reflection extension of a line of n samples: index i outside [0, n).
// f(i + T) = f(i) + 2 (f_{n-1} - f_0) with T = 2(n-1); inside one period the second half is the
// reflection about n-1.  The value is a*F[rb] + b*F[n-1] + c*F[0].
struct ExtIdx { int rb; float a, b, c; };

__device__ __forceinline__ ExtIdx ext_index(int i, int n)
{
    const int T = 2 * (n - 1);
    int q = i / T, r = i - q * T;
    if (r < 0) { r += T; q -= 1; }
    ExtIdx e;
    const bool mir = r > n - 1;
    e.rb = mir ? T - r : r;
    e.a = mir ? -1.0f : 1.0f;
    e.b = (mir ? 2.0f : 0.0f) + 2.0f * (float)q;
    e.c = -2.0f * (float)q;
    return e;
}

// one sample of the x-extended real row p (length n) at column c outside [0, n)
__device__ __forceinline__ float ext_x(const float* p, int c, int n)
{
    if (c < -EXT || c >= n + EXT) return 0.f;
    const ExtIdx e = ext_index(c, n);
    return fmaf(e.a, __ldg(p + e.rb), fmaf(e.b, __ldg(p + n - 1), e.c * __ldg(p)));
}

// four consecutive samples (columns c .. c+3) of the real row `row`, x-extended; any c
__device__ __forceinline__ float4 real4(const float* in, int w, int row, int c)
{
    const float* p = in + (size_t)row * w;
    float v[4];
#pragma unroll 1
    for (int j = 0; j < 4; ++j) {
        const int cc = c + j;
        const float t = (cc >= 0 && cc < w) ? __ldg(p + cc) : ext_x(p, cc, w);
        v[0] = j == 0 ? t : v[0]; v[1] = j == 1 ? t : v[1]; v[2] = j == 2 ? t : v[2]; v[3] = j == 3 ? t : v[3];
    }
    return make_float4(v[0], v[1], v[2], v[3]);
}

// COLD path (kept out of line so that the hot loop stays small): four consecutive samples of row `row`
// of the extended image, for lanes / rows that are not entirely inside the image.
__device__ __noinline__ float4 slow4(const float* in, int w, int h, int row, int c)
{
    if (row >= 0 && row < h) return real4(in, w, row, c);
    if (row < -EXT || row >= h + EXT) return make_float4(0.f, 0.f, 0.f, 0.f);
    const ExtIdx e = ext_index(row, h);
    float4 t = real4(in, w, e.rb, c);
    float4 r = make_float4(e.a * t.x, e.a * t.y, e.a * t.z, e.a * t.w);
    if (e.b != 0.f) {
        t = real4(in, w, h - 1, c);
        r.x = fmaf(e.b, t.x, r.x); r.y = fmaf(e.b, t.y, r.y); r.z = fmaf(e.b, t.z, r.z); r.w = fmaf(e.b, t.w, r.w);
    }
    if (e.c != 0.f) {
        t = real4(in, w, 0, c);
        r.x = fmaf(e.c, t.x, r.x); r.y = fmaf(e.c, t.y, r.y); r.z = fmaf(e.c, t.z, r.z); r.w = fmaf(e.c, t.w, r.w);
    }
    return r;
}

// How a lane fetches one half (4 consecutive columns starting at c) of a real row, fixed per item:
//   mode 0: aligned 128-bit load at c (all four columns inside the image)
//   mode 1: the point-reflected columns, RAW: p[mb - j]; the reflection arithmetic 2 p[e] - (.) is applied
//           when the row is consumed (x_fix), so that the load itself never waits for its data
//   mode 2: out of line, finished values (images smaller than 2 EXT + 8, halves that straddle an edge)
//   mode 3: as mode 0 with four scalar loads (rows not 16-byte aligned: w % 4 != 0)
//   mode 4: zeros (columns farther than EXT from the image: never used by a kept output)
struct HalfCfg { int mode, c, mb; };

__device__ __forceinline__ HalfCfg half_cfg(int c, int w, bool vec, bool simple)
{
    HalfCfg hc;
    hc.c = c; hc.mb = 0; hc.mode = 2;
    if (c >= 0 && c + 4 <= w) hc.mode = vec ? 0 : 3;
    else if (simple && c + 3 < 0) { hc.mode = c >= -EXT ? 1 : 4; hc.mb = -c; }
    else if (simple && c >= w) { hc.mode = c + 3 < w + EXT ? 1 : 4; hc.mb = 2 * (w - 1) - c; }
    return hc;
}

__device__ __forceinline__ float4 load_half(const Item& it, int row, const HalfCfg& hc)
{
    const float* p = it.in + (size_t)row * it.w;
    if (hc.mode == 0) return __ldg(reinterpret_cast<const float4*>(p + hc.c));
    if (hc.mode == 1) {
        const float* q = p + hc.mb;
        return make_float4(__ldg(q), __ldg(q - 1), __ldg(q - 2), __ldg(q - 3));
    }
    if (hc.mode == 3) return make_float4(__ldg(p + hc.c), __ldg(p + hc.c + 1), __ldg(p + hc.c + 2), __ldg(p + hc.c + 3));
    if (hc.mode == 4) return make_float4(0.f, 0.f, 0.f, 0.f);
    return slow4(it.in, it.w, it.h, row, hc.c);
}

// the lane's 8 samples of source row `row` (warp-uniform).  simple: raw values of the real row that stands
// behind `row` (itself, or its mirror image about the near edge), to be finished by x_fix / the y reflection
// when consumed; otherwise finished values from the out-of-line path.
__device__ __forceinline__ void load_row(const Item& it, int row, bool simple, const HalfCfg& h0, const HalfCfg& h1,
                                         float (&f)[V])
{
    float4 a, b;
    if (simple) {
        const int ra = row < 0 ? -row : (row >= it.h ? 2 * (it.h - 1) - row : row);
        if (row < -EXT || row >= it.h + EXT) { a = make_float4(0.f, 0.f, 0.f, 0.f); b = a; }
        else { a = load_half(it, ra, h0); b = load_half(it, ra, h1); }
    } else if (row >= 0 && row < it.h) {
        a = load_half(it, row, h0); b = load_half(it, row, h1);
    } else {
        a = slow4(it.in, it.w, it.h, row, h0.c); b = slow4(it.in, it.w, it.h, row, h1.c);
    }
    f[0] = a.x; f[1] = a.y; f[2] = a.z; f[3] = a.w; f[4] = b.x; f[5] = b.y; f[6] = b.z; f[7] = b.w;
}

// per-lane description of the reflected halves of a strip (simple case only)
struct XFix {
    int pL, pR;            // raw position (lane*8 + j) of image columns 0 and w-1 in the warp, -1: no reflected half on that side
    bool l0, l1, r0, r1;   // this lane's half 0 / 1 is reflected about the left / right edge
};

__device__ __forceinline__ float pick(const float (&c)[V], int j)
{
    float v = c[0];
#pragma unroll
    for (int i = 1; i < V; ++i) v = (j == i) ? c[i] : v;
    return v;
}

// finish the reflected halves of one raw row: v <- 2 f(edge) - v (warp-uniform branches)
__device__ __forceinline__ void x_fix(const XFix& xf, float (&f)[V])
{
    if (xf.pL >= 0) {
        const float ed = 2.0f * __shfl_sync(FULL, pick(f, xf.pL & 7), xf.pL >> 3);
#pragma unroll
        for (int j = 0; j < 4; ++j) { f[j] = xf.l0 ? ed - f[j] : f[j]; f[4 + j] = xf.l1 ? ed - f[4 + j] : f[4 + j]; }
    }
    if (xf.pR >= 0) {
        const float ed = 2.0f * __shfl_sync(FULL, pick(f, xf.pR & 7), xf.pR >> 3);
#pragma unroll
        for (int j = 0; j < 4; ++j) { f[j] = xf.r0 ? ed - f[j] : f[j]; f[4 + j] = xf.r1 ? ed - f[4 + j] : f[4 + j]; }
    }
}

// f[j] <- element j + r of (own 8 samples, next lane's 8 samples), r in 0..3 warp-uniform
__device__ __forceinline__ void realign(float (&f)[V], int r)
{
    const bool b1 = r & 1, b2 = r & 2;
    const float n0 = __shfl_down_sync(FULL, f[0], 1);
#pragma unroll
    for (int j = 0; j < V - 1; ++j) f[j] = b1 ? f[j + 1] : f[j];
    f[V - 1] = b1 ? n0 : f[V - 1];
    const float m0 = __shfl_down_sync(FULL, f[0], 1);
    const float m1 = __shfl_down_sync(FULL, f[1], 1);
#pragma unroll
    for (int j = 0; j < V - 2; ++j) f[j] = b2 ? f[j + 2] : f[j];
    f[V - 2] = b2 ? m0 : f[V - 2];
    f[V - 1] = b2 ? m1 : f[V - 1];
}

// x pass of G rows at once (independent rows interleave and hide the FMA latency): f[i] = the lane's 8
// source samples of row i (columns x_j + m); on exit f[i] = the 8 x-shifted values.
// na = -a (0 on an identity axis), na8 = na^8, wx = the four weights times 6a (times 1 on an identity axis).
template <int G>
__device__ __forceinline__ void x_pass(float na, float na8, const float (&wx)[4], float (&f)[G][V])
{
    float z[G], gp[G];
    // causal: zero-state response of the lane, carry from the two lanes before it, then the real sweep
#pragma unroll
    for (int i = 0; i < G; ++i) z[i] = f[i][0];
#pragma unroll
    for (int j = 1; j < V; ++j)
#pragma unroll
        for (int i = 0; i < G; ++i) z[i] = fmaf(na, z[i], f[i][j]);
#pragma unroll
    for (int i = 0; i < G; ++i) {
        const float zz = fmaf(na8, __shfl_up_sync(FULL, z[i], 1), z[i]);
        gp[i] = __shfl_up_sync(FULL, zz, 1);       // lanes 0, 1 get garbage: they are halo
    }
#pragma unroll
    for (int j = 0; j < V; ++j)
#pragma unroll
        for (int i = 0; i < G; ++i) { gp[i] = fmaf(na, gp[i], f[i][j]); f[i][j] = gp[i]; }
    // anti-causal, mirrored
#pragma unroll
    for (int i = 0; i < G; ++i) z[i] = f[i][V - 1];
#pragma unroll
    for (int j = V - 2; j >= 0; --j)
#pragma unroll
        for (int i = 0; i < G; ++i) z[i] = fmaf(na, z[i], f[i][j]);
#pragma unroll
    for (int i = 0; i < G; ++i) {
        const float zz = fmaf(na8, __shfl_down_sync(FULL, z[i], 1), z[i]);
        gp[i] = __shfl_down_sync(FULL, zz, 1);     // lanes 30, 31: halo
    }
#pragma unroll
    for (int j = V - 1; j >= 0; --j)
#pragma unroll
        for (int i = 0; i < G; ++i) { gp[i] = fmaf(na, gp[i], f[i][j]); f[i][j] = gp[i]; }
    // 4-tap evaluation; f[i][j] is overwritten in place from the left
#pragma unroll
    for (int i = 0; i < G; ++i) {
        const float cl = __shfl_up_sync(FULL, f[i][7], 1);
        const float cr0 = __shfl_down_sync(FULL, f[i][0], 1);
        const float cr1 = __shfl_down_sync(FULL, f[i][1], 1);
        float prev = cl;
#pragma unroll
        for (int j = 0; j < V; ++j) {
            const float c1 = f[i][j];
            const float c2 = j + 1 < V ? f[i][j + 1] : cr0;
            const float c3 = j + 2 < V ? f[i][j + 2] : (j + 2 == V ? cr0 : cr1);
            f[i][j] = fmaf(wx[3], c3, fmaf(wx[2], c2, fmaf(wx[1], c1, wx[0] * prev)));
            prev = c1;
        }
    }
}

template <bool VEC>
__device__ __forceinline__ void store_row(const Item& it, int y, int x, bool lane_on, const float (&v)[V])
{
    if (!lane_on) return;
    float* p = it.out + (size_t)y * it.w + x;
    if (VEC) {
        *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);   // lane_on: x < w, and w % 4 == 0
        if (x + 4 < it.w) *reinterpret_cast<float4*>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
    } else {
#pragma unroll
        for (int j = 0; j < V; ++j)
            if (x + j < it.w) p[j] = v[j];
    }
}

struct YCtx {
    float na;          // -a along y (0 on an identity axis)
    float wy[4];       // y weights times 6a (times 1 on an identity axis)
    int my, ylo, yhi;  // interval k -> output row k - my, kept when in [ylo, yhi]
    int x0;            // the lane's first output column
    bool lane_on;
    unsigned xmask;    // bit j: column x0 + j lies in the x footprint
};

template <bool VEC>
__device__ __forceinline__ void emit(const Item& it, const YCtx& yc, int k, const float (&a0)[V], const float (&a1)[V],
                                     const float (&a2)[V], const float (&a3)[V])
{
    const int y = k - yc.my;
    if (y < yc.ylo || y > yc.yhi) return;      // warp-uniform
    float v[V];
#pragma unroll
    for (int j = 0; j < V; ++j) v[j] = fmaf(yc.wy[3], a3[j], fmaf(yc.wy[2], a2[j], fmaf(yc.wy[1], a1[j], yc.wy[0] * a0[j])));
    if (yc.xmask != 0xffu) {
#pragma unroll
        for (int j = 0; j < V; ++j) v[j] = ((yc.xmask >> j) & 1u) ? v[j] : it.fill;
    }
    store_row<VEC>(it, y, yc.x0, yc.lane_on, v);
}

// backward sweep of one block (rows start .. start+7) out of the ring, evaluation and store of the 8
// intervals start-2 .. start+5.  cA = c' of row start+7 (the accumulated anti-causal start value);
// s1, s2, s3 = c' of rows start-1, -2, -3 (left by the previous block), replaced on exit.
template <bool VEC>
__device__ __forceinline__ void sweep_block(const Item& it, const YCtx& yc, const float4* ring4, int sb, int start,
                                            const float (&cA)[V], float (&s1)[V], float (&s2)[V], float (&s3)[V], int lane)
{
    float c0[V], c1[V], c2[V], c3[V], n2[V], n3[V];
#pragma unroll
    for (int j = 0; j < V; ++j) { c0[j] = cA[j]; c1[j] = 0.f; c2[j] = 0.f; c3[j] = 0.f; n2[j] = 0.f; n3[j] = 0.f; }
#pragma unroll
    for (int q = RB - 2; q >= 0; --q) {
        const float4 ga = ring4[((sb + q) * 2 + 0) * 32 + lane];
        const float4 gb = ring4[((sb + q) * 2 + 1) * 32 + lane];
        const float gg[V] = {ga.x, ga.y, ga.z, ga.w, gb.x, gb.y, gb.z, gb.w};
#pragma unroll
        for (int j = 0; j < V; ++j) { c3[j] = c2[j]; c2[j] = c1[j]; c1[j] = c0[j]; c0[j] = fmaf(yc.na, c1[j], gg[j]); }
        if (q == RB - 2) {
#pragma unroll
            for (int j = 0; j < V; ++j) n2[j] = c0[j];
        }
        if (q == RB - 3) {
#pragma unroll
            for (int j = 0; j < V; ++j) n3[j] = c0[j];
        }
        if (q <= RB - 4) emit<VEC>(it, yc, start + q + 1, c0, c1, c2, c3);   // window rows k-1 .. k+2
    }
    // the three intervals that straddle into the previous block: rows (s3, s2, s1 | c0, c1, c2)
    emit<VEC>(it, yc, start, s1, c0, c1, c2);
    emit<VEC>(it, yc, start - 1, s2, s1, c0, c1);
    emit<VEC>(it, yc, start - 2, s3, s2, s1, c0);
#pragma unroll
    for (int j = 0; j < V; ++j) { s1[j] = cA[j]; s2[j] = n2[j]; s3[j] = n3[j]; }
}

// MODE 0: x and y pass fused (one read, one write per pixel).
// MODE 1: x pass only, `out` = the x-shifted rows (every row of the band, no y footprint, no fill).
// MODE 2: y pass only on x-shifted rows: no halo lanes, no realignment, columns map one to one.
// Modes 1 + 2 are the two-kernel route for stacks small enough to keep the intermediate in L2.
template <int MODE> struct ModeGeom {
    static constexpr int HL = MODE == 2 ? 0 : HALO_L, HR = MODE == 2 ? 0 : HALO_R;
    static constexpr int OUTC = (32 - HL - HR) * V;
};

template <bool VEC, int MODE>
__device__ void warp_item(const Item& it, float* ring, int lane)
{
    constexpr int HL = ModeGeom<MODE>::HL, HR = ModeGeom<MODE>::HR, OUTC = ModeGeom<MODE>::OUTC;
    const Axis& ax = it.ax;
    const Axis& ay = it.ay;
    YCtx yc;
    yc.x0 = it.XA + V * lane;
    yc.lane_on = lane >= HL && lane < 32 - HR && yc.x0 < it.w;
    const int Xs = it.XA + V * HL;                                     // first kept column of the strip
    const int Xe = min(Xs + OUTC, it.w);                               // one past the last
    float fillv[V];
#pragma unroll
    for (int j = 0; j < V; ++j) fillv[j] = it.fill;

    // rows of the band that can hold data; everything else is fill
    const bool x_any = max(Xs, ax.lo) <= min(Xe - 1, ax.hi);
    int ylo = max(it.ya, ay.lo), yhi = min(it.yb - 1, ay.hi);
    if (MODE == 1) {
        if (!x_any) return;                        // the y pass writes fill there without reading
        ylo = it.ya; yhi = it.yb - 1;
    } else {
        if (!x_any) { ylo = it.yb; yhi = it.yb - 1; }
        for (int y = it.ya; y < min(ylo, it.yb); ++y) store_row<VEC>(it, y, yc.x0, yc.lane_on, fillv);
        for (int y = max(yhi + 1, it.ya); y < it.yb; ++y) store_row<VEC>(it, y, yc.x0, yc.lane_on, fillv);
        if (ylo > yhi) return;
    }

    if (MODE == 0 && ax.ident && ay.ident) {     // pure integer translation: copy with 16 independent loads in flight per lane
        const int xa = max(Xs, ax.lo), xb = min(Xe - 1, ax.hi);       // columns that carry data (x_any: xa <= xb)
        for (int y = ylo; y <= yhi; ++y) {                            // fill left and right of the footprint
            float* dst = it.out + (size_t)y * it.w;
            for (int x = Xs + lane; x < xa; x += 32) dst[x] = it.fill;
            for (int x = xb + 1 + lane; x < Xe; x += 32) dst[x] = it.fill;
        }
        const int nrow = yhi - ylo + 1;
        if (VEC && ((ax.m & 3) == 0) && ((xa & 3) == 0) && ((xb & 3) == 3)) {
            const int c4 = (xb - xa + 1) >> 2, tot = c4 * nrow;
            for (int base = 0; base < tot; base += 32 * 16) {
                float4 v[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const int idx = base + lane + 32 * i;
                    if (idx < tot) {
                        const int yy = idx / c4, xx = xa + 4 * (idx - yy * c4);
                        v[i] = __ldg(reinterpret_cast<const float4*>(it.in + (size_t)(ylo + yy + ay.m) * it.w + xx + ax.m));
                    }
                }
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const int idx = base + lane + 32 * i;
                    if (idx < tot) {
                        const int yy = idx / c4, xx = xa + 4 * (idx - yy * c4);
                        *reinterpret_cast<float4*>(it.out + (size_t)(ylo + yy) * it.w + xx) = v[i];
                    }
                }
            }
        } else {
            const int c1 = xb - xa + 1, tot = c1 * nrow;
            for (int base = 0; base < tot; base += 32 * 16) {
                float v[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const int idx = base + lane + 32 * i;
                    if (idx < tot) {
                        const int yy = idx / c1, xx = xa + (idx - yy * c1);
                        v[i] = __ldg(it.in + (size_t)(ylo + yy + ay.m) * it.w + xx + ax.m);
                    }
                }
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const int idx = base + lane + 32 * i;
                    if (idx < tot) {
                        const int yy = idx / c1, xx = xa + (idx - yy * c1);
                        it.out[(size_t)(ylo + yy) * it.w + xx] = v[i];
                    }
                }
            }
        }
        return;
    }

    // constants of the two axes
    const float nax = ax.ident ? 0.f : -U_INF;
    const float nax2 = nax * nax, nax4 = nax2 * nax2, nax8 = nax4 * nax4;
    const float scx = ax.ident ? 1.f : 6.0f * U_INF, scy = ay.ident ? 1.f : 6.0f * U_INF;
    const float wx[4] = {scx * ax.w[0], scx * ax.w[1], scx * ax.w[2], scx * ax.w[3]};
    yc.na = ay.ident ? 0.f : -U_INF;
#pragma unroll
    for (int i = 0; i < 4; ++i) yc.wy[i] = scy * ay.w[i];
    yc.my = ay.m; yc.ylo = ylo; yc.yhi = yhi;
    yc.xmask = 0u;
#pragma unroll
    for (int j = 0; j < V; ++j)
        if (yc.x0 + j >= ax.lo && yc.x0 + j <= ax.hi) yc.xmask |= 1u << j;

    // x geometry of the lane
    const int KC0 = MODE == 2 ? it.XA : it.XA + ax.m;   // source column under output column XA
    const int r = (VEC && MODE != 2) ? (KC0 & 3) : 0;   // aligned loads start r columns early
    const int col_load = KC0 - r + V * lane;
    const bool simple = it.w >= 2 * EXT + 8 && it.h >= 2 * EXT + 8;
    HalfCfg h0 = half_cfg(col_load, it.w, VEC, simple), h1 = half_cfg(col_load + 4, it.w, VEC, simple);
    if (MODE == 2) {                              // columns beyond the image are never stored: no reflection
        if (h0.mode == 1) h0.mode = 4;
        if (h1.mode == 1) h1.mode = 4;
    }
    XFix xf;
    xf.l0 = h0.mode == 1 && h0.c < 0; xf.l1 = h1.mode == 1 && h1.c < 0;
    xf.r0 = h0.mode == 1 && h0.c > 0; xf.r1 = h1.mode == 1 && h1.c > 0;
    xf.pL = __any_sync(FULL, xf.l0 || xf.l1) ? -(KC0 - r) : -1;
    xf.pR = __any_sync(FULL, xf.r0 || xf.r1) ? it.w - 1 - (KC0 - r) : -1;
    if (xf.pL > WARPCOLS - 1) xf.pL = -1;         // column 0 not in the warp: no kept output needs the reflection
    if (xf.pR > WARPCOLS - 1 || it.w - 1 - (KC0 - r) < 0) xf.pR = -1;
    const bool all_in = VEC && __all_sync(FULL, h0.mode == 0 && h1.mode == 0);
    float edge_row[V];                            // finished row 0 or h-1 (raw alignment), for the y reflection
    int edge_is = -1;
#pragma unroll
    for (int j = 0; j < V; ++j) edge_row[j] = 0.f;

    // y schedule
    const int ka = ylo + ay.m, kb = yhi + 1 + ay.m;     // intervals [ka, kb)
    const int r0 = MODE == 1 ? ylo : ka - WARM;         // first source row processed
    const int NB = MODE == 1 ? (yhi - ylo + RB) / RB : (kb - ka + 18) / RB + 3;   // blocks (of RB rows) processed

    float gprev[V], A1[V], A2[V], s1[V], s2[V], s3[V];
#pragma unroll
    for (int j = 0; j < V; ++j) { gprev[j] = 0.f; A1[j] = 0.f; A2[j] = 0.f; s1[j] = 0.f; s2[j] = 0.f; s3[j] = 0.f; }
    float pi1 = 0.f, pi2 = 0.f;
    float4* ring4 = reinterpret_cast<float4*>(ring);    // [slot][half][lane]

    constexpr int GR = 4;                               // rows per group: loaded, x-passed and y-advanced together
    float nxt[GR][V];
#pragma unroll
    for (int i = 0; i < GR; ++i)
#pragma unroll
        for (int j = 0; j < V; ++j) nxt[i][j] = 0.f;

    const int NG = NB * (RB / GR);
    // iteration gi loads group gi+1 and processes group gi; gi = -1 only loads (one load site keeps the code small)
#pragma unroll 1
    for (int gi = -1; gi < NG; ++gi) {
        const int row0 = r0 + GR * gi;
        float cur[GR][V];
#pragma unroll
        for (int i = 0; i < GR; ++i)
#pragma unroll
            for (int j = 0; j < V; ++j) cur[i][j] = nxt[i][j];
#pragma unroll
        if (all_in && row0 + GR >= 0 && row0 + 2 * GR <= it.h) {
            const float4* p = reinterpret_cast<const float4*>(it.in + (size_t)(row0 + GR) * it.w + col_load);
#pragma unroll
            for (int i = 0; i < GR; ++i) {
                const float4 a = __ldg(p), b = __ldg(p + 1);
                nxt[i][0] = a.x; nxt[i][1] = a.y; nxt[i][2] = a.z; nxt[i][3] = a.w;
                nxt[i][4] = b.x; nxt[i][5] = b.y; nxt[i][6] = b.z; nxt[i][7] = b.w;
                p += it.w >> 2;
            }
        } else {
#pragma unroll
            for (int i = 0; i < GR; ++i) load_row(it, row0 + GR + i, simple, h0, h1, nxt[i]);
        }
        if (gi < 0) continue;
        const int slot0 = (GR * gi) % (NRING * RB);
        if (simple) {
            // finish what the loads left raw: reflected columns, then reflected rows (both warp-uniform)
            if (xf.pL >= 0 || xf.pR >= 0) {
#pragma unroll
                for (int i = 0; i < GR; ++i) x_fix(xf, cur[i]);
            }
            if (MODE != 1 && (row0 < 0 || row0 + GR > it.h)) {
#pragma unroll 1
                for (int i = 0; i < GR; ++i) {
                    const int row = row0 + i;
                    if ((row >= 0 && row < it.h) || row < -EXT || row >= it.h + EXT) continue;
                    const int rb = row < 0 ? 0 : it.h - 1;
                    if (edge_is != rb) {
                        load_row(it, rb, simple, h0, h1, edge_row);
                        x_fix(xf, edge_row);
                        edge_is = rb;
                    }
#pragma unroll
                    for (int ii = 0; ii < GR; ++ii)
                        if (ii == i) {
#pragma unroll
                            for (int j = 0; j < V; ++j) cur[ii][j] = fmaf(2.0f, edge_row[j], -cur[ii][j]);
                        }
                }
            }
        }
        if (MODE != 2) {
            if (VEC) {
#pragma unroll
                for (int i = 0; i < GR; ++i) realign(cur[i], r);
            }
            x_pass<GR>(nax, nax8, wx, cur);
        }
        if (MODE == 1) {
#pragma unroll
            for (int i = 0; i < GR; ++i)
                if (row0 + i <= yhi) store_row<VEC>(it, row0 + i, yc.x0, yc.lane_on, cur[i]);
            continue;
        }
#pragma unroll
        for (int i = 0; i < GR; ++i) {
#pragma unroll
            for (int j = 0; j < V; ++j) {
                const float g = fmaf(yc.na, gprev[j], cur[i][j]);
                gprev[j] = g;
                cur[i][j] = g;
                A1[j] = fmaf(pi1, g, A1[j]);
                A2[j] = fmaf(pi2, g, A2[j]);
            }
            pi1 *= yc.na; pi2 *= yc.na;
            ring4[((slot0 + i) * 2 + 0) * 32 + lane] = make_float4(cur[i][0], cur[i][1], cur[i][2], cur[i][3]);
            ring4[((slot0 + i) * 2 + 1) * 32 + lane] = make_float4(cur[i][4], cur[i][5], cur[i][6], cur[i][7]);
        }
        if ((gi & (RB / GR - 1)) == RB / GR - 1) {
            // a block is complete: A2 holds c' of the last row of block n-2 -> sweep that block backwards
            const int n = gi / (RB / GR);
            if (n >= 4) {
                const int b = n - 2;
                sweep_block<VEC>(it, yc, ring4, (b % NRING) * RB, r0 + RB * b, A2, s1, s2, s3, lane);
            }
#pragma unroll
            for (int j = 0; j < V; ++j) { A2[j] = A1[j]; A1[j] = gprev[j]; }
            pi2 = pi1; pi1 = yc.na;
        }
    }
}

}  // namespace rs

using namespace rs;

template <int MODE>
__global__ void __launch_bounds__(32, MODE == 1 ? 16 : 8) k_resample(const float* __restrict__ in, int n, int w, int h,
                                                     const __grid_constant__ HostShifts hs,
                                                     const double* __restrict__ dshift, float fill,
                                                     float* __restrict__ out, int4* __restrict__ fp_dev, int BH, int vec)
{
    extern __shared__ __align__(16) float s_ring[];
    const int k = blockIdx.z;
    // (sx, sy): by value from the host call, or minus the estimated content displacement (device)
    const double sx = dshift ? -dshift[2 * k] : hs.s[k][0];
    const double sy = dshift ? -dshift[2 * k + 1] : hs.s[k][1];
    const size_t np = (size_t)w * h;
    Item it;
    it.in = in + (size_t)k * np;
    it.out = out + (size_t)k * np;
    it.w = w; it.h = h; it.fill = fill;
    it.ax = make_axis(w, sx);
    it.ay = make_axis(h, sy);
    it.XA = (int)blockIdx.x * ModeGeom<MODE>::OUTC - V * ModeGeom<MODE>::HL;
    it.ya = (int)blockIdx.y * BH;
    it.yb = min(it.ya + BH, h);
    if (MODE != 1 && fp_dev && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0)
        fp_dev[k] = make_int4(it.ax.lo, it.ax.hi, it.ay.lo, it.ay.hi);
    if (vec) warp_item<true, MODE>(it, s_ring, threadIdx.x);
    else warp_item<false, MODE>(it, s_ring, threadIdx.x);
}

}  // namespace mred
