// resample_ypass.cuh -- the y pass of the two-kernel route as a kernel of its own: one THREAD per 4 adjacent columns
// (a 128-bit load per row), no shuffles, no halo lanes.  Same arithmetic as the y part of warp_item (resample_warp.cuh):
// causal recursion g = t - a g_prev down the rows, the anti-causal start value of every 8-row block accumulated from
// the 16 rows that follow it, a backward sweep out of a per-thread shared-memory ring (24 rows x 16 B), the 4 y taps,
// 128-bit stores.  Half the state per thread of the 8-column version, so twice as many warps for the same band
// height: it is used when w % 4 == 0 (rows 16-byte aligned); other widths take k_resample<2>.
#pragma once

namespace mred {
namespace rs {

constexpr int YT = 128;                       // threads per block: 512 columns
constexpr int YRING = NRING * RB;             // rows in the ring

// 4 samples (columns x .. x+3) of row `row` of the y-extended x-shifted plane T (row is block-uniform)
__device__ __forceinline__ float4 ypass_load(const float* T, int w, int h, int row, int x)
{
    if (row >= 0 && row < h) return __ldg(reinterpret_cast<const float4*>(T + (size_t)row * w + x));
    if (row < -EXT || row >= h + EXT) return make_float4(0.f, 0.f, 0.f, 0.f);
    const ExtIdx e = ext_index(row, h);       // a T[rb] + b T[h-1] + c T[0]
    const float4 t = __ldg(reinterpret_cast<const float4*>(T + (size_t)e.rb * w + x));
    float4 r = make_float4(e.a * t.x, e.a * t.y, e.a * t.z, e.a * t.w);
    if (e.b != 0.f) {
        const float4 u = __ldg(reinterpret_cast<const float4*>(T + (size_t)(h - 1) * w + x));
        r.x = fmaf(e.b, u.x, r.x); r.y = fmaf(e.b, u.y, r.y); r.z = fmaf(e.b, u.z, r.z); r.w = fmaf(e.b, u.w, r.w);
    }
    if (e.c != 0.f) {
        const float4 u = __ldg(reinterpret_cast<const float4*>(T + x));
        r.x = fmaf(e.c, u.x, r.x); r.y = fmaf(e.c, u.y, r.y); r.z = fmaf(e.c, u.z, r.z); r.w = fmaf(e.c, u.w, r.w);
    }
    return r;
}

struct Y4 {
    float na, w0, w1, w2, w3;   // -a and the four weights times 6a (1 on an identity axis)
    int my, ylo, yhi;           // interval k -> output row k - my, kept when in [ylo, yhi]
    float* out;                 // output plane + the thread's first column
    int w;
    unsigned xmask;             // bit j: column x + j lies in the x footprint
    float fill;
};

__device__ __forceinline__ void y4_emit(const Y4& c, int k, const float4& a0, const float4& a1, const float4& a2, const float4& a3)
{
    const int y = k - c.my;
    if (y < c.ylo || y > c.yhi) return;      // block-uniform
    float4 v;
    v.x = fmaf(c.w3, a3.x, fmaf(c.w2, a2.x, fmaf(c.w1, a1.x, c.w0 * a0.x)));
    v.y = fmaf(c.w3, a3.y, fmaf(c.w2, a2.y, fmaf(c.w1, a1.y, c.w0 * a0.y)));
    v.z = fmaf(c.w3, a3.z, fmaf(c.w2, a2.z, fmaf(c.w1, a1.z, c.w0 * a0.z)));
    v.w = fmaf(c.w3, a3.w, fmaf(c.w2, a2.w, fmaf(c.w1, a1.w, c.w0 * a0.w)));
    if (c.xmask != 0xfu) {
        v.x = (c.xmask & 1u) ? v.x : c.fill; v.y = (c.xmask & 2u) ? v.y : c.fill;
        v.z = (c.xmask & 4u) ? v.z : c.fill; v.w = (c.xmask & 8u) ? v.w : c.fill;
    }
    *reinterpret_cast<float4*>(c.out + (size_t)y * c.w) = v;
}

__device__ __forceinline__ float4 f4_fma(float s, const float4& a, const float4& b)   // s * a + b
{
    return make_float4(fmaf(s, a.x, b.x), fmaf(s, a.y, b.y), fmaf(s, a.z, b.z), fmaf(s, a.w, b.w));
}

}  // namespace rs

using namespace rs;

// grid (ceil(w / 512), bands, n), block 128
__global__ void __launch_bounds__(YT) k_ypass4(const float* __restrict__ T, int n, int w, int h,
                                               const __grid_constant__ HostShifts hs, const double* __restrict__ dshift,
                                               float fill, float* __restrict__ out, int4* __restrict__ fp_dev, int BH)
{
    __shared__ float4 s_ring[YRING][YT];
    const int k = blockIdx.z;
    const double sx = dshift ? -dshift[2 * k] : hs.s[k][0];
    const double sy = dshift ? -dshift[2 * k + 1] : hs.s[k][1];
    const Axis ax = make_axis(w, sx);
    const Axis ay = make_axis(h, sy);
    if (fp_dev && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) fp_dev[k] = make_int4(ax.lo, ax.hi, ay.lo, ay.hi);
    const size_t np = (size_t)w * h;
    const int x = ((int)blockIdx.x * YT + (int)threadIdx.x) * 4;
    const bool on = x < w;                                    // w % 4 == 0: all four columns or none
    const int xs = on ? x : 0;                                // idle threads shadow column 0 and never store
    const float* Tk = T + (size_t)k * np;
    const int ya = (int)blockIdx.y * BH, yb = min(ya + BH, h);
    const int Xs = (int)blockIdx.x * YT * 4, Xe = min(Xs + YT * 4, w);
    const bool x_any = max(Xs, ax.lo) <= min(Xe - 1, ax.hi);
    int ylo = max(ya, ay.lo), yhi = min(yb - 1, ay.hi);
    if (!x_any) { ylo = yb; yhi = yb - 1; }
    const float4 fill4 = make_float4(fill, fill, fill, fill);
    float* outk = out + (size_t)k * np + xs;
    if (on) {
        for (int y = ya; y < min(ylo, yb); ++y) *reinterpret_cast<float4*>(outk + (size_t)y * w) = fill4;
        for (int y = max(yhi + 1, ya); y < yb; ++y) *reinterpret_cast<float4*>(outk + (size_t)y * w) = fill4;
    }
    if (ylo > yhi) return;                                    // block-uniform

    Y4 c;
    const float sc = ay.ident ? 1.f : 6.0f * U_INF;
    c.na = ay.ident ? 0.f : -U_INF;
    c.w0 = sc * ay.w[0]; c.w1 = sc * ay.w[1]; c.w2 = sc * ay.w[2]; c.w3 = sc * ay.w[3];
    c.my = ay.m; c.ylo = on ? ylo : yb; c.yhi = on ? yhi : yb - 1;     // idle threads emit nothing
    c.out = outk; c.w = w; c.fill = fill;
    c.xmask = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j)
        if (x + j >= ax.lo && x + j <= ax.hi) c.xmask |= 1u << j;

    const int ka = ylo + ay.m, kb = yhi + 1 + ay.m;           // intervals [ka, kb)
    const int r0 = ka - WARM;
    const int NB = (kb - ka + 18) / RB + 3;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 gprev = zero, A1 = zero, A2 = zero, s1 = zero, s2 = zero, s3 = zero;
    float pi1 = 0.f, pi2 = 0.f;
    constexpr int GR = 4;
    float4 nxt[GR];
#pragma unroll
    for (int i = 0; i < GR; ++i) nxt[i] = ypass_load(Tk, w, h, r0 + i, xs);
    const int NG = NB * (RB / GR);
#pragma unroll 1
    for (int gi = 0; gi < NG; ++gi) {
        const int row0 = r0 + GR * gi;
        const int slot0 = (GR * gi) % YRING;
        float4 cur[GR];
#pragma unroll
        for (int i = 0; i < GR; ++i) cur[i] = nxt[i];
#pragma unroll
        for (int i = 0; i < GR; ++i) nxt[i] = ypass_load(Tk, w, h, row0 + GR + i, xs);
#pragma unroll
        for (int i = 0; i < GR; ++i) {
            const float4 g = f4_fma(c.na, gprev, cur[i]);
            gprev = g;
            A1 = f4_fma(pi1, g, A1);
            A2 = f4_fma(pi2, g, A2);
            pi1 *= c.na; pi2 *= c.na;
            s_ring[slot0 + i][threadIdx.x] = g;
        }
        if ((gi & (RB / GR - 1)) == RB / GR - 1) {
            const int nblk = gi / (RB / GR);
            if (nblk >= 4) {
                // A2 = c' of the last row of block nblk-2: sweep that block backwards out of the ring
                const int b = nblk - 2, start = r0 + RB * b, sb = (b % NRING) * RB;
                float4 c0 = A2, c1 = zero, c2 = zero, c3 = zero, n2 = zero, n3 = zero;
#pragma unroll
                for (int q = RB - 2; q >= 0; --q) {
                    const float4 g = s_ring[sb + q][threadIdx.x];
                    c3 = c2; c2 = c1; c1 = c0; c0 = f4_fma(c.na, c1, g);
                    if (q == RB - 2) n2 = c0;
                    if (q == RB - 3) n3 = c0;
                    if (q <= RB - 4) y4_emit(c, start + q + 1, c0, c1, c2, c3);
                }
                y4_emit(c, start, s1, c0, c1, c2);
                y4_emit(c, start - 1, s2, s1, c0, c1);
                y4_emit(c, start - 2, s3, s2, s1, c0);
                s1 = A2; s2 = n2; s3 = n3;
            }
            A2 = A1; A1 = gprev;
            pi2 = pi1; pi1 = c.na;
        }
    }
}

}  // namespace mred
