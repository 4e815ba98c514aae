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

// per-lane x coefficients (constant over the rows of an item)
struct XCoef {
    float P[V], nQ[V], nU[V];
    float QF, UF;      // products of nQ / nU over the lane: response of the lane's far end to its carry-in
    int pl, pr;        // flat position (lane*8 + j) of source columns -1 and n inside the warp, or -1000
};

__device__ __forceinline__ float pick(const float (&c)[V], int j)
{
    float v = c[0];
#pragma unroll
    for (int i = 1; i < V; ++i) v = (j == i) ? c[i] : v;
    return v;
}

// f[j] <- element j + r of (own 8 samples, next lane's 8 samples); r is warp-uniform
__device__ __forceinline__ void realign(float (&f)[V], int r)
{
    if (r == 0) return;
    const float n0 = __shfl_down_sync(FULL, f[0], 1);
    if (r == 1) {
#pragma unroll
        for (int j = 0; j < 7; ++j) f[j] = f[j + 1];
        f[7] = n0;
        return;
    }
    const float n1 = __shfl_down_sync(FULL, f[1], 1);
    if (r == 2) {
#pragma unroll
        for (int j = 0; j < 6; ++j) f[j] = f[j + 2];
        f[6] = n0; f[7] = n1;
        return;
    }
    const float n2 = __shfl_down_sync(FULL, f[2], 1);
#pragma unroll
    for (int j = 0; j < 5; ++j) f[j] = f[j + 3];
    f[5] = n0; f[6] = n1; f[7] = n2;
}

// x pass of one row: f = the lane's 8 source samples (columns x_j + m), t = the 8 x-shifted values
__device__ __forceinline__ void x_pass(const XCoef& xc, const Axis& ax, const float (&f)[V], float (&t)[V], int lane)
{
    float pf[V];
#pragma unroll
    for (int j = 0; j < V; ++j) pf[j] = xc.P[j] * f[j];
    // causal: zero-state response of the lane, carry from the two lanes before it, then the real sweep
    float z = 0.f;
#pragma unroll
    for (int j = 0; j < V; ++j) z = fmaf(xc.nQ[j], z, pf[j]);
    float zp = __shfl_up_sync(FULL, z, 1);
    zp = lane == 0 ? 0.f : zp;
    const float zz = fmaf(xc.QF, zp, z);
    float gp = __shfl_up_sync(FULL, zz, 1);
    gp = lane == 0 ? 0.f : gp;
    float g[V];
#pragma unroll
    for (int j = 0; j < V; ++j) { gp = fmaf(xc.nQ[j], gp, pf[j]); g[j] = gp; }
    // anti-causal, mirrored
    float zc = 0.f;
#pragma unroll
    for (int j = V - 1; j >= 0; --j) zc = fmaf(xc.nU[j], zc, g[j]);
    float zn = __shfl_down_sync(FULL, zc, 1);
    zn = lane == 31 ? 0.f : zn;
    const float zzc = fmaf(xc.UF, zn, zc);
    float cn = __shfl_down_sync(FULL, zzc, 1);
    cn = lane == 31 ? 0.f : cn;
    float c[V];
#pragma unroll
    for (int j = V - 1; j >= 0; --j) { cn = fmaf(xc.nU[j], cn, g[j]); c[j] = cn; }
    // virtual coefficients c_{-1} = 2c_0 - c_1 and c_n = 2c_{n-1} - c_{n-2} (warp-uniform branches)
    if (xc.pl >= 0) {
        const int p = xc.pl;
        float a = pick(c, (p + 1) & 7), b = pick(c, (p + 2) & 7);
        a = __shfl_sync(FULL, a, (p + 1) >> 3);
        b = __shfl_sync(FULL, b, (p + 2) >> 3);
        const float v = 2.0f * a - b;
        if (lane == (p >> 3)) {
#pragma unroll
            for (int j = 0; j < V; ++j) c[j] = ((p & 7) == j) ? v : c[j];
        }
    }
    if (xc.pr >= 0) {
        const int p = xc.pr;
        float a = pick(c, (p - 1) & 7), b = pick(c, (p - 2) & 7);
        a = __shfl_sync(FULL, a, (p - 1) >> 3);
        b = __shfl_sync(FULL, b, (p - 2) >> 3);
        const float v = 2.0f * a - b;
        if (lane == (p >> 3)) {
#pragma unroll
            for (int j = 0; j < V; ++j) c[j] = ((p & 7) == j) ? v : c[j];
        }
    }
    const float cl = __shfl_up_sync(FULL, c[7], 1);
    const float cr0 = __shfl_down_sync(FULL, c[0], 1);
    const float cr1 = __shfl_down_sync(FULL, c[1], 1);
    const float w0 = ax.w[0], w1 = ax.w[1], w2 = ax.w[2], w3 = ax.w[3];
    t[0] = fmaf(w3, c[2], fmaf(w2, c[1], fmaf(w1, c[0], w0 * cl)));
#pragma unroll
    for (int j = 1; j < 6; ++j) t[j] = fmaf(w3, c[j + 2], fmaf(w2, c[j + 1], fmaf(w1, c[j], w0 * c[j - 1])));
    t[6] = fmaf(w3, cr0, fmaf(w2, c[7], fmaf(w1, c[6], w0 * c[5])));
    t[7] = fmaf(w3, cr1, fmaf(w2, cr0, fmaf(w1, c[7], w0 * c[6])));
}

// raw (aligned) load of the lane's 8 samples of one source row; zero outside the image
template <bool VEC>
__device__ __forceinline__ void load_row(const Item& it, int row, int col, float (&f)[V])
{
#pragma unroll
    for (int j = 0; j < V; ++j) f[j] = 0.f;
    if (row < 0 || row >= it.h) return;
    const float* p = it.in + (size_t)row * it.w;
    if (VEC) {
        if (col >= 0 && col < it.w) {
            const float4 a = __ldg(reinterpret_cast<const float4*>(p + col));
            f[0] = a.x; f[1] = a.y; f[2] = a.z; f[3] = a.w;
        }
        if (col + 4 >= 0 && col + 4 < it.w) {
            const float4 a = __ldg(reinterpret_cast<const float4*>(p + col + 4));
            f[4] = a.x; f[5] = a.y; f[6] = a.z; f[7] = a.w;
        }
    } else {
#pragma unroll
        for (int j = 0; j < V; ++j)
            if (col + j >= 0 && col + j < it.w) f[j] = __ldg(p + col + j);
    }
}

template <bool VEC>
__device__ __forceinline__ void store_row(const Item& it, int y, int x, bool lane_on, const float (&v)[V])
{
    if (!lane_on) return;
    float* p = it.out + (size_t)y * it.w + x;
    if (VEC) {
        if (x < it.w) *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
        if (x + 4 < it.w) *reinterpret_cast<float4*>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
    } else {
#pragma unroll
        for (int j = 0; j < V; ++j)
            if (x + j < it.w) p[j] = v[j];
    }
}

// y weights of interval k with the virtual rows folded in (k is warp-uniform)
__device__ __forceinline__ void y_weights(const Axis& ay, int k, float (&wy)[4])
{
    wy[0] = ay.w[0]; wy[1] = ay.w[1]; wy[2] = ay.w[2]; wy[3] = ay.w[3];
    if (!ay.ident) {
        if (k == 0) { wy[1] = wy[1] + 2.0f * wy[0]; wy[2] = wy[2] - wy[0]; }
        if (k == ay.n - 2) { wy[1] = wy[1] - wy[3]; wy[2] = wy[2] + 2.0f * wy[3]; }
    }
}

template <bool VEC>
__device__ void warp_item(const Item& it, float* ring, int lane)
{
    const Axis& ax = it.ax;
    const Axis& ay = it.ay;
    const int x0 = it.XA + V * lane;                                   // the lane's first output column
    const bool lane_on = lane >= HALO_L && lane < 32 - HALO_R && x0 < it.w;
    const int Xs = it.XA + V * HALO_L;                                 // first kept column of the strip
    const int Xe = min(Xs + OUTCOLS, it.w);                            // one past the last
    float fillv[V];
#pragma unroll
    for (int j = 0; j < V; ++j) fillv[j] = it.fill;

    // rows of the band that can hold data; everything else is fill
    const bool x_any = max(Xs, ax.lo) <= min(Xe - 1, ax.hi);
    int ylo = max(it.ya, ay.lo), yhi = min(it.yb - 1, ay.hi);
    if (!x_any) { ylo = it.yb; yhi = it.yb - 1; }
    for (int y = it.ya; y < it.yb; ++y)
        if (y < ylo || y > yhi) store_row<VEC>(it, y, x0, lane_on, fillv);
    if (ylo > yhi) return;

    if (ax.ident && ay.ident) {     // pure integer translation: copy
        for (int y = ylo; y <= yhi; ++y) {
            const float* src = it.in + (size_t)(y + ay.m) * it.w;
            float* dst = it.out + (size_t)y * it.w;
            for (int x = Xs + lane; x < Xe; x += 32) dst[x] = (x >= ax.lo && x <= ax.hi) ? __ldg(src + x + ax.m) : it.fill;
        }
        return;
    }

    // x geometry of the lane
    const int KC0 = it.XA + ax.m;                 // source column under output column XA
    const int r = VEC ? (KC0 & 3) : 0;            // realignment (aligned loads start at KC0 - r)
    const int col_load = KC0 - r + V * lane;
    XCoef xc;
    xc.QF = 1.f; xc.UF = 1.f;
    unsigned xmask = 0u;
#pragma unroll
    for (int j = 0; j < V; ++j) {
        const Coef c = coef(KC0 + V * lane + j, ax.n, ax.ident);
        xc.P[j] = c.P; xc.nQ[j] = c.nQ; xc.nU[j] = c.nU;
        xc.QF *= c.nQ; xc.UF *= c.nU;
        if (x0 + j >= ax.lo && x0 + j <= ax.hi) xmask |= 1u << j;
    }
    xc.pl = -1000; xc.pr = -1000;
    if (!ax.ident) {
        const int pl = -1 - KC0, pr = ax.n - KC0;
        if (pl >= 0 && pl + 2 < WARPCOLS) xc.pl = pl;
        if (pr - 2 >= 0 && pr < WARPCOLS) xc.pr = pr;
    }

    // y schedule
    const int ka = ylo + ay.m, kb = yhi + 1 + ay.m;     // intervals [ka, kb)
    const int r0 = ka - WARM;                           // first source row processed
    const int NB = (kb - ka + 18) / RB + 3;             // blocks processed

    float gprev[V], A1[V], A2[V], s1[V], s2[V], s3[V];
#pragma unroll
    for (int j = 0; j < V; ++j) { gprev[j] = 0.f; A1[j] = 0.f; A2[j] = 0.f; s1[j] = 0.f; s2[j] = 0.f; s3[j] = 0.f; }
    float pi1 = 0.f, pi2 = 0.f;
    float4* ring4 = reinterpret_cast<float4*>(ring);    // [slot][half][lane]

    constexpr int GR = 4;                               // rows per load group (prefetch distance)
    float nxt[GR][V];
#pragma unroll
    for (int i = 0; i < GR; ++i) load_row<VEC>(it, r0 + i, col_load, nxt[i]);

    for (int n = 0; n < NB; ++n) {
        const int rowb = r0 + RB * n;
        const int slotb = (n % NRING) * RB;
#pragma unroll
        for (int gq = 0; gq < RB / GR; ++gq) {
            float cur[GR][V];
#pragma unroll
            for (int i = 0; i < GR; ++i)
#pragma unroll
                for (int j = 0; j < V; ++j) cur[i][j] = nxt[i][j];
#pragma unroll
            for (int i = 0; i < GR; ++i) load_row<VEC>(it, rowb + GR * (gq + 1) + i, col_load, nxt[i]);
#pragma unroll
            for (int i = 0; i < GR; ++i) {
                const int jr = gq * GR + i;
                const int row = rowb + jr;
                realign(cur[i], r);
                float t[V];
                x_pass(xc, ax, cur[i], t, lane);
                const Coef cy = coef(row, ay.n, ay.ident);
                float g[V];
#pragma unroll
                for (int j = 0; j < V; ++j) {
                    g[j] = fmaf(cy.nQ, gprev[j], cy.P * t[j]);
                    gprev[j] = g[j];
                    A1[j] = fmaf(pi1, g[j], A1[j]);
                    A2[j] = fmaf(pi2, g[j], A2[j]);
                }
                pi1 *= cy.nU; pi2 *= cy.nU;
                ring4[((slotb + jr) * 2 + 0) * 32 + lane] = make_float4(g[0], g[1], g[2], g[3]);
                ring4[((slotb + jr) * 2 + 1) * 32 + lane] = make_float4(g[4], g[5], g[6], g[7]);
                if (jr == RB - 1) {
                    // A2 now holds c of the last row of block n-2: sweep that block backwards
                    if (n >= 4) {
                        const int b = n - 2;
                        const int start = r0 + RB * b;
                        const int sb = (b % NRING) * RB;
                        float c0[V], c1[V], c2[V], c3[V], n1[V], n2[V], n3[V];
#pragma unroll
                        for (int j = 0; j < V; ++j) { c0[j] = A2[j]; c1[j] = 0.f; c2[j] = 0.f; c3[j] = 0.f; n1[j] = A2[j]; n2[j] = 0.f; n3[j] = 0.f; }
#pragma unroll
                        for (int q = RB - 1; q >= 0; --q) {
                            // c0 = c of row start+q; (c1, c2, c3) = rows start+q+1..+3 once computed
                            if (q < RB - 1) {
                                const float nU = coef(start + q, ay.n, ay.ident).nU;
                                const float4 ga = ring4[((sb + q) * 2 + 0) * 32 + lane];
                                const float4 gb = ring4[((sb + q) * 2 + 1) * 32 + lane];
                                const float gg[V] = {ga.x, ga.y, ga.z, ga.w, gb.x, gb.y, gb.z, gb.w};
#pragma unroll
                                for (int j = 0; j < V; ++j) { c3[j] = c2[j]; c2[j] = c1[j]; c1[j] = c0[j]; c0[j] = fmaf(nU, c1[j], gg[j]); }
                                if (q == RB - 2) {
#pragma unroll
                                    for (int j = 0; j < V; ++j) n2[j] = c0[j];
                                }
                                if (q == RB - 3) {
#pragma unroll
                                    for (int j = 0; j < V; ++j) n3[j] = c0[j];
                                }
                            }
                            if (q <= RB - 4) {
                                const int k = start + q + 1;           // window rows k-1..k+2 = c0..c3
                                const int y = k - ay.m;
                                if (y >= ylo && y <= yhi) {
                                    float wy[4];
                                    y_weights(ay, k, wy);
                                    float v[V];
#pragma unroll
                                    for (int j = 0; j < V; ++j) {
                                        const float e = fmaf(wy[3], c3[j], fmaf(wy[2], c2[j], fmaf(wy[1], c1[j], wy[0] * c0[j])));
                                        v[j] = ((xmask >> j) & 1u) ? e : it.fill;
                                    }
                                    store_row<VEC>(it, y, x0, lane_on, v);
                                }
                            }
                        }
                        // the three intervals that straddle into the previous block: rows (s3, s2, s1 | c0, c1, c2)
#pragma unroll
                        for (int e = 0; e < 3; ++e) {
                            const int k = start - e;
                            const int y = k - ay.m;
                            if (y >= ylo && y <= yhi) {
                                float wy[4];
                                y_weights(ay, k, wy);
                                float v[V];
#pragma unroll
                                for (int j = 0; j < V; ++j) {
                                    const float a0 = e == 0 ? s1[j] : (e == 1 ? s2[j] : s3[j]);
                                    const float a1 = e == 0 ? c0[j] : (e == 1 ? s1[j] : s2[j]);
                                    const float a2 = e == 0 ? c1[j] : (e == 1 ? c0[j] : s1[j]);
                                    const float a3 = e == 0 ? c2[j] : (e == 1 ? c1[j] : c0[j]);
                                    const float ev = fmaf(wy[3], a3, fmaf(wy[2], a2, fmaf(wy[1], a1, wy[0] * a0)));
                                    v[j] = ((xmask >> j) & 1u) ? ev : it.fill;
                                }
                                store_row<VEC>(it, y, x0, lane_on, v);
                            }
                        }
#pragma unroll
                        for (int j = 0; j < V; ++j) { s1[j] = n1[j]; s2[j] = n2[j]; s3[j] = n3[j]; }
                    }
#pragma unroll
                    for (int j = 0; j < V; ++j) { A2[j] = A1[j]; A1[j] = g[j]; }
                    pi2 = pi1; pi1 = cy.nU;
                }
            }
        }
    }
}

}  // namespace rs

using namespace rs;

__global__ void __launch_bounds__(32, 8) k_resample(const float* __restrict__ in, int n, int w, int h,
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
    it.XA = (int)blockIdx.x * OUTCOLS - V * HALO_L;
    it.ya = (int)blockIdx.y * BH;
    it.yb = min(it.ya + BH, h);
    if (fp_dev && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0)
        fp_dev[k] = make_int4(it.ax.lo, it.ax.hi, it.ay.lo, it.ay.hi);
    if (vec) warp_item<true>(it, s_ring, threadIdx.x);
    else warp_item<false>(it, s_ring, threadIdx.x);
}

int launch_resample(const float* in, int n, int w, int h, const double* sx_host, const double* sy_host,
                    const double* dshift_dev, float fill, float* out, int32_t* fp_dev, cudaStream_t st)
{
    HostShifts hs;
    if (!dshift_dev)
        for (int k = 0; k < n; ++k) { hs.s[k][0] = sx_host[k]; hs.s[k][1] = sy_host[k]; }
    const int strips = (w + OUTCOLS - 1) / OUTCOLS;
    // bands: enough warps to fill 148 SMs x 8 resident warps, but no band shorter than 64 rows
    // (each band pays ~42 extra rows of warm-up and look-ahead)
    const long long cols = (long long)strips * n;
    long long bands = (148 * 8 + cols - 1) / cols;
    const long long maxb = (h + 63) / 64;
    if (bands > maxb) bands = maxb;
    if (bands < 1) bands = 1;
    int BH = (int)((h + bands - 1) / bands);
    BH = (BH + 7) / 8 * 8;
    const int nb = (h + BH - 1) / BH;
    const int vec = (w % 4 == 0) ? 1 : 0;
    const size_t smem = (size_t)NRING * RB * WARPCOLS * sizeof(float);
    static bool attr_done = false;   // idempotent: the same value every time, so a race is harmless
    if (!attr_done) {
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        attr_done = true;
    }
    dim3 grid(strips, nb, n);
    k_resample<<<grid, 32, smem, st>>>(in, n, w, h, hs, dshift_dev, fill, out, reinterpret_cast<int4*>(fp_dev), BH, vec);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
