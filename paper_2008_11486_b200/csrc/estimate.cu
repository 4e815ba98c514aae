// estimate.cu -- per-frame offset estimation from marginal profiles (O4, reading Q10).
// The paper obtains relative positions from FITS WCS headers on the CPU;
// with no headers here the north star asks for an image-based estimate.
//
//   k_profiles : one streaming pass over the frames (the only HBM traffic, N*4wh B): float64 column
//                partial sums per 64-row band and complete float64 row sums, valid-pixel counts.
//   k_finalize : per (frame, axis): fixed-order band sum, mean, median by a shared-memory bitonic sort, subtract.
//   k_correlate: per (frame, axis): C(l) = sum_j a[j] b[j+l], l in [-R, R]; argmax with ties to the
//                smaller |l| then smaller l; 3-point parabola.
// No float atomics: every sum has a fixed order, so the integer result is reproducible.
#include "common.cuh"

namespace mred {

constexpr int PROF_BR = 16;        // rows per band
constexpr int PROF_MAXLEN = 4096;  // longest profile the finalize kernel holds in shared memory

struct EstimateWs {
    double* colpart;  // [n][nbands][w]
    int* colcnt;      // [n][nbands][w]
    double* rowsum;   // [n][h]
    int* rowcnt;      // [n][h]
    double* prof;     // [n][2][plen]  median-subtracted profiles (x then y)
    size_t bytes;
    int nbands, plen;
};

static EstimateWs carve_est(void* ws, int w, int h, int n)
{
    EstimateWs e;
    char* p = static_cast<char*>(ws);
    auto take = [&](size_t b) { char* q = p; p += align_up(b, 16); return q; };
    e.nbands = (h + PROF_BR - 1) / PROF_BR;
    e.plen = w > h ? w : h;
    e.colpart = reinterpret_cast<double*>(take(8 * (size_t)n * e.nbands * w));
    e.colcnt = reinterpret_cast<int*>(take(4 * (size_t)n * e.nbands * w));
    e.rowsum = reinterpret_cast<double*>(take(8 * (size_t)n * h));
    e.rowcnt = reinterpret_cast<int*>(take(4 * (size_t)n * h));
    e.prof = reinterpret_cast<double*>(take(8 * (size_t)n * 2 * e.plen));
    e.bytes = (size_t)(p - static_cast<char*>(ws));
    return e;
}

size_t estimate_ws_bytes(int w, int h, int n) { return carve_est(nullptr, w, h, n).bytes; }

__global__ void __launch_bounds__(256) k_profiles(const float* __restrict__ frames, int w, int h,
                                                  const uint8_t* __restrict__ bad, EstimateWs e, int vec_ok)
{
    __shared__ double s_row[PROF_BR][8];
    __shared__ int s_cnt[PROF_BR][8];
    const int band = blockIdx.x, k = blockIdx.y;
    const int y0 = band * PROF_BR, y1 = min(y0 + PROF_BR, h);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const float* f = frames + (size_t)k * w * h;
    for (int i = threadIdx.x; i < PROF_BR * 8; i += blockDim.x) { (&s_row[0][0])[i] = 0.0; (&s_cnt[0][0])[i] = 0; }
    __syncthreads();
    for (int xc = 0; xc < w; xc += 1024) {
        const int x = xc + 4 * threadIdx.x;
        const int nv = max(0, min(4, w - x));
        double cs[4] = {0.0, 0.0, 0.0, 0.0};
        int cc[4] = {0, 0, 0, 0};
        for (int yb = y0; yb < y1; yb += 4) {       // 4 rows in flight per thread
            float v[4][4];
            bool ok[4][4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
#pragma unroll
                for (int i = 0; i < 4; ++i) { v[u][i] = 0.f; ok[u][i] = false; }
                const int y = yb + u;
                if (y >= y1) continue;
                const size_t p = (size_t)y * w + x;
                if (nv == 4 && vec_ok) {
                    const float4 t = __ldcs(reinterpret_cast<const float4*>(f + p));
                    v[u][0] = t.x; v[u][1] = t.y; v[u][2] = t.z; v[u][3] = t.w;
                    ok[u][0] = ok[u][1] = ok[u][2] = ok[u][3] = true;
                    if (bad) {
                        const uchar4 b = __ldg(reinterpret_cast<const uchar4*>(bad + p));
                        ok[u][0] = !b.x; ok[u][1] = !b.y; ok[u][2] = !b.z; ok[u][3] = !b.w;
                    }
                } else {
                    for (int i = 0; i < nv; ++i) { v[u][i] = __ldcs(f + p + i); ok[u][i] = bad ? !__ldg(bad + p + i) : true; }
                }
            }
            double rs[4] = {0.0, 0.0, 0.0, 0.0};
            int rc[4] = {0, 0, 0, 0};
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (ok[u][i]) { const double d = (double)v[u][i]; cs[i] += d; ++cc[i]; rs[u] += d; ++rc[u]; }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int u = 0; u < 4; ++u) { rs[u] += __shfl_xor_sync(0xffffffffu, rs[u], o); rc[u] += __shfl_xor_sync(0xffffffffu, rc[u], o); }
            if (lane == 0) {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (yb + u < y1) { s_row[yb + u - y0][warp] += rs[u]; s_cnt[yb + u - y0][warp] += rc[u]; }
            }
        }
        for (int i = 0; i < nv; ++i) {
            e.colpart[((size_t)k * e.nbands + band) * w + x + i] = cs[i];
            e.colcnt[((size_t)k * e.nbands + band) * w + x + i] = cc[i];
        }
    }
    __syncthreads();
    for (int r = threadIdx.x; r < y1 - y0; r += blockDim.x) {
        double t = 0.0;
        int c = 0;
        for (int i = 0; i < 8; ++i) { t += s_row[r][i]; c += s_cnt[r][i]; }
        e.rowsum[(size_t)k * h + y0 + r] = t;
        e.rowcnt[(size_t)k * h + y0 + r] = c;
    }
}

// grid (n, 2): axis 0 = x profile (length w), axis 1 = y profile (length h).  Mean profile, then its median
// by a bitonic sort in shared memory (invalid lines sort to the end as +inf), then the subtraction.
__global__ void __launch_bounds__(1024) k_finalize(int w, int h, EstimateWs e)
{
    __shared__ double s_p[PROF_MAXLEN];
    __shared__ int s_m;
    const int k = blockIdx.x, axis = blockIdx.y;
    const int len = axis == 0 ? w : h;
    int P = 1;
    while (P < len) P <<= 1;
    if (threadIdx.x == 0) s_m = 0;
    __syncthreads();
    double* out = e.prof + ((size_t)k * 2 + axis) * e.plen;
    const double INF = __longlong_as_double(0x7ff0000000000000LL);
    int mine = 0;
    for (int i = threadIdx.x; i < P; i += blockDim.x) {
        double v = INF;
        if (i < len) {
            double s = 0.0;
            int c = 0;
            if (axis == 0) {
                for (int b = 0; b < e.nbands; ++b) {
                    s += e.colpart[((size_t)k * e.nbands + b) * w + i];
                    c += e.colcnt[((size_t)k * e.nbands + b) * w + i];
                }
            } else {
                s = e.rowsum[(size_t)k * h + i];
                c = e.rowcnt[(size_t)k * h + i];
            }
            if (c > 0) { v = s / (double)c; ++mine; }
            out[i] = v;
        }
        s_p[i] = v;
    }
    if (mine) atomicAdd(&s_m, mine);
    __syncthreads();
    for (int kk = 2; kk <= P; kk <<= 1) {
        for (int j = kk >> 1; j > 0; j >>= 1) {
            for (int i = threadIdx.x; i < P; i += blockDim.x) {
                const int l = i ^ j;
                if (l > i) {
                    const double a = s_p[i], b = s_p[l];
                    const bool up = (i & kk) == 0;
                    if ((a > b) == up) { s_p[i] = b; s_p[l] = a; }
                }
            }
            __syncthreads();
        }
    }
    const int m = s_m;
    double med = 0.0;
    if (m > 0) {
        const double a = s_p[(m - 1) >> 1], b = s_p[m >> 1];
        med = (m & 1) ? a : 0.5 * (a + b);
    }
    for (int i = threadIdx.x; i < len; i += blockDim.x) {
        const double v = out[i];
        out[i] = (v == INF) ? 0.0 : v - med;
    }
}

// grid (n, 2), block 1024: one lag per warp and round
__global__ void __launch_bounds__(1024) k_correlate(int w, int h, int n, int ref, int R, EstimateWs e,
                                                   int32_t* __restrict__ ishift, double* __restrict__ shift)
{
    __shared__ double s_C[2 * MRED_MAX_LAG + 1];
    const int k = blockIdx.x, axis = blockIdx.y;
    if (k == ref) {
        if (threadIdx.x == 0) { ishift[2 * k + axis] = 0; shift[2 * k + axis] = 0.0; }
        return;
    }
    const int len = axis == 0 ? w : h;
    const double* a = e.prof + ((size_t)ref * 2 + axis) * e.plen;
    const double* b = e.prof + ((size_t)k * 2 + axis) * e.plen;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int l = -R + warp; l <= R; l += 32) {
        const int j0 = max(0, -l), j1 = min(len, len - l);
        double s = 0.0;
        for (int j = j0 + lane; j < j1; j += 32) s = fma(a[j], b[j + l], s);
        s = warp_sum(s);
        if (lane == 0) s_C[l + R] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int best = 0;
        for (int l = -R; l <= R; ++l) {
            const double c = s_C[l + R], cb = s_C[best + R];
            const int al = l < 0 ? -l : l, ab = best < 0 ? -best : best;
            if (c > cb || (c == cb && (al < ab || (al == ab && l < best)))) best = l;
        }
        double delta = 0.0;
        const int ab = best < 0 ? -best : best;
        if (ab < R) {
            const double cm = s_C[best - 1 + R], c0 = s_C[best + R], cp = s_C[best + 1 + R];
            const double den = cm - 2.0 * c0 + cp;
            if (den < 0.0) {
                delta = 0.5 * (cm - cp) / den;
                delta = delta > 0.5 ? 0.5 : (delta < -0.5 ? -0.5 : delta);
            }
        }
        ishift[2 * k + axis] = best;
        shift[2 * k + axis] = (double)best + delta;
    }
}

int launch_estimate(const float* frames, int n, int w, int h, int ref, int max_lag, const uint8_t* bad,
                    int32_t* ishift, double* shift, void* ws, cudaStream_t st)
{
    const EstimateWs e = carve_est(ws, w, h, n);
    const int vec_ok = (w % 4 == 0) ? 1 : 0;
    k_profiles<<<dim3(e.nbands, n), 256, 0, st>>>(frames, w, h, bad, e, vec_ok);
    MRED_LAUNCH_CHECK();
    k_finalize<<<dim3(n, 2), 1024, 0, st>>>(w, h, e);
    MRED_LAUNCH_CHECK();
    k_correlate<<<dim3(n, 2), 1024, 0, st>>>(w, h, n, ref, max_lag, e, ishift, shift);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
