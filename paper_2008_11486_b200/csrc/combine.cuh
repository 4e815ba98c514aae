// combine.cuh -- per-pixel combine of an N-frame column held in registers (O6):
// median (Batcher odd-even merge sorting network), mean, k-sigma-clipped mean.
// Used by the master-frame kernels (all N values valid) and by the co-add kernel (values outside a
// frame's footprint are absent).  Everything is fully unrolled over the compile-time capacity NMAX
// so that v[] lives in registers.
#pragma once
#include "common.cuh"
#include <math_constants.h>

namespace mred {

// Batcher's odd-even merge sort as a fixed compare-exchange network on NMAX (power of two) slots.
// The (p, k) stages are template parameters so that every loop bound is a compile-time constant
// and the whole network unrolls onto registers.
template <int NMAX, int P, int K>
__device__ __forceinline__ void oem_stage(float (&v)[NMAX])
{
#pragma unroll
    for (int j = K % P; j + K < NMAX; j += 2 * K) {
#pragma unroll
        for (int i = 0; i < K; ++i) {
            if (i + j + K < NMAX && ((i + j) / (2 * P) == (i + j + K) / (2 * P))) {
                const float a = v[i + j], b = v[i + j + K];
                v[i + j] = fminf(a, b);
                v[i + j + K] = fmaxf(a, b);
            }
        }
    }
}
template <int NMAX, int P, int K>
struct OemK {
    static __device__ __forceinline__ void run(float (&v)[NMAX])
    {
        oem_stage<NMAX, P, K>(v);
        if constexpr (K > 1) OemK<NMAX, P, K / 2>::run(v);
    }
};
template <int NMAX, int P>
struct OemP {
    static __device__ __forceinline__ void run(float (&v)[NMAX])
    {
        OemK<NMAX, P, P>::run(v);
        if constexpr (2 * P < NMAX) OemP<NMAX, 2 * P>::run(v);
    }
};
template <int NMAX>
__device__ __forceinline__ void sort_network(float (&v)[NMAX])
{
    if constexpr (NMAX > 1) OemP<NMAX, 1>::run(v);
}

// Result of one column.
struct Combined {
    float value;
    int count;
};

// Median of the m valid entries; absent entries must hold +INF on entry (they sort to the end).
template <int NMAX>
__device__ __forceinline__ Combined combine_median(float (&v)[NMAX], int m)
{
    sort_network<NMAX>(v);
    float a = 0.f, b = 0.f;
    if (NMAX <= 16 && m == NMAX) {   // full short column (the usual case): fixed slots (measured slower for 20+ slots)
        a = v[(NMAX - 1) >> 1];
        b = v[NMAX >> 1];
    } else {
        const int ia = (m - 1) >> 1, ib = m >> 1;
#pragma unroll
        for (int i = 0; i < NMAX; ++i) {
            a = (i == ia) ? v[i] : a;
            b = (i == ib) ? v[i] : b;
        }
    }
    Combined r;
    r.count = m;
    r.value = m > 0 ? 0.5f * a + 0.5f * b : 0.f;     // a == b for odd m: exact
    return r;
}

// Median of a partly filled column whose absent slots the caller has PADDED ON BOTH SIDES: of the NMAX - n absent slots,
// L = (NMAX - n) >> 1 hold -INF and the others +INF (pad_slot below).  The n values then sort into slots [L, L + n), and the
// middle of that range is the same pair of slots whatever n is -- so, as for a full column, the outputs are compile-time
// slots and the compiler prunes the network to the comparators that reach them (the +INF-only padding of combine_median
// moves the middle with n: every slot is a possible output, the whole network stays).  n >= 1.
//   NMAX even: slots NMAX/2 - 1 and NMAX/2 for even n, slot NMAX/2 - 1 alone for odd n;
//   NMAX odd:  slot (NMAX-1)/2 alone for odd n, slots (NMAX-3)/2 and (NMAX-1)/2 for even n.
template <int NMAX>
__device__ __forceinline__ float pad_slot(int k, int n)      // value of absent slot k >= n
{
    return k < n + ((NMAX - n) >> 1) ? -CUDART_INF_F : CUDART_INF_F;
}
template <int NMAX>
__device__ __forceinline__ float median_padded(float (&v)[NMAX], int n)
{
    sort_network<NMAX>(v);
    float a, b;
    if (NMAX == 1) { a = v[0]; b = a; }
    else if (NMAX % 2 == 0) { a = v[NMAX / 2 - 1]; b = (n & 1) ? a : v[NMAX / 2]; }
    else { b = v[(NMAX - 1) / 2]; a = (n & 1) ? b : v[NMAX >= 3 ? (NMAX - 3) / 2 : 0]; }
    return 0.5f * a + 0.5f * b;                      // a == b for odd n: exact
}

// Median-centred clip (Q29): each pass is centred on the median of the survivors, sigma =
// their r.m.s. about it, keep |v - med| <= k sigma; the result is the mean of the survivors.  The column is SORTED once
// (absent entries hold +INF and sort to the end); a pass can only reject from the two ends of the sorted survivors, so
// they stay a contiguous range [lo, hi], whose median is the middle slot(s).  On exit [vlo, vhi] is the value range of
// the survivors (empty: vlo > vhi): frame k was used iff its value lies inside, which is how the caller builds the mask.
template <int NMAX>
__device__ __forceinline__ Combined combine_medclip(float (&v)[NMAX], int m, float ksigma, int max_iter, float& vlo, float& vhi)
{
    Combined r;
    r.count = m;
    r.value = 0.f;
    vlo = CUDART_INF_F;
    vhi = -CUDART_INF_F;
    if (m <= 0) return r;
    sort_network<NMAX>(v);
    int lo = 0, hi = m - 1;
    for (int it = 0; it < max_iter && lo <= hi; ++it) {
        const int cnt = hi - lo + 1;
        const int ia = lo + ((cnt - 1) >> 1), ib = lo + (cnt >> 1);
        float a = 0.f, b = 0.f;
#pragma unroll
        for (int i = 0; i < NMAX; ++i) {
            a = (i == ia) ? v[i] : a;
            b = (i == ib) ? v[i] : b;
        }
        const float med = 0.5f * a + 0.5f * b;
        float S = 0.f;
#pragma unroll
        for (int i = 0; i < NMAX; ++i) {
            const float d = v[i] - med;
            S = (i >= lo && i <= hi) ? fmaf(d, d, S) : S;
        }
        const float thr = fmaf(ksigma, sqrtf(S / (float)cnt), 1e-10f * fabsf(med));
        int nlo = 0, nhi = 0;
#pragma unroll
        for (int i = 0; i < NMAX; ++i) {
            const float d = v[i] - med;
            const bool in = i >= lo && i <= hi;
            nlo += (in && d < -thr) ? 1 : 0;
            nhi += (in && d > thr) ? 1 : 0;
        }
        if (nlo + nhi == 0) break;
        lo += nlo;
        hi -= nhi;
    }
    const int cnt = hi - lo + 1;
    r.count = cnt > 0 ? cnt : 0;
    if (cnt > 0) {
        float sum = 0.f;
#pragma unroll
        for (int i = 0; i < NMAX; ++i) {
            const bool in = i >= lo && i <= hi;
            sum += in ? v[i] : 0.f;
            vlo = (i == lo) ? v[i] : vlo;
            vhi = (i == hi) ? v[i] : vhi;
        }
        const float c = sum / (float)cnt;
        float r1 = 0.f;
#pragma unroll
        for (int i = 0; i < NMAX; ++i) r1 += (i >= lo && i <= hi) ? v[i] - c : 0.f;
        r.value = c + r1 / (float)cnt;
    }
    return r;
}

// Fast path of the mean / sigma-clipped mean for a column whose NMAX entries are all present: the same float
// operations in the same order as combine_mean_clip (so the same bits), without the absent-entry bookkeeping,
// and v[] is left untouched.  Returns false when the first clip pass would reject something: the caller then runs
// combine_mean_clip on the same values.
template <int NMAX>
__device__ __forceinline__ bool combine_full_noreject(const float (&v)[NMAX], bool clip, float ksigma, int max_iter, float& value)
{
    float sum = 0.f;
#pragma unroll
    for (int i = 0; i < NMAX; ++i) sum += v[i];
    const float c = sum / (float)NMAX;
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int i = 0; i < NMAX; ++i) { const float d = v[i] - c; s1 += d; s2 = fmaf(d, d, s2); }
    const float mean = s1 / (float)NMAX;
    if (clip && max_iter > 0) {
        const float S = fmaxf(s2 - mean * s1, 0.f);
        const float thr = fmaf(ksigma, sqrtf(S / (float)NMAX), 1e-10f * fabsf(c));
        bool any = false;
#pragma unroll
        for (int i = 0; i < NMAX; ++i) any = any || (fabsf((v[i] - c) - mean) > thr);
        if (any) return false;
    }
    value = c + mean;
    return true;
}

// Mean / sigma-clipped mean.  On entry absent entries hold NaN and `m` counts the valid ones;
// on exit every entry that was not used holds NaN (so the caller can build the rejection mask).
//   c      = sum(v)/m                       (float32 approximation of the mean)
//   d_i    = v_i - c                        (exact-ish: inliers are close to c)
//   pass:  keep iff |d - mean| <= k sqrt(S/cnt), mean = survivors' mean (about c), S = their centred
//          sum of squares.  The sweep that applies the test also accumulates the survivors' first
//          and second moments about the old mean, from which the new (mean, S) follow; when the
//          mean moved by a good fraction of sigma (a large outlier left) S is recomputed about the
//          new mean in a sweep of its own, which keeps the moment form free of cancellation.
template <int NMAX>
__device__ __forceinline__ Combined combine_mean_clip(float (&v)[NMAX], int m, bool clip, float ksigma, int max_iter)
{
    Combined r;
    r.count = m;
    r.value = 0.f;
    if (m <= 0) return r;
    float sum = 0.f;
#pragma unroll
    for (int i = 0; i < NMAX; ++i) sum += (v[i] == v[i]) ? v[i] : 0.f;
    const float c = sum / (float)m;
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int i = 0; i < NMAX; ++i) {
        const float d = v[i] - c;            // NaN stays NaN
        v[i] = d;
        if (d == d) { s1 += d; s2 = fmaf(d, d, s2); }
    }
    int cnt = m;
    float mean = s1 / (float)cnt;            // mean of the survivors, in d-space (about c)
    float S = fmaxf(s2 - mean * s1, 0.f);    // centred sum of squares of the survivors
    if (clip) {
        for (int it = 0; it < max_iter; ++it) {
            // + 1e-10|c|: identical inputs give S = 0 while t carries a few ulp(d) of rounding from the
            // running sums; the slack (1e-7 ADU at 1000 ADU) keeps them, and is far below any tie margin
            const float thr = fmaf(ksigma, sqrtf(S / (float)cnt), 1e-10f * fabsf(c));
            // cheap look first: most columns lose nothing in a pass (NaN compares false: absent entries never count)
            // (only for short columns: with 32+ frames some lane of the warp nearly always rejects, and the look costs a sweep)
            if (NMAX <= 24) {
                bool any = false;
#pragma unroll
                for (int i = 0; i < NMAX; ++i) any = any || (fabsf(v[i] - mean) > thr);
                if (!any) break;
            }
            float n1 = 0.f, n2 = 0.f;
            int ncnt = 0;
#pragma unroll
            for (int i = 0; i < NMAX; ++i) {
                const float t = v[i] - mean;
                const bool keep = fabsf(t) <= thr;        // false for NaN (absent / already rejected)
                v[i] = keep ? v[i] : CUDART_NAN_F;
                if (keep) { ++ncnt; n1 += t; n2 = fmaf(t, t, n2); }
            }
            if (ncnt == cnt) break;                       // nothing rejected
            cnt = ncnt;
            if (cnt == 0) break;
            const float dm = n1 / (float)cnt;             // shift of the mean caused by the rejections
            mean += dm;
            S = fmaxf(n2 - dm * n1, 0.f);                 // = sum t^2 - cnt dm^2
            if (dm * dm * (float)cnt > 0.25f * S) {
                // the mean moved by a good fraction of sigma (a large outlier left): the moment form
                // above cancels, so take the second moment about the new mean in a sweep of its own
                float q1 = 0.f, q2 = 0.f;
#pragma unroll
                for (int i = 0; i < NMAX; ++i) {
                    const float t = v[i] - mean;
                    if (t == t) { q1 += t; q2 = fmaf(t, t, q2); }
                }
                const float dq = q1 / (float)cnt;
                mean += dq;
                S = fmaxf(q2 - dq * q1, 0.f);
            }
        }
    }
    r.count = cnt;
    r.value = cnt > 0 ? c + mean : 0.f;
    return r;
}

}  // namespace mred
