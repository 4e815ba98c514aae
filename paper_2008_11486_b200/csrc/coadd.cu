// coadd.cu -- per-pixel rejection co-add along the stack axis (O6; PAPER.md L63, L99,
// L107 "sigma-clipped-mean algorithm", L182).
//
// One thread per output pixel keeps that pixel's N-frame column in registers (NMAX = 8..128
// compile-time capacities; all N loads of a thread are issued before the first use, so a CTA has
// N x 256 x 4 B in flight).  HBM roofline: N*4 B read + 4 B value + 2 B count (+ 4*ceil(N/32) B
// mask) written per pixel.
#include "combine.cuh"
#include "coadd_stream.cuh"

namespace mred {

template <int NMAX, int MODE>
__global__ void __launch_bounds__(256) k_coadd(const float* __restrict__ stack, int n, int w, int h,
                                               const int4* __restrict__ fp_dev, int use_fp,
                                               const __grid_constant__ HostFootprints hfp, float ksigma, int max_iter,
                                               float* __restrict__ out, uint16_t* __restrict__ count,
                                               uint32_t* __restrict__ rejmask)
{
    constexpr int NW = (NMAX + 31) / 32;
    __shared__ int4 s_fp[NMAX];
    __shared__ uint32_t s_in[NW], s_part[NW];
    const size_t np = (size_t)w * h;
    // Classify every frame against the block's 256 consecutive pixels: footprint covers all of them (the
    // usual case: bit in s_in, no per-pixel test), none of them, or some (bit in s_part: per-pixel test).
    {
        const int k = threadIdx.x;
        if (k < NW * 32) {          // only these warps pay for the two integer divisions
            const size_t p0 = (size_t)blockIdx.x * blockDim.x;
            const size_t p1 = min(p0 + blockDim.x, np) - 1;
            const int ya = (int)((unsigned)p0 / (unsigned)w), yb = (int)((unsigned)p1 / (unsigned)w);   // w*h < 2^31 (api.cu)
            const int xa = (int)(p0 - (size_t)ya * w), xb = (int)(p1 - (size_t)yb * w);
            int cls = 0;                                   // 0 none, 1 all, 2 some
            if (k < n) {
                int4 f = make_int4(0, w - 1, 0, h - 1);
                if (use_fp) f = fp_dev ? fp_dev[k] : hfp.fp[k];
                if (k < NMAX) s_fp[k] = f;
                const bool rows_in = ya >= f.z && yb <= f.w, rows_out = yb < f.z || ya > f.w || f.x > f.y;
                if (ya == yb) {
                    const bool cols_in = xa >= f.x && xb <= f.y, cols_out = xb < f.x || xa > f.y;
                    cls = (rows_in && cols_in) ? 1 : ((rows_out || cols_out) ? 0 : 2);
                } else {
                    cls = (rows_in && f.x <= 0 && f.y >= w - 1) ? 1 : (rows_out ? 0 : 2);
                }
            }
            const uint32_t bin = __ballot_sync(0xffffffffu, cls == 1), bpart = __ballot_sync(0xffffffffu, cls == 2);
            if ((k & 31) == 0) { s_in[k >> 5] = bin; s_part[k >> 5] = bpart; }
        }
        __syncthreads();
    }
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const float ABSENT = (MODE == MRED_MEDIAN || MODE == MRED_MEDCLIP) ? CUDART_INF_F : CUDART_NAN_F;
    float v[NMAX];
    uint32_t inside[NW];
#pragma unroll
    for (int i = 0; i < NW; ++i) inside[i] = s_in[i];
#pragma unroll
    for (int i = 0; i < NW; ++i) {
        uint32_t part = s_part[i];
        while (part) {                                     // block-uniform, rarely non-zero (footprint edges): the pixel's
            const int y = (int)((unsigned)p / (unsigned)w), x = (int)((unsigned)p - (unsigned)y * (unsigned)w);   // (x, y) only here
            const int b = __ffs(part) - 1;
            part &= part - 1;
            const int4 f = s_fp[32 * i + b];
            if (x >= f.x && x <= f.y && y >= f.z && y <= f.w) inside[i] |= 1u << b;
        }
    }
    int m = 0, nin = 0;                                    // nin: frames that cover every pixel of the block (block-uniform)
#pragma unroll
    for (int i = 0; i < NW; ++i) { m += __popc(inside[i]); nin += __popc(s_in[i]); }
    const float* src = stack + p;
    if (MODE != MRED_MEDIAN && MODE != MRED_MEDCLIP && NMAX <= 24 && n == NMAX && m == NMAX) {
        // short column, every frame covers this pixel (the usual case; with 32+ frames some lane of the warp
        // nearly always rejects something and the attempt would be wasted): unconditional loads, and a clip loop that only has to
        // find out that nothing is rejected (bit-identical to the general path below, which takes over otherwise)
#pragma unroll
        for (int k = 0; k < NMAX; ++k) { v[k] = __ldcs(src); src += np; }
        float value;
        if (combine_full_noreject<NMAX>(v, MODE == MRED_SIGCLIP, ksigma, max_iter, value)) {
            out[p] = value;
            if (count) count[p] = (uint16_t)NMAX;
            if (rejmask) {
#pragma unroll
                for (int i = 0; i < NW; ++i) rejmask[(size_t)i * np + p] = 0u;
            }
            return;
        }
    } else if (MODE == MRED_MEDIAN && NMAX <= 64 && nin == n) {
        // median, every frame covers the whole block (block-uniform, the usual case): the absent slots are exactly k >= n,
        // so they can be padded on both sides (combine.cuh, median_padded) and the network is pruned to the two middle
        // slots at compile time.  Bit-identical to the general path: the median is the same value either way.
#pragma unroll
        for (int k = 0; k < NMAX; ++k) {
            v[k] = k < n ? __ldcs(src) : pad_slot<NMAX>(k, n);
            src += np;
        }
        out[p] = median_padded<NMAX>(v, n);
        if (count) count[p] = (uint16_t)n;
        if (rejmask) {
            const int words = (n + 31) >> 5;
#pragma unroll
            for (int i = 0; i < NW; ++i)
                if (i < words) rejmask[(size_t)i * np + p] = 0u;
        }
        return;
    } else {
#pragma unroll
        for (int k = 0; k < NMAX; ++k) {
            const bool ok = (inside[k >> 5] >> (k & 31)) & 1u;
            v[k] = ok ? __ldcs(src) : ABSENT;
            src += np;
        }
    }
    Combined r;
    uint32_t rej[(NMAX + 31) / 32];
    if (MODE == MRED_MEDIAN) {
        r = combine_median<NMAX>(v, m);
#pragma unroll
        for (int i = 0; i < (NMAX + 31) / 32; ++i) rej[i] = ~inside[i];
    } else if (MODE == MRED_MEDCLIP) {
        // the sort has lost which value belongs to which frame: a frame was used iff its value lies in the survivors' range,
        // so for the mask the column is read once more (out of L2; only when a mask is asked for)
        float vlo, vhi;
        r = combine_medclip<NMAX>(v, m, ksigma, max_iter, vlo, vhi);
#pragma unroll
        for (int i = 0; i < (NMAX + 31) / 32; ++i) rej[i] = ~inside[i];
        if (rejmask && r.count < m) {
            const float* s2 = stack + p;
#pragma unroll
            for (int k = 0; k < NMAX; ++k) {
                const bool ok = (inside[k >> 5] >> (k & 31)) & 1u;
                if (ok) { const float t = __ldg(s2); if (t < vlo || t > vhi) rej[k >> 5] |= 1u << (k & 31); }
                s2 += np;
            }
        }
    } else {
        r = combine_mean_clip<NMAX>(v, m, MODE == MRED_SIGCLIP, ksigma, max_iter);
#pragma unroll
        for (int i = 0; i < (NMAX + 31) / 32; ++i) rej[i] = 0u;
#pragma unroll
        for (int k = 0; k < NMAX; ++k)
            if (!(v[k] == v[k])) rej[k >> 5] |= 1u << (k & 31);
    }
    out[p] = r.value;
    if (count) count[p] = (uint16_t)r.count;
    if (rejmask) {
        const int words = (n + 31) >> 5;
#pragma unroll
        for (int i = 0; i < (NMAX + 31) / 32; ++i) {
            if (i < words) {
                const int nb = n - 32 * i;
                const uint32_t valid = nb >= 32 ? 0xffffffffu : ((1u << nb) - 1u);
                rejmask[(size_t)i * np + p] = rej[i] & valid;
            }
        }
    }
}

// In-place ascending heap sort of s[0..m) in local memory: O(m log m), where selection by rank counting is O(m^2)
// (median of 255 frames: 38 ms per 512 x 512 plane by counting).
__device__ __forceinline__ void sift_down(float* s, int i, int m)
{
    const float t = s[i];
    while (2 * i + 1 < m) {
        int c = 2 * i + 1;
        if (c + 1 < m && s[c + 1] > s[c]) ++c;
        if (t >= s[c]) break;
        s[i] = s[c];
        i = c;
    }
    s[i] = t;
}
__device__ __forceinline__ void heap_sort(float* s, int m)
{
    for (int i = m / 2 - 1; i >= 0; --i) sift_down(s, i, m);
    for (int e = m - 1; e > 0; --e) {
        const float t = s[0];
        s[0] = s[e];
        s[e] = t;
        sift_down(s, 0, e);
    }
}

// Any N up to 255: the column lives in local memory (L1-backed); dynamic loops.  Correct for every
// n, used only above the largest register capacity.
template <int MODE>
__global__ void __launch_bounds__(128) k_coadd_any(const float* __restrict__ stack, int n, int w, int h,
                                                   const int4* __restrict__ fp_dev, int use_fp,
                                                   const __grid_constant__ HostFootprints hfp, float ksigma, int max_iter,
                                                   float* __restrict__ out, uint16_t* __restrict__ count,
                                                   uint32_t* __restrict__ rejmask)
{
    const size_t np = (size_t)w * h;
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const int y = (int)(p / w), x = (int)(p - (size_t)y * w);
    const int4* fp = fp_dev ? fp_dev : hfp.fp;
    float v[MRED_MAX_STACK];
    unsigned char used[MRED_MAX_STACK];
    int m = 0;
    for (int k = 0; k < n; ++k) {
        bool ok = true;
        if (use_fp) { const int4 f = fp[k]; ok = (x >= f.x) && (x <= f.y) && (y >= f.z) && (y <= f.w); }
        used[k] = ok;
        v[k] = ok ? __ldcs(stack + (size_t)k * np + p) : 0.f;
        m += ok;
    }
    float value = 0.f;
    int cnt = m;
    if (m > 0) {
        if (MODE == MRED_MEDIAN || MODE == MRED_MEDCLIP) {
            // the valid entries, sorted once (heap sort in local memory)
            float s[MRED_MAX_STACK];
            {
                int q = 0;
                for (int k = 0; k < n; ++k) if (used[k]) s[q++] = v[k];
            }
            heap_sort(s, m);
            if (MODE == MRED_MEDIAN) {
                value = 0.5f * s[(m - 1) >> 1] + 0.5f * s[m >> 1];
            } else {
                // NEXT-2 variant (Q29): each pass is centred on the median of the survivors, sigma = their r.m.s.
                // about it; a pass can only reject from the two ends of the sorted survivors, which stay a contiguous
                // range [lo, hi] (combine_medclip does the same on registers); result = mean of the survivors
                int lo = 0, hi = m - 1;
                for (int it = 0; it < max_iter && lo <= hi; ++it) {
                    const int c2 = hi - lo + 1;
                    const float med = 0.5f * s[lo + ((c2 - 1) >> 1)] + 0.5f * s[lo + (c2 >> 1)];
                    float S = 0.f;
                    for (int i = lo; i <= hi; ++i) S = fmaf(s[i] - med, s[i] - med, S);
                    const float thr = fmaf(ksigma, sqrtf(S / (float)c2), 1e-10f * fabsf(med));
                    int nlo = 0, nhi = 0;
                    while (lo + nlo <= hi && s[lo + nlo] - med < -thr) ++nlo;
                    while (hi - nhi >= lo + nlo && s[hi - nhi] - med > thr) ++nhi;
                    if (nlo + nhi == 0) break;
                    lo += nlo;
                    hi -= nhi;
                }
                cnt = hi >= lo ? hi - lo + 1 : 0;
                if (cnt > 0) {
                    const float vlo = s[lo], vhi = s[hi];
                    float sum = 0.f;
                    for (int i = lo; i <= hi; ++i) sum += s[i];
                    const float c = sum / (float)cnt;
                    float r1 = 0.f;
                    for (int i = lo; i <= hi; ++i) r1 += s[i] - c;
                    value = c + r1 / (float)cnt;
                    for (int k = 0; k < n; ++k) if (used[k] && (v[k] < vlo || v[k] > vhi)) used[k] = 0;
                } else {
                    for (int k = 0; k < n; ++k) used[k] = 0;
                }
            }
        } else if (MODE == MRED_MINMAX) {
            // one minimum and one maximum (first occurrences) left out, mean of the rest; fewer than 3 values: plain mean
            float sum = 0.f, mn = CUDART_INF_F, mx = -CUDART_INF_F;
            int imn = -1, imx = -1;
            for (int k = 0; k < n; ++k)
                if (used[k]) { sum += v[k]; if (v[k] < mn) { mn = v[k]; imn = k; } if (v[k] > mx) { mx = v[k]; imx = k; } }
            if (m >= 3) {
                if (imx == imn) { imx = -1; for (int k = 0; k < n && imx < 0; ++k) if (used[k] && k != imn) imx = k; }
                const float c = sum / (float)m;
                float r1 = 0.f;
                for (int k = 0; k < n; ++k) if (used[k]) r1 += v[k] - c;
                value = c + ((r1 - (mn - c)) - (mx - c)) / (float)(m - 2);
                used[imn] = 0; used[imx] = 0;
                cnt = m - 2;
            } else {
                value = sum / (float)m;
            }
        } else {
            float sum = 0.f;
            for (int k = 0; k < n; ++k) if (used[k]) sum += v[k];
            const float c = sum / (float)m;
            float mean = 0.f;
            for (int k = 0; k < n; ++k) if (used[k]) { v[k] -= c; mean += v[k]; }
            mean /= (float)m;
            if (MODE == MRED_SIGCLIP) {
                for (int it = 0; it < max_iter && cnt > 0; ++it) {
                    float S = 0.f;
                    for (int k = 0; k < n; ++k) if (used[k]) S = fmaf(v[k] - mean, v[k] - mean, S);
                    const float thr = fmaf(ksigma, sqrtf(S / (float)cnt), 1e-10f * fabsf(c));
                    int ncnt = 0;
                    float n1 = 0.f;
                    for (int k = 0; k < n; ++k) {
                        if (!used[k]) continue;
                        if (fabsf(v[k] - mean) <= thr) { ++ncnt; n1 += v[k] - mean; } else used[k] = 0;
                    }
                    if (ncnt == cnt) break;
                    cnt = ncnt;
                    if (cnt > 0) {
                        mean += n1 / (float)cnt;
                        float q = 0.f;
                        for (int k = 0; k < n; ++k) if (used[k]) q += v[k] - mean;
                        mean += q / (float)cnt;
                    }
                }
            }
            value = cnt > 0 ? c + mean : 0.f;
        }
    }
    out[p] = value;
    if (count) count[p] = (uint16_t)cnt;
    if (rejmask) {
        const int words = (n + 31) >> 5;
        for (int i = 0; i < words; ++i) {
            uint32_t bits = 0u;
            for (int b = 0; b < 32 && 32 * i + b < n; ++b) if (!used[32 * i + b]) bits |= 1u << b;
            rejmask[(size_t)i * np + p] = bits;
        }
    }
}

template <int NMAX>
static void launch_mode(int mode, dim3 grid, cudaStream_t st, const float* stack, int n, int w, int h,
                        const int4* fp_dev, int use_fp, const HostFootprints& hfp, float ks, int mi, float* out,
                        uint16_t* count, uint32_t* rejmask)
{
    if (mode == MRED_MEDIAN)
        k_coadd<NMAX, MRED_MEDIAN><<<grid, 256, 0, st>>>(stack, n, w, h, fp_dev, use_fp, hfp, ks, mi, out, count, rejmask);
    else if (mode == MRED_MEAN)
        k_coadd<NMAX, MRED_MEAN><<<grid, 256, 0, st>>>(stack, n, w, h, fp_dev, use_fp, hfp, ks, mi, out, count, rejmask);
    else if (mode == MRED_MEDCLIP)
        k_coadd<NMAX, MRED_MEDCLIP><<<grid, 256, 0, st>>>(stack, n, w, h, fp_dev, use_fp, hfp, ks, mi, out, count, rejmask);
    else
        k_coadd<NMAX, MRED_SIGCLIP><<<grid, 256, 0, st>>>(stack, n, w, h, fp_dev, use_fp, hfp, ks, mi, out, count, rejmask);
}

int launch_coadd(const float* stack, int n, int w, int h, const int32_t* fp_host, const int32_t* fp_dev,
                 const mred_comb_opts& o, float* out, uint16_t* count, uint32_t* rejmask, cudaStream_t st)
{
    HostFootprints local;          // passed by value as a kernel parameter (copied at launch)
    const int use_fp = (fp_host || fp_dev) ? 1 : 0;
    if (fp_host)
        for (int k = 0; k < n; ++k)
            local.fp[k] = make_int4(fp_host[4 * k], fp_host[4 * k + 1], fp_host[4 * k + 2], fp_host[4 * k + 3]);
    const size_t np = (size_t)w * h;
    const int4* fpd = reinterpret_cast<const int4*>(fp_dev);
    const float ks = o.ksigma;
    const int mi = o.max_iter;
    if (o.mode != MRED_MEDIAN && o.mode != MRED_MEDCLIP && np % 4 == 0 && np >= (size_t)cs::TPS) {
        // mean / sigma-clipped mean: streaming pass + compacted clip pass on bulk-copy-staged tiles (coadd_stream.cuh);
        // planes whose size is not a multiple of 4 pixels (tiles not 16-byte aligned) keep the register kernels below
        static PerDeviceOnce once;
        int dev;
        if (once.pending(dev)) {
            MRED_CUDA_TRY(cudaFuncSetAttribute(k_coadd_stream, cudaFuncAttributeMaxDynamicSharedMemorySize, MRED_MAX_STACK * cs::TPS * 4));
            MRED_CUDA_TRY(cudaFuncSetAttribute(k_coadd_stream, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
            once.mark(dev);
        }
        CUtensorMap tm;
        const cuuint64_t dims[2] = {(cuuint64_t)np, (cuuint64_t)n};
        const cuuint64_t strides[1] = {(cuuint64_t)np * 4};
        const cuuint32_t box[2] = {(cuuint32_t)cs::TPS, (cuuint32_t)n};
        if (!tma::encode_f32_map(&tm, stack, 2, dims, strides, box)) { set_cuda_error(cudaErrorInvalidValue); return MRED_ECUDA; }
        k_coadd_stream<<<dim3((unsigned)((np + cs::TP - 1) / cs::TP)), cs::TP, (size_t)n * cs::TPS * 4, st>>>(
            tm, n, w, h, fpd, use_fp, local, o.mode, ks, mi, out, count, rejmask);
        MRED_LAUNCH_CHECK();
        return MRED_OK;
    }
    if (o.mode == MRED_MEDCLIP && n > 128) {      // above the largest register capacity: the any-N kernel (heap sort)
        k_coadd_any<MRED_MEDCLIP><<<dim3((unsigned)((np + 127) / 128)), 128, 0, st>>>(stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
        MRED_LAUNCH_CHECK();
        return MRED_OK;
    }
    if (o.mode == MRED_MINMAX) {       // planes whose size is not a multiple of 4: the any-N kernel
        k_coadd_any<MRED_MINMAX><<<dim3((unsigned)((np + 127) / 128)), 128, 0, st>>>(stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
        MRED_LAUNCH_CHECK();
        return MRED_OK;
    }
    if (n <= 128) {
        dim3 grid((unsigned)((np + 255) / 256));
#define MRED_CO(N) launch_mode<N>(o.mode, grid, st, stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask)
        if (n <= 4) MRED_CO(4);
        else if (n <= 5) MRED_CO(5);
        else if (n <= 8) MRED_CO(8);
        else if (n <= 10) MRED_CO(10);
        else if (n <= 12) MRED_CO(12);
        else if (n <= 16) MRED_CO(16);
        else if (n <= 20) MRED_CO(20);
        else if (n <= 24) MRED_CO(24);
        else if (n <= 32) MRED_CO(32);
        else if (n <= 48) MRED_CO(48);
        else if (n <= 60) MRED_CO(60);
        else if (n <= 64) MRED_CO(64);
        else if (n <= 100) MRED_CO(100);
        else MRED_CO(128);
#undef MRED_CO
    } else if (o.mode == MRED_MEDIAN) {
        // 129..255 frames: the sorting network on a 256-slot column (about 100 of the 256 values spill, but with static
        // indices): 279 us per 512 x 512 x 255, where a heap sort with dynamic indexing in local memory (k_coadd_any)
        // takes 5.7 ms and selection by rank counting took 38 ms
        k_coadd<256, MRED_MEDIAN><<<dim3((unsigned)((np + 255) / 256)), 256, 0, st>>>(stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
    } else {
        dim3 grid((unsigned)((np + 127) / 128));
        if (o.mode == MRED_MEDIAN)
            k_coadd_any<MRED_MEDIAN><<<grid, 128, 0, st>>>(stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
        else if (o.mode == MRED_MEAN)
            k_coadd_any<MRED_MEAN><<<grid, 128, 0, st>>>(stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
        else
            k_coadd_any<MRED_SIGCLIP><<<grid, 128, 0, st>>>(stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
    }
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
