// coadd.cu -- per-pixel rejection co-add along the stack axis (O6; PAPER.md L63, L99,
// L107 "sigma-clipped-mean algorithm", L182).
//
// One thread per output pixel keeps that pixel's N-frame column in registers (NMAX = 8..128
// compile-time capacities; all N loads of a thread are issued before the first use, so a CTA has
// N x 256 x 4 B in flight).  HBM roofline: N*4 B read + 4 B value + 2 B count (+ 4*ceil(N/32) B
// mask) written per pixel.
#include "combine.cuh"

namespace mred {

template <int NMAX, int MODE>
__global__ void __launch_bounds__(256) k_coadd(const float* __restrict__ stack, int n, int w, int h,
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
    const float ABSENT = (MODE == MRED_MEDIAN) ? CUDART_INF_F : CUDART_NAN_F;
    float v[NMAX];
    uint32_t inside[(NMAX + 31) / 32];
#pragma unroll
    for (int i = 0; i < (NMAX + 31) / 32; ++i) inside[i] = 0u;
    int m = 0;
#pragma unroll
    for (int k = 0; k < NMAX; ++k) {
        bool ok = k < n;
        if (use_fp && ok) {
            const int4 f = fp[k];
            ok = (x >= f.x) && (x <= f.y) && (y >= f.z) && (y <= f.w);
        }
        v[k] = ok ? __ldcs(stack + (size_t)k * np + p) : ABSENT;
        if (ok) { ++m; inside[k >> 5] |= 1u << (k & 31); }
    }
    Combined r;
    uint32_t rej[(NMAX + 31) / 32];
    if (MODE == MRED_MEDIAN) {
        r = combine_median<NMAX>(v, m);
#pragma unroll
        for (int i = 0; i < (NMAX + 31) / 32; ++i) rej[i] = ~inside[i];
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
        if (MODE == MRED_MEDIAN) {
            // selection by rank counting over the valid entries
            const int ia = (m - 1) >> 1, ib = m >> 1;
            float a = 0.f, b = 0.f;
            for (int i = 0; i < n; ++i) {
                if (!used[i]) continue;
                int rank = 0;
                for (int j = 0; j < n; ++j)
                    if (used[j] && (v[j] < v[i] || (v[j] == v[i] && j < i))) ++rank;
                if (rank == ia) a = v[i];
                if (rank == ib) b = v[i];
            }
            value = 0.5f * a + 0.5f * b;
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
    if (n <= 128) {
        dim3 grid((unsigned)((np + 255) / 256));
        if (n <= 8) launch_mode<8>(o.mode, grid, st, stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
        else if (n <= 16) launch_mode<16>(o.mode, grid, st, stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
        else if (n <= 32) launch_mode<32>(o.mode, grid, st, stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
        else if (n <= 64) launch_mode<64>(o.mode, grid, st, stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
        else launch_mode<128>(o.mode, grid, st, stack, n, w, h, fpd, use_fp, local, ks, mi, out, count, rejmask);
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
