// masters.cu -- master bias / dark / flat construction (O2; the paper uses master frames
// for bias/dark/flat correction, without describing how they are made).
//
//   MB = comb_k(B_k - L_k);  MD = comb_k(D_k - L_k - MB);
//   G_k = F_k - L_k - MB - r MD, r = t_flat/t_dark;  MF = comb_k(G_k/<G_k>) / <comb_k(..)>
//
// <G_k> needs no pass of its own: <G_k> = <F_k> - L_k - <MB> - r<MD>, with <F_k> an exact integer
// sum (k_frame_sums) and <MB>, <MD> fixed-order float64 block sums of the planes just written.
// Per-pixel columns live in registers (combine.cuh).  HBM roofline: every uint16 input read once,
// three float32 planes written (+ MB/MD re-read by the flat pass and the 4 MB normalisation pass,
// both L2-resident).
#include "combine.cuh"

namespace mred {

struct MastersWs {            // layout of the caller's workspace (all 16-byte aligned)
    unsigned long long* os_b; // [nb] overscan sums
    unsigned long long* os_d; // [nd]
    unsigned long long* os_f; // [nf]
    unsigned long long* img_f;// [nf] image-rectangle sums of the flats
    double* part_bd;          // [nblocks][2] block sums of MB, MD
    double* part_f;           // [nblocks]    block sums of the un-normalised MF
    float* inv_gm;            // [nf] 1/<G_k>
    float* inv_mf;            // [1]  1/<MF_raw>
    size_t bytes;
};

static MastersWs carve(void* ws, const Geom& g, int nb, int nd, int nf)
{
    MastersWs m;
    char* p = static_cast<char*>(ws);
    auto take = [&](size_t b) { char* q = p; p += align_up(b, 16); return q; };
    const size_t nblocks = ((size_t)g.w * g.h + 255) / 256;
    m.os_b = reinterpret_cast<unsigned long long*>(take(8 * (size_t)nb));
    m.os_d = reinterpret_cast<unsigned long long*>(take(8 * (size_t)nd));
    m.os_f = reinterpret_cast<unsigned long long*>(take(8 * (size_t)nf));
    m.img_f = reinterpret_cast<unsigned long long*>(take(8 * (size_t)nf));
    m.part_bd = reinterpret_cast<double*>(take(16 * nblocks));
    m.part_f = reinterpret_cast<double*>(take(8 * nblocks));
    m.inv_gm = reinterpret_cast<float*>(take(4 * (size_t)nf));
    m.inv_mf = reinterpret_cast<float*>(take(16));
    m.bytes = (size_t)(p - static_cast<char*>(ws));
    return m;
}

size_t masters_ws_bytes(const Geom& g, int n)
{
    return carve(nullptr, g, n, n, n).bytes;   // n = max(nb, nd, nf) is an upper bound for each
}

// deterministic block sum of one double per thread (256 threads): shuffle tree, then warp 0 adds the
// eight warp totals in index order.  Result valid in thread 0.
__device__ __forceinline__ double block_sum_256(double v, double* s8)
{
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) s8[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < 8; ++i) t += s8[i];
    __syncthreads();
    return t;
}

template <int NMAX, int MODE>
__device__ __forceinline__ float combine_all(float (&v)[NMAX], int n, float ksigma, int max_iter)
{
    if (MODE == MRED_MEDIAN) return combine_median<NMAX>(v, n).value;
    return combine_mean_clip<NMAX>(v, n, MODE == MRED_SIGCLIP, ksigma, max_iter).value;
}

// ---- bias + dark ----------------------------------------------------------------------------
template <int NMAX, int MODE>
__global__ void __launch_bounds__(256) k_masters_bd(const uint16_t* __restrict__ bias, int nb,
                                                    const uint16_t* __restrict__ dark, int nd, Geom g,
                                                    const unsigned long long* __restrict__ os_b,
                                                    const unsigned long long* __restrict__ os_d, float ksigma,
                                                    int max_iter, float* __restrict__ MB, float* __restrict__ MD,
                                                    double* __restrict__ part_bd)
{
    __shared__ float s_lb[MRED_MAX_STACK + 1], s_ld[MRED_MAX_STACK + 1];
    __shared__ double s8[8];
    const long long cnt = (long long)(g.os_x1 - g.os_x0) * g.H;
    for (int k = threadIdx.x; k < nb; k += blockDim.x) s_lb[k] = cnt > 0 ? (float)((double)os_b[k] / (double)cnt) : 0.f;
    for (int k = threadIdx.x; k < nd; k += blockDim.x) s_ld[k] = cnt > 0 ? (float)((double)os_d[k] / (double)cnt) : 0.f;
    __syncthreads();
    const size_t np = (size_t)g.w * g.h, fs = (size_t)g.W * g.H;
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = p < np;
    const float ABSENT = (MODE == MRED_MEDIAN) ? CUDART_INF_F : CUDART_NAN_F;
    float mb = 0.f, md = 0.f;
    if (live) {
        const int y = (int)(p / g.w), x = (int)(p - (size_t)y * g.w);
        const size_t q = (size_t)(y + g.y0) * g.W + (x + g.x0);
        float v[NMAX];
#pragma unroll
        for (int k = 0; k < NMAX; ++k) v[k] = k < nb ? (float)__ldcs(bias + (size_t)k * fs + q) - s_lb[k] : ABSENT;
        mb = combine_all<NMAX, MODE>(v, nb, ksigma, max_iter);
#pragma unroll
        for (int k = 0; k < NMAX; ++k)
            v[k] = k < nd ? ((float)__ldcs(dark + (size_t)k * fs + q) - s_ld[k]) - mb : ABSENT;
        md = combine_all<NMAX, MODE>(v, nd, ksigma, max_iter);
        MB[p] = mb;
        MD[p] = md;
    }
    const double sb = block_sum_256((double)mb, s8);
    const double sd = block_sum_256((double)md, s8);
    if (threadIdx.x == 0) { part_bd[2 * (size_t)blockIdx.x] = sb; part_bd[2 * (size_t)blockIdx.x + 1] = sd; }
}

// ---- <G_k> from the sums (one block) -----------------------------------------------------------
__global__ void __launch_bounds__(256) k_flat_means(const double* __restrict__ part_bd, int nblocks, Geom g, int nf,
                                                    const unsigned long long* __restrict__ os_f,
                                                    const unsigned long long* __restrict__ img_f, double r,
                                                    float* __restrict__ inv_gm)
{
    __shared__ double s8[8];
    __shared__ double s_mean[2];
    double a = 0.0, b = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += blockDim.x) { a += part_bd[2 * (size_t)i]; b += part_bd[2 * (size_t)i + 1]; }
    const double sa = block_sum_256(a, s8);
    const double sb = block_sum_256(b, s8);
    const double np = (double)g.w * (double)g.h;
    if (threadIdx.x == 0) { s_mean[0] = sa / np; s_mean[1] = sb / np; }
    __syncthreads();
    const long long cnt = (long long)(g.os_x1 - g.os_x0) * g.H;
    for (int k = threadIdx.x; k < nf; k += blockDim.x) {
        const double L = cnt > 0 ? (double)os_f[k] / (double)cnt : 0.0;
        const double gm = (double)img_f[k] / np - L - s_mean[0] - r * s_mean[1];
        inv_gm[k] = (float)(1.0 / gm);
    }
}

// ---- flat -----------------------------------------------------------------------------------
template <int NMAX, int MODE>
__global__ void __launch_bounds__(256) k_masters_f(const uint16_t* __restrict__ flat, int nf, Geom g,
                                                   const unsigned long long* __restrict__ os_f,
                                                   const float* __restrict__ inv_gm, float r, float ksigma, int max_iter,
                                                   const float* __restrict__ MB, const float* __restrict__ MD,
                                                   float* __restrict__ MF, double* __restrict__ part_f)
{
    __shared__ float s_lf[MRED_MAX_STACK + 1], s_ig[MRED_MAX_STACK + 1];
    __shared__ double s8[8];
    const long long cnt = (long long)(g.os_x1 - g.os_x0) * g.H;
    for (int k = threadIdx.x; k < nf; k += blockDim.x) {
        s_lf[k] = cnt > 0 ? (float)((double)os_f[k] / (double)cnt) : 0.f;
        s_ig[k] = inv_gm[k];
    }
    __syncthreads();
    const size_t np = (size_t)g.w * g.h, fs = (size_t)g.W * g.H;
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const float ABSENT = (MODE == MRED_MEDIAN) ? CUDART_INF_F : CUDART_NAN_F;
    float mf = 0.f;
    if (p < np) {
        const int y = (int)(p / g.w), x = (int)(p - (size_t)y * g.w);
        const size_t q = (size_t)(y + g.y0) * g.W + (x + g.x0);
        const float off = fmaf(r, MD[p], MB[p]);
        float v[NMAX];
#pragma unroll
        for (int k = 0; k < NMAX; ++k)
            v[k] = k < nf ? (((float)__ldg(flat + (size_t)k * fs + q) - s_lf[k]) - off) * s_ig[k] : ABSENT;
        mf = combine_all<NMAX, MODE>(v, nf, ksigma, max_iter);
        MF[p] = mf;
    }
    const double s = block_sum_256((double)mf, s8);
    if (threadIdx.x == 0) part_f[blockIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_mf_mean(const double* __restrict__ part_f, int nblocks, double np,
                                                 float* __restrict__ inv_mf)
{
    __shared__ double s8[8];
    double a = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += blockDim.x) a += part_f[i];
    const double s = block_sum_256(a, s8);
    if (threadIdx.x == 0) inv_mf[0] = (float)(np / s);
}

__global__ void __launch_bounds__(256) k_mf_scale(float* __restrict__ MF, size_t np, const float* __restrict__ inv_mf)
{
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < np) MF[p] *= inv_mf[0];
}

template <int NMAX>
static void launch_bd(int mode, dim3 grid, cudaStream_t st, const uint16_t* bias, int nb, const uint16_t* dark, int nd,
                      const Geom& g, const MastersWs& m, float ks, int mi, float* MB, float* MD)
{
    if (mode == MRED_MEDIAN)
        k_masters_bd<NMAX, MRED_MEDIAN><<<grid, 256, 0, st>>>(bias, nb, dark, nd, g, m.os_b, m.os_d, ks, mi, MB, MD, m.part_bd);
    else if (mode == MRED_MEAN)
        k_masters_bd<NMAX, MRED_MEAN><<<grid, 256, 0, st>>>(bias, nb, dark, nd, g, m.os_b, m.os_d, ks, mi, MB, MD, m.part_bd);
    else
        k_masters_bd<NMAX, MRED_SIGCLIP><<<grid, 256, 0, st>>>(bias, nb, dark, nd, g, m.os_b, m.os_d, ks, mi, MB, MD, m.part_bd);
}

template <int NMAX>
static void launch_f(int mode, dim3 grid, cudaStream_t st, const uint16_t* flat, int nf, const Geom& g,
                     const MastersWs& m, float r, float ks, int mi, const float* MB, const float* MD, float* MF)
{
    if (mode == MRED_MEDIAN)
        k_masters_f<NMAX, MRED_MEDIAN><<<grid, 256, 0, st>>>(flat, nf, g, m.os_f, m.inv_gm, r, ks, mi, MB, MD, MF, m.part_f);
    else if (mode == MRED_MEAN)
        k_masters_f<NMAX, MRED_MEAN><<<grid, 256, 0, st>>>(flat, nf, g, m.os_f, m.inv_gm, r, ks, mi, MB, MD, MF, m.part_f);
    else
        k_masters_f<NMAX, MRED_SIGCLIP><<<grid, 256, 0, st>>>(flat, nf, g, m.os_f, m.inv_gm, r, ks, mi, MB, MD, MF, m.part_f);
}

#define MRED_BUCKET(n, CALL)                 \
    do {                                     \
        if ((n) <= 4) { CALL(4); }           \
        else if ((n) <= 8) { CALL(8); }      \
        else if ((n) <= 16) { CALL(16); }    \
        else if ((n) <= 32) { CALL(32); }    \
        else if ((n) <= 64) { CALL(64); }    \
        else if ((n) <= 128) { CALL(128); }  \
        else { CALL(256); }                  \
    } while (0)

int launch_build_masters(const Geom& g, const uint16_t* bias, int nb, const uint16_t* dark, int nd, float t_dark,
                         const uint16_t* flat, int nf, float t_flat, const mred_comb_opts& o, float* MB, float* MD,
                         float* MF, void* ws, cudaStream_t st)
{
    const MastersWs m = carve(ws, g, nb, nd, nf);
    int rc;
    if ((rc = launch_frame_sums(bias, g, nb, m.os_b, nullptr, st))) return rc;
    if ((rc = launch_frame_sums(dark, g, nd, m.os_d, nullptr, st))) return rc;
    if ((rc = launch_frame_sums(flat, g, nf, m.os_f, m.img_f, st))) return rc;
    const size_t np = (size_t)g.w * g.h;
    const int nblocks = (int)((np + 255) / 256);
    dim3 grid(nblocks);
    const int nbd = nb > nd ? nb : nd;
    const float r = t_flat / t_dark;
#define CALL_BD(N) launch_bd<N>(o.mode, grid, st, bias, nb, dark, nd, g, m, o.ksigma, o.max_iter, MB, MD)
    MRED_BUCKET(nbd, CALL_BD);
#undef CALL_BD
    MRED_LAUNCH_CHECK();
    k_flat_means<<<1, 256, 0, st>>>(m.part_bd, nblocks, g, nf, m.os_f, m.img_f, (double)t_flat / (double)t_dark, m.inv_gm);
    MRED_LAUNCH_CHECK();
#define CALL_F(N) launch_f<N>(o.mode, grid, st, flat, nf, g, m, r, o.ksigma, o.max_iter, MB, MD, MF)
    MRED_BUCKET(nf, CALL_F);
#undef CALL_F
    MRED_LAUNCH_CHECK();
    k_mf_mean<<<1, 256, 0, st>>>(m.part_f, nblocks, (double)np, m.inv_mf);
    MRED_LAUNCH_CHECK();
    k_mf_scale<<<grid, 256, 0, st>>>(MF, np, m.inv_mf);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
