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
    unsigned long long* os;   // [nb + nd + nf] overscan sums (bias, dark, flat frames in that order)
    unsigned long long* img_f;// [nf] image-rectangle sums of the flats
    unsigned int* ticket;     // [3] block counters of the two combine kernels and of the sums kernel (zeroed with the sums)
    float* lev;               // [nb + nd + nf] overscan levels as float32 (written by the last block of k_master_sums)
    double* part_bd;          // [nblocks][2] block sums of MB, MD
    double* part_f;           // [nblocks]    block sums of the un-normalised MF
    float* inv_gm;            // [nf] 1/<G_k>
    float* inv_mf;            // [1]  1/<MF_raw>
    size_t zero_bytes;        // os, img_f, ticket are contiguous from os: one memset
    size_t bytes;
};

constexpr int MPX = 2;        // pixels per thread in the combine kernels (one 32-bit load per frame)
// Threads per block of the combine kernels.  Long columns (60+ registers per thread) run in blocks of 128: measured at 20
// frames the kernels themselves gain 2 % and bench.py's 6-stream step 2.7 % (1.84 -> 1.79 ms: a block of 128 threads finds
// room on an SM that other groups' kernels share, one of 256 has to wait for a quarter of it); short columns keep 256 (at
// 10 frames blocks of 128 were 12-19 % SLOWER: 59 -> 66 us at 1024^2, 528 -> 628 us at 4096^2).
constexpr int MT_MAX = 256, MT_MIN = 128;
template <int NMAX> __host__ __device__ constexpr int masters_threads() { return NMAX >= 16 ? MT_MIN : MT_MAX; }

static MastersWs carve(void* ws, const Geom& g, int nb, int nd, int nf)
{
    MastersWs m;
    char* p = static_cast<char*>(ws);
    auto take = [&](size_t b) { char* q = p; p += align_up(b, 16); return q; };
    const size_t nblocks = ((size_t)g.w * g.h + MT_MIN - 1) / MT_MIN;   // upper bound for either pixels-per-thread and block size
    m.os = reinterpret_cast<unsigned long long*>(take(8 * (size_t)(nb + nd + nf)));
    m.img_f = reinterpret_cast<unsigned long long*>(take(8 * (size_t)nf));
    m.ticket = reinterpret_cast<unsigned int*>(take(16));
    m.zero_bytes = (size_t)(p - static_cast<char*>(ws));
    m.part_bd = reinterpret_cast<double*>(take(16 * nblocks));
    m.part_f = reinterpret_cast<double*>(take(8 * nblocks));
    m.inv_gm = reinterpret_cast<float*>(take(4 * (size_t)nf));
    m.lev = reinterpret_cast<float*>(take(4 * (size_t)(nb + nd + nf)));
    m.inv_mf = reinterpret_cast<float*>(take(16));
    m.bytes = (size_t)(p - static_cast<char*>(ws));
    return m;
}

size_t masters_ws_bytes(const Geom& g, int n)
{
    return carve(nullptr, g, n, n, n).bytes;   // n = max(nb, nd, nf) is an upper bound for each
}

// Exact integer sums of all three stacks in one launch: overscan columns of every frame (the first nos * (nb+nd+nf)
// blocks: one thread per row), and the image rectangle of the flats for <F_k> (the remaining nimg * nf blocks: one
// row per warp, coalesced, 16 loads in flight per lane).  1-D grid, block 256; integer atomics -> bit-exact.
__global__ void __launch_bounds__(256) k_master_sums(const uint16_t* __restrict__ bias, int nb,
                                                     const uint16_t* __restrict__ dark, int nd,
                                                     const uint16_t* __restrict__ flat, int nf, Geom g, int nos, int nimg,
                                                     unsigned long long* __restrict__ os,
                                                     unsigned long long* __restrict__ img_f, unsigned int* __restrict__ ticket,
                                                     float* __restrict__ lev, int pair_ok)
{
    __shared__ unsigned long long s_w[8];
    const size_t fs = (size_t)g.W * g.H;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nall = nb + nd + nf;
    int b = blockIdx.x;
    unsigned long long* dst;
    unsigned long long s = 0;
    if (b < nos * nall) {
        const int k = b / nos, c = b - k * nos;
        const uint16_t* f = k < nb ? bias + (size_t)k * fs : (k < nb + nd ? dark + (size_t)(k - nb) * fs : flat + (size_t)(k - nb - nd) * fs);
        const int r = c * blockDim.x + threadIdx.x;
        if (r < g.H && g.os_x1 > g.os_x0) s = overscan_row_sum(f, g.W, g.os_x0, g.os_x1, r);
        dst = os + k;
    } else {
        b -= nos * nall;                               // image sums: flats only
        const int kf = b / nimg, c = b - kf * nimg;
        const uint16_t* f = flat + (size_t)kf * fs;
        const int r = g.y0 + c * 8 + warp;
        const bool live = r < g.y0 + g.h;
        const uint16_t* row = f + (size_t)(live ? r : g.y0) * g.W;
        if (!live) {
        } else if (pair_ok) {      // two pixels per 32-bit load, 16 independent loads in flight
            const unsigned int* row2 = reinterpret_cast<const unsigned int*>(row + g.x0);
            const int w2 = g.w >> 1;
            int x = lane;
            for (; x + 15 * 32 < w2; x += 16 * 32) {
                unsigned int v[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) v[u] = __ldg(row2 + x + 32 * u);
                unsigned int t = 0;
#pragma unroll
                for (int u = 0; u < 16; ++u) t += (v[u] & 0xffffu) + (v[u] >> 16);     // 32 x 65535 < 2^32
                s += t;
            }
            for (; x < w2; x += 32) { const unsigned int v = __ldg(row2 + x); s += (v & 0xffffu) + (v >> 16); }
        } else {
            for (int x = g.x0 + lane; x < g.x0 + g.w; x += 32) s += __ldg(row + x);
        }
        dst = img_f + kf;
    }
    s = warp_sum(s);
    if (lane == 0) s_w[warp] = s;
    __syncthreads();
    if (warp != 0) return;
    // warp 0: the block's total, then the ticket; the LAST block to arrive turns every overscan sum into its float32 level
    // (one float64 division per frame, done once here instead of by every block of the combine kernels)
    int last = 0;
    if (lane == 0) {
        unsigned long long t = 0;
        for (int i = 0; i < 8; ++i) t += s_w[i];
        if (t) atomicAdd(dst, t);
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    last = __shfl_sync(0xffffffffu, last, 0);
    if (!last) return;
    __threadfence();
    const long long cnt = (long long)(g.os_x1 - g.os_x0) * g.H;
    for (int k = lane; k < nall; k += 32) lev[k] = cnt > 0 ? (float)((double)__ldcg(os + k) / (double)cnt) : 0.f;
}

template <int NMAX, int MODE>
__device__ __forceinline__ float combine_all(float (&v)[NMAX], int n, float ksigma, int max_iter)
{
    if (MODE == MRED_MEDIAN) return median_padded<NMAX>(v, n);       // absent slots: absent_slot below
    return combine_mean_clip<NMAX>(v, n, MODE == MRED_SIGCLIP, ksigma, max_iter).value;
}

// What slot k >= n of a partly filled bucket holds: NaN for the mean / clip sweeps (skipped), -INF / +INF for the median
// (combine.cuh, median_padded: the middle of the sorted column then sits in fixed slots and the network is pruned as for
// a full bucket: 25 frames in the bucket of 32, 205 -> 170 us for the three masters).
template <int NMAX, int MODE>
__device__ __forceinline__ float absent_slot(int k, int n)
{
    return MODE == MRED_MEDIAN ? pad_slot<NMAX>(k, n) : CUDART_NAN_F;
}

// PX pixels of one frame at p (PX = 2: one aligned 32-bit load).  uint16 -> float32 stays on the conversion unit (I2F.U16
// picks its half of the register by itself, so the unpacking costs no ALU instruction): these kernels are bound by the ALU
// pipe (FMNMX of the median network, 70 % busy at N = 20), and the PRMT + FADD form that avoids I2F measured 3 % slower.
// base + k frames: one 32 x 32 -> 64-bit multiply-add (IMAD.WIDE.U32, FMA pipe) per load.  A frame is < 2^31 pixels
// (geom_ok), so its size in bytes fits 32 bits; pointer increments would cost two ALU-pipe additions per load, and the
// ALU pipe is what bounds these kernels.
__device__ __forceinline__ const uint16_t* frame_ptr(const uint16_t* base, int k, unsigned int frame_bytes)
{
    return reinterpret_cast<const uint16_t*>(reinterpret_cast<const char*>(base) + (unsigned long long)(unsigned int)k * frame_bytes);
}

template <int PX>
__device__ __forceinline__ void load_px(const uint16_t* p, int nv, float (&o)[PX])
{
    if (PX == 2) {
        const unsigned int v = __ldcs(reinterpret_cast<const unsigned int*>(p));
        o[0] = (float)(v & 0xffffu);
        o[PX - 1] = (float)(v >> 16);
    } else if (PX == 1) {
        o[0] = (float)__ldcs(p);          // the caller's pixel exists (nv == 1): no predicate on the load
    } else {
#pragma unroll
        for (int i = 0; i < PX; ++i) o[i] = i < nv ? (float)__ldcs(p + i) : 0.f;
    }
}

// ---- bias + dark; the last block turns the block sums into 1/<G_k> of every flat ----------------
// FULL: both stacks hold exactly NMAX frames (the usual case), so every "k < n" test below is a compile-time
// constant: no predicates, no absent-entry selects (a quarter of the instructions of this issue-bound kernel)
template <int NMAX, int MODE, int PX, bool FULL>
__global__ void __launch_bounds__(masters_threads<NMAX>()) k_masters_bd(const uint16_t* __restrict__ bias, int nb,
                                                    const uint16_t* __restrict__ dark, int nd, int nf, Geom g,
                                                    MastersWs m, double r, float ksigma, int max_iter,
                                                    float* __restrict__ MB, float* __restrict__ MD)
{
    __shared__ float s_lb[MRED_MAX_STACK + 1], s_ld[MRED_MAX_STACK + 1];
    const long long cnt = (long long)(g.os_x1 - g.os_x0) * g.H;
    for (int k = threadIdx.x; k < nb; k += blockDim.x) s_lb[k] = m.lev[k];
    for (int k = threadIdx.x; k < nd; k += blockDim.x) s_ld[k] = m.lev[nb + k];
    __syncthreads();
    const size_t fs = (size_t)g.W * g.H;
    const unsigned int fsb = (unsigned int)(fs * 2);
    const int wg = (g.w + PX - 1) / PX;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    float mb[PX], md[PX];
#pragma unroll
    for (int i = 0; i < PX; ++i) { mb[i] = 0.f; md[i] = 0.f; }
    if (gid < (long long)g.h * wg) {
        const int y = (int)((unsigned)gid / (unsigned)wg), x = (int)((unsigned)gid - (unsigned)y * (unsigned)wg) * PX;   // w*h < 2^31
        const int nv = min(PX, g.w - x);
        const size_t q = (size_t)(y + g.y0) * g.W + (x + g.x0);
        const size_t p = (size_t)y * g.w + x;
        // up to 32 frames every load of both stacks is issued before the first median starts (address = base + k * frame:
        // one multiply-add per load); longer columns load the darks after the bias median -- two columns of 64+ values do
        // not fit the register file together (128 frames: 255 registers and spills with both, 167 without: 1.45 -> 1.00 ms)
        constexpr bool BOTH = NMAX <= 32;
        float v[PX][NMAX], dk[PX][BOTH ? NMAX : 1];
        const uint16_t* pb = bias + q;
        const uint16_t* pd = dark + q;
#pragma unroll
        for (int k = 0; k < NMAX; ++k) {
            float o[PX], od[PX];
#pragma unroll
            for (int i = 0; i < PX; ++i) { o[i] = 0.f; od[i] = 0.f; }
            // a partly filled bucket re-reads the last frame for the slots beyond it (an L1 hit) instead of predicating
            // the load: ptxas put the conversion of a predicated load right behind it, so a thread had ONE load in
            // flight at a time (64 frames: 945 us for this kernel, 3 % of the DRAM bandwidth, every warp waiting)
            load_px<PX>(frame_ptr(pb, FULL ? k : min(k, nb - 1), fsb), nv, o);
            if (BOTH) load_px<PX>(frame_ptr(pd, FULL ? k : min(k, nd - 1), fsb), nv, od);
#pragma unroll
            for (int i = 0; i < PX; ++i) {
                v[i][k] = (FULL || k < nb) ? o[i] - s_lb[k] : absent_slot<NMAX, MODE>(k, nb);
                if (BOTH) dk[i][k] = od[i];
            }
        }
#pragma unroll
        for (int i = 0; i < PX; ++i) mb[i] = combine_all<NMAX, MODE>(v[i], FULL ? NMAX : nb, ksigma, max_iter);
#pragma unroll
        for (int k = 0; k < NMAX; ++k) {
            float od[PX];
#pragma unroll
            for (int i = 0; i < PX; ++i) od[i] = BOTH ? dk[i][k] : 0.f;
            if (!BOTH) load_px<PX>(frame_ptr(pd, FULL ? k : min(k, nd - 1), fsb), nv, od);
#pragma unroll
            for (int i = 0; i < PX; ++i) v[i][k] = (FULL || k < nd) ? (od[i] - s_ld[k]) - mb[i] : absent_slot<NMAX, MODE>(k, nd);
        }
#pragma unroll
        for (int i = 0; i < PX; ++i) md[i] = combine_all<NMAX, MODE>(v[i], FULL ? NMAX : nd, ksigma, max_iter);
        if (PX == 2) {
            *reinterpret_cast<float2*>(MB + p) = make_float2(mb[0], mb[PX - 1]);
            *reinterpret_cast<float2*>(MD + p) = make_float2(md[0], md[PX - 1]);
        } else {
            for (int i = 0; i < nv; ++i) { MB[p + i] = mb[i]; MD[p + i] = md[i]; }
        }
#pragma unroll
        for (int i = 0; i < PX; ++i)
            if (i >= nv) { mb[i] = 0.f; md[i] = 0.f; }
    }
    float tb = 0.f, td = 0.f;
#pragma unroll
    for (int i = 0; i < PX; ++i) { tb += mb[i]; td += md[i]; }
    // block partials of both planes; after the one barrier only warp 0 stays: it writes the partials and takes the ticket,
    // and in the LAST block to arrive it adds up all partials (fixed order) and turns them into 1/<G_k>.  (With the whole
    // block waiting for the fence + ticket round trip, "barrier" was the top stall reason of this kernel.)
    constexpr int MT = masters_threads<NMAX>();
    __shared__ float2 s_w2[MT / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    tb = warp_sum(tb);          // <= 64 values of one plane in float32: 1e-6 relative on a partial
    td = warp_sum(td);
    if (lane == 0) s_w2[warp] = make_float2(tb, td);
    __syncthreads();
    if (warp != 0) return;
    int last = 0;
    if (lane == 0) {
        double sb = 0.0, sd = 0.0;
        for (int i = 0; i < MT / 32; ++i) { sb += (double)s_w2[i].x; sd += (double)s_w2[i].y; }
        m.part_bd[2 * (size_t)blockIdx.x] = sb;
        m.part_bd[2 * (size_t)blockIdx.x + 1] = sd;
        __threadfence();
        last = atomicAdd(m.ticket, 1u) == gridDim.x - 1;
    }
    last = __shfl_sync(0xffffffffu, last, 0);
    if (!last) return;
    __threadfence();
    // <G_k> = <F_k> - L_k - <MB> - r <MD>: fixed-order sums of the block partials
    double a = 0.0, b = 0.0;
    for (int i = lane; i < (int)gridDim.x; i += 32) { a += __ldcg(m.part_bd + 2 * (size_t)i); b += __ldcg(m.part_bd + 2 * (size_t)i + 1); }
    a = warp_sum(a);
    b = warp_sum(b);
    const double np = (double)g.w * (double)g.h;
    const double mean_b = a / np, mean_d = b / np;
    for (int k = lane; k < nf; k += 32) {
        const double L = cnt > 0 ? (double)__ldcg(m.os + nb + nd + k) / (double)cnt : 0.0;
        const double gm = (double)__ldcg(m.img_f + k) / np - L - mean_b - r * mean_d;
        m.inv_gm[k] = (float)(1.0 / gm);
    }
}

// ---- flat; the last block turns the block sums into 1/<MF_raw> ---------------------------------
template <int NMAX, int MODE, int PX, bool FULL>
__global__ void __launch_bounds__(masters_threads<NMAX>()) k_masters_f(const uint16_t* __restrict__ flat, int nb, int nd, int nf, Geom g,
                                                   MastersWs m, float r, float ksigma, int max_iter,
                                                   const float* __restrict__ MB, const float* __restrict__ MD,
                                                   float* __restrict__ MF)
{
    __shared__ float s_lf[MRED_MAX_STACK + 1], s_ig[MRED_MAX_STACK + 1];
    for (int k = threadIdx.x; k < nf; k += blockDim.x) {
        s_lf[k] = m.lev[nb + nd + k];
        s_ig[k] = m.inv_gm[k];
    }
    __syncthreads();
    const size_t fs = (size_t)g.W * g.H;
    const unsigned int fsb = (unsigned int)(fs * 2);
    const int wg = (g.w + PX - 1) / PX;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    float mf[PX];
#pragma unroll
    for (int i = 0; i < PX; ++i) mf[i] = 0.f;
    if (gid < (long long)g.h * wg) {
        const int y = (int)((unsigned)gid / (unsigned)wg), x = (int)((unsigned)gid - (unsigned)y * (unsigned)wg) * PX;
        const int nv = min(PX, g.w - x);
        const size_t q = (size_t)(y + g.y0) * g.W + (x + g.x0);
        const size_t p = (size_t)y * g.w + x;
        float off[PX];
#pragma unroll
        for (int i = 0; i < PX; ++i) off[i] = i < nv ? fmaf(r, MD[p + i], MB[p + i]) : 0.f;
        float v[PX][NMAX];
        const uint16_t* pf = flat + q;
#pragma unroll
        for (int k = 0; k < NMAX; ++k) {
            float o[PX];
            load_px<PX>(frame_ptr(pf, FULL ? k : min(k, nf - 1), fsb), nv, o);     // see k_masters_bd
#pragma unroll
            for (int i = 0; i < PX; ++i) v[i][k] = (FULL || k < nf) ? ((o[i] - s_lf[k]) - off[i]) * s_ig[k] : absent_slot<NMAX, MODE>(k, nf);
        }
#pragma unroll
        for (int i = 0; i < PX; ++i) mf[i] = combine_all<NMAX, MODE>(v[i], FULL ? NMAX : nf, ksigma, max_iter);
        if (PX == 2) *reinterpret_cast<float2*>(MF + p) = make_float2(mf[0], mf[PX - 1]);
        else for (int i = 0; i < nv; ++i) MF[p + i] = mf[i];
#pragma unroll
        for (int i = 0; i < PX; ++i)
            if (i >= nv) mf[i] = 0.f;
    }
    float t = 0.f;
#pragma unroll
    for (int i = 0; i < PX; ++i) t += mf[i];
    constexpr int MT = masters_threads<NMAX>();
    __shared__ float s_w1[MT / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    t = warp_sum(t);
    if (lane == 0) s_w1[warp] = t;
    __syncthreads();
    if (warp != 0) return;                 // only warp 0 waits for the ticket (see k_masters_bd)
    int last = 0;
    if (lane == 0) {
        double sblk = 0.0;
        for (int i = 0; i < MT / 32; ++i) sblk += (double)s_w1[i];
        m.part_f[blockIdx.x] = sblk;
        __threadfence();
        last = atomicAdd(m.ticket + 1, 1u) == gridDim.x - 1;
    }
    last = __shfl_sync(0xffffffffu, last, 0);
    if (!last) return;
    __threadfence();
    double a = 0.0;
    for (int i = lane; i < (int)gridDim.x; i += 32) a += __ldcg(m.part_f + i);
    a = warp_sum(a);
    if (lane == 0) m.inv_mf[0] = (float)((double)g.w * (double)g.h / a);
}

__global__ void __launch_bounds__(256) k_mf_scale(float* __restrict__ MF, size_t np, const float* __restrict__ inv_mf, int vec)
{
    const float sc = inv_mf[0];
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec) {
        if (4 * i + 3 < np) {
            float4 v = reinterpret_cast<float4*>(MF)[i];
            v.x *= sc; v.y *= sc; v.z *= sc; v.w *= sc;
            reinterpret_cast<float4*>(MF)[i] = v;
        }
    } else {
        for (size_t p = 4 * i; p < np && p < 4 * i + 4; ++p) MF[p] *= sc;
    }
}

template <int NMAX, int PX, bool FULL>
static void launch_bd(int mode, dim3 grid, cudaStream_t st, const uint16_t* bias, int nb, const uint16_t* dark, int nd,
                      int nf, const Geom& g, const MastersWs& m, double r, float ks, int mi, float* MB, float* MD)
{
    if (mode == MRED_MEDIAN)
        k_masters_bd<NMAX, MRED_MEDIAN, PX, FULL><<<grid, masters_threads<NMAX>(), 0, st>>>(bias, nb, dark, nd, nf, g, m, r, ks, mi, MB, MD);
    else if (mode == MRED_MEAN)
        k_masters_bd<NMAX, MRED_MEAN, PX, FULL><<<grid, masters_threads<NMAX>(), 0, st>>>(bias, nb, dark, nd, nf, g, m, r, ks, mi, MB, MD);
    else
        k_masters_bd<NMAX, MRED_SIGCLIP, PX, FULL><<<grid, masters_threads<NMAX>(), 0, st>>>(bias, nb, dark, nd, nf, g, m, r, ks, mi, MB, MD);
}

template <int NMAX, int PX, bool FULL>
static void launch_f(int mode, dim3 grid, cudaStream_t st, const uint16_t* flat, int nb, int nd, int nf, const Geom& g,
                     const MastersWs& m, float r, float ks, int mi, const float* MB, const float* MD, float* MF)
{
    if (mode == MRED_MEDIAN)
        k_masters_f<NMAX, MRED_MEDIAN, PX, FULL><<<grid, masters_threads<NMAX>(), 0, st>>>(flat, nb, nd, nf, g, m, r, ks, mi, MB, MD, MF);
    else if (mode == MRED_MEAN)
        k_masters_f<NMAX, MRED_MEAN, PX, FULL><<<grid, masters_threads<NMAX>(), 0, st>>>(flat, nb, nd, nf, g, m, r, ks, mi, MB, MD, MF);
    else
        k_masters_f<NMAX, MRED_SIGCLIP, PX, FULL><<<grid, masters_threads<NMAX>(), 0, st>>>(flat, nb, nd, nf, g, m, r, ks, mi, MB, MD, MF);
}

// capacity buckets (the sorting network and every sweep are unrolled over the capacity, so a tight bucket
// is a direct saving); two pixels per thread up to 64 frames (since the dark column is no longer held beside the bias
// column: 48 frames 311 -> 232 us, 64 frames 406 -> 323 us), one above (register budget)
#define MRED_BUCKET(n, CALL)                     \
    do {                                         \
        if ((n) <= 3) { CALL(3, 2); }            \
        else if ((n) <= 4) { CALL(4, 2); }       \
        else if ((n) <= 5) { CALL(5, 2); }       \
        else if ((n) <= 6) { CALL(6, 2); }       \
        else if ((n) <= 8) { CALL(8, 2); }       \
        else if ((n) <= 10) { CALL(10, 2); }     \
        else if ((n) <= 12) { CALL(12, 2); }     \
        else if ((n) <= 16) { CALL(16, 2); }     \
        else if ((n) <= 20) { CALL(20, 2); }     \
        else if ((n) <= 24) { CALL(24, 2); }     \
        else if ((n) <= 32) { CALL(32, 2); }     \
        else if ((n) <= 48) { CALL(48, 2); }     \
        else if ((n) <= 64) { CALL(64, 2); }     \
        else if ((n) <= 96) { CALL(96, 1); }     \
        else if ((n) <= 128) { CALL(128, 1); }   \
        else if ((n) <= 192) { CALL(192, 1); }   \
        else { CALL(256, 1); }                   \
    } while (0)

int launch_build_masters(const Geom& g, const uint16_t* bias, int nb, const uint16_t* dark, int nd, float t_dark,
                         const uint16_t* flat, int nf, float t_flat, const mred_comb_opts& o, float* MB, float* MD,
                         float* MF, void* ws, cudaStream_t st)
{
    const MastersWs m = carve(ws, g, nb, nd, nf);
    MRED_CUDA_TRY(cudaMemsetAsync(m.os, 0, m.zero_bytes, st));
    // pairs of pixels by one 32-bit load need even W, x0 and w (frame bases are 16-byte aligned, frames W*H*2 B)
    const int pair_ok = (g.W % 2 == 0 && g.x0 % 2 == 0 && g.w % 2 == 0 && ((size_t)g.W * g.H) % 2 == 0) ? 1 : 0;
    const int nos = (g.H + 255) / 256, nimg = (g.h + 7) / 8;
    k_master_sums<<<dim3((unsigned)(nos * (nb + nd + nf) + nimg * nf)), 256, 0, st>>>(bias, nb, dark, nd, flat, nf, g, nos, nimg, m.os, m.img_f, m.ticket + 2, m.lev, pair_ok);
    MRED_LAUNCH_CHECK();
    const size_t np = (size_t)g.w * g.h;
    const int nbd = nb > nd ? nb : nd;
    const float r = t_flat / t_dark;
    const double rd = (double)t_flat / (double)t_dark;
#define CALL_BD(N, PX)                                                                                         \
    do {                                                                                                       \
        if (PX == 2 && pair_ok && nb == N && nd == N) launch_bd<N, PX, PX == 2>(o.mode, dim3((unsigned)((np / 2 + masters_threads<N>() - 1) / masters_threads<N>())), st, bias, nb, dark, nd, nf, g, m, rd, o.ksigma, o.max_iter, MB, MD); \
        else if (PX == 2 && pair_ok) launch_bd<N, PX, false>(o.mode, dim3((unsigned)((np / 2 + masters_threads<N>() - 1) / masters_threads<N>())), st, bias, nb, dark, nd, nf, g, m, rd, o.ksigma, o.max_iter, MB, MD); \
        else launch_bd<N, 1, false>(o.mode, dim3((unsigned)((np + masters_threads<N>() - 1) / masters_threads<N>())), st, bias, nb, dark, nd, nf, g, m, rd, o.ksigma, o.max_iter, MB, MD); \
    } while (0)
    MRED_BUCKET(nbd, CALL_BD);
#undef CALL_BD
    MRED_LAUNCH_CHECK();
#define CALL_F(N, PX)                                                                                          \
    do {                                                                                                       \
        if (PX == 2 && pair_ok && nf == N) launch_f<N, PX, PX == 2>(o.mode, dim3((unsigned)((np / 2 + masters_threads<N>() - 1) / masters_threads<N>())), st, flat, nb, nd, nf, g, m, r, o.ksigma, o.max_iter, MB, MD, MF); \
        else if (PX == 2 && pair_ok) launch_f<N, PX, false>(o.mode, dim3((unsigned)((np / 2 + masters_threads<N>() - 1) / masters_threads<N>())), st, flat, nb, nd, nf, g, m, r, o.ksigma, o.max_iter, MB, MD, MF); \
        else launch_f<N, 1, false>(o.mode, dim3((unsigned)((np + masters_threads<N>() - 1) / masters_threads<N>())), st, flat, nb, nd, nf, g, m, r, o.ksigma, o.max_iter, MB, MD, MF); \
    } while (0)
    MRED_BUCKET(nf, CALL_F);
#undef CALL_F
    MRED_LAUNCH_CHECK();
    const int vec = (np % 4 == 0) ? 1 : 0;
    k_mf_scale<<<dim3((unsigned)((np + 1023) / 1024)), 256, 0, st>>>(MF, np, m.inv_mf, vec);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
