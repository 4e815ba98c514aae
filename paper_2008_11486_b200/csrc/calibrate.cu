// calibrate.cu -- overscan level (O1) and the fused trim + level + bias/dark + flat pass (O3).
// PAPER.md L63 / L99: overscan cutout, bias subtraction, dark subtraction, flat fielding.
//
// HBM roofline: per science pixel 2 B (uint16) in + 4 B (float32) out; the three master planes
// (12 B/px) are loaded ONCE per thread and kept in registers while the thread walks FC frames, so
// they cost 12/FC B/px of L2 traffic instead of 12 (which would make the pass L2-bound).
#include "common.cuh"

namespace mred {

// ---------------------------------------------------------------------------------------------
// Exact integer sums of the overscan columns of every frame, as per-block partials: block (c, k) writes the sum
// of rows [256c, 256c + 256) of frame k to os_part[k * nos + c].  No atomics, so nothing has to be zeroed first;
// the consumers add the nos = ceil(H/256) partials (integers: exact in any order).
// Side job for the chained path: the blocks also clear `zero` (the accumulators of the kernels that follow on the
// same stream), which saves the memset nodes between the stages.
// grid (nos * n) (1-D, so the frame count is not bound by the 65535 of gridDim.y), block 256: one thread per row
// of the overscan strip
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_frame_sums(const uint16_t* __restrict__ raw, Geom g, int n, int nos,
                                                    unsigned long long* __restrict__ os_part,
                                                    uint4* __restrict__ zero, size_t zero_n16)
{
    __shared__ unsigned long long s_w[8];
    const int k = blockIdx.x / nos, c = blockIdx.x - k * nos;
    const int r = c * blockDim.x + threadIdx.x;
    if (zero) {
        const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        const size_t nth = (size_t)gridDim.x * blockDim.x;
        for (size_t i = tid; i < zero_n16; i += nth) zero[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    unsigned long long s = 0;
    if (r < g.H && g.os_x1 > g.os_x0) s = overscan_row_sum(raw + (size_t)k * g.W * g.H, g.W, g.os_x0, g.os_x1, r);
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int i = 0; i < 8; ++i) t += s_w[i];
        os_part[blockIdx.x] = t;          // = os_part[k * nos + c]
    }
}

int frame_sums_parts(const Geom& g) { return (g.H + 255) / 256; }

int launch_frame_sums(const uint16_t* raw, const Geom& g, int n, unsigned long long* os_part, void* zero,
                      size_t zero_bytes, cudaStream_t st)
{
    const int nos = frame_sums_parts(g);
    k_frame_sums<<<dim3((unsigned)(nos * n)), 256, 0, st>>>(raw, g, n, nos, os_part, static_cast<uint4*>(zero), zero ? zero_bytes / 16 : 0);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

// overscan level of frame k from the block partials (O1: exact integer sum, one float64 division)
__device__ __forceinline__ double level_of(const unsigned long long* __restrict__ os_part, int nos, int k, const Geom& g)
{
    const long long cnt = (long long)(g.os_x1 - g.os_x0) * g.H;
    unsigned long long t = 0;
    for (int i = 0; i < nos; ++i) t += os_part[(size_t)k * nos + i];
    return cnt > 0 ? (double)t / (double)cnt : 0.0;
}

// ---------------------------------------------------------------------------------------------
// calibrate: thread = 4 consecutive image pixels of one row, for the FC frames of its chunk.
// grid.x covers h * ceil(w/4) pixel groups, grid.y the frame chunks.
// ---------------------------------------------------------------------------------------------
constexpr int CAL_MAXFC = 16;   // frames per chunk (masters re-read once per chunk)

__device__ __forceinline__ void load4_u16(const uint16_t* p, int nv, float v[4])
{
    if (nv == 4 && ((reinterpret_cast<uintptr_t>(p) & 3u) == 0)) {
        const unsigned int a = __ldcs(reinterpret_cast<const unsigned int*>(p));
        const unsigned int b = __ldcs(reinterpret_cast<const unsigned int*>(p) + 1);
        v[0] = (float)(a & 0xffffu); v[1] = (float)(a >> 16);
        v[2] = (float)(b & 0xffffu); v[3] = (float)(b >> 16);
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = i < nv ? (float)__ldcs(p + i) : 0.f;
    }
}

__global__ void __launch_bounds__(256) k_calibrate(const uint16_t* __restrict__ raw, Geom g, int n, int fc,
                                                   float dark_scale, const float* __restrict__ MB,
                                                   const float* __restrict__ MD, const float* __restrict__ MF,
                                                   float* __restrict__ out, const unsigned long long* __restrict__ os_part,
                                                   int nos, double* __restrict__ level_out, int vec_ok)
{
    __shared__ float s_level[CAL_MAXFC];
    const int k0 = blockIdx.y * fc, k1 = min(k0 + fc, n);
    if (threadIdx.x < k1 - k0) {
        const double L = level_of(os_part, nos, k0 + threadIdx.x, g);
        s_level[threadIdx.x] = (float)L;
        if (level_out && blockIdx.x == 0) level_out[k0 + threadIdx.x] = L;
    }
    __syncthreads();
    const int w4 = (g.w + 3) >> 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)g.h * w4) return;
    const int y = (int)((unsigned)gid / (unsigned)w4), x = (int)((unsigned)gid - (unsigned)y * (unsigned)w4) * 4;   // w*h < 2^31 (api.cu)
    const int nv = min(4, g.w - x);
    const size_t p = (size_t)y * g.w + x;
    float mb[4], ms[4], inv[4];
    if (vec_ok) {
        const float4 a = __ldg(reinterpret_cast<const float4*>(MB + p));
        const float4 b = __ldg(reinterpret_cast<const float4*>(MD + p));
        const float4 c = __ldg(reinterpret_cast<const float4*>(MF + p));
        mb[0] = a.x; mb[1] = a.y; mb[2] = a.z; mb[3] = a.w;
        ms[0] = b.x; ms[1] = b.y; ms[2] = b.z; ms[3] = b.w;
        inv[0] = c.x; inv[1] = c.y; inv[2] = c.z; inv[3] = c.w;
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            mb[i] = i < nv ? MB[p + i] : 0.f; ms[i] = i < nv ? MD[p + i] : 0.f; inv[i] = i < nv ? MF[p + i] : 1.f;
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        // offset = MB + s*MD (one rounding more than the oracle's left-to-right sum; << tolerance)
        mb[i] = fmaf(dark_scale, ms[i], mb[i]);
        // MF <= 0 or non-finite -> 0 (reading Q7): a zero reciprocal zeroes the product
        const float f = inv[i];
        inv[i] = (f > 0.f && f <= 3.402823466e+38f) ? __fdividef(1.0f, f) : 0.f;      // MUFU.RCP, 1 ulp
    }
    const size_t fs = (size_t)g.W * g.H, np = (size_t)g.w * g.h;
    const uint16_t* src = raw + (size_t)k0 * fs + (size_t)(y + g.y0) * g.W + g.x0 + x;
    float* dst = out + (size_t)k0 * np + p;
    int k = k0;
    for (; k + 4 <= k1; k += 4) {       // 4 frames in flight per thread
        float v[4][4];
#pragma unroll
        for (int j = 0; j < 4; ++j) load4_u16(src + (size_t)j * fs, nv, v[j]);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float L = s_level[k - k0 + j];
            float r[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) r[i] = ((v[j][i] - L) - mb[i]) * inv[i];
            if (vec_ok) *reinterpret_cast<float4*>(dst + (size_t)j * np) = make_float4(r[0], r[1], r[2], r[3]);
            else for (int i = 0; i < nv; ++i) dst[(size_t)j * np + i] = r[i];
        }
        src += 4 * fs; dst += 4 * np;
    }
    for (; k < k1; ++k) {
        float v[4];
        load4_u16(src, nv, v);
        const float L = s_level[k - k0];
        float r[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) r[i] = ((v[i] - L) - mb[i]) * inv[i];
        if (vec_ok) *reinterpret_cast<float4*>(dst) = make_float4(r[0], r[1], r[2], r[3]);
        else for (int i = 0; i < nv; ++i) dst[i] = r[i];
        src += fs; dst += np;
    }
}

// ---------------------------------------------------------------------------------------------
// calibrate + marginal profiles in one pass (chained path; an optional bad-pixel mask keeps pixels out of the sums): the calibrated pixels are summed
// into the row / column profiles of O4 while they are still in registers, so estimate_shifts never re-reads the
// calibrated stack (N*4wh bytes of HBM traffic and a kernel less; SURVEY 8(d) "0 if fused into calibrate").
// Block = 256 threads = tile of 128 columns x 8 rows (warp = one 128-pixel row segment, lane = 4 pixels) of 4
// frames; all loads of a thread are issued up front.  Row segment sums by warp shuffle; column sums over the 8
// rows through shared memory (one barrier, then thread = (frame, column)); both are added to the global int64
// fixed-point accumulators (value * 2^14) with integer atomics: exact and order-independent.
// Tiles of 16 rows (512 threads, half as many column atomics) measured 1-2 % slower (config 3 90.5 against 89.9 us,
// config 5 2.08 against 2.04 ms: twice as many warps wait at the barrier for the slowest one's loads), tiles of 4 rows
// slower again (92.3 us).
// grid (ceil(n/4), ceil(w/128), ceil(h/8)).
// ---------------------------------------------------------------------------------------------
constexpr int CP_ROWS = 8, CP_COLS = 128, CP_FB = 4;      // tile and frames per block
constexpr int CP_THREADS = 32 * CP_ROWS;                  // one warp per row of the tile

// NKF > 0 (fast body): the tile lies inside the image, holds exactly NKF frames, rows are 16-byte aligned in the
// output and 4-byte aligned in the raw frames: no per-thread bounds, tails or alignment tests (they were 40 % of the
// instructions issued).  NKF = 0: the general body.
template <int NKF, bool MASK>
__device__ __forceinline__ void calibrate_prof_body(const uint16_t* __restrict__ raw, const Geom& g, int n,
                                                    float dark_scale, const float* __restrict__ MB,
                                                    const float* __restrict__ MD, const float* __restrict__ MF,
                                                    float* __restrict__ out, const unsigned long long* __restrict__ os_part,
                                                    int nos, const uint8_t* __restrict__ bad, long long* __restrict__ colsum,
                                                    long long* __restrict__ rowsum, int vec_ok, float (&s_level)[CP_FB],
                                                    float (&s_col)[CP_FB][CP_ROWS][CP_COLS])
{
    constexpr bool FAST = NKF > 0;
    // blockIdx.x = frame chunk (fastest): the blocks that share a tile of the master planes run together, so the
    // masters come out of HBM once and out of L2 for the other chunks (they exceed L2 at 4096^2)
    const int k0 = blockIdx.x * CP_FB, nk = FAST ? NKF : min(CP_FB, n - k0);
    // (the last warp takes the levels: its float64 division then delays nobody else's loads)
    if (threadIdx.x >= CP_THREADS - CP_FB && (int)threadIdx.x - (CP_THREADS - CP_FB) < nk)
        s_level[threadIdx.x - (CP_THREADS - CP_FB)] = (float)level_of(os_part, nos, k0 + (int)threadIdx.x - (CP_THREADS - CP_FB), g);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int x = blockIdx.y * CP_COLS + 4 * lane, y = blockIdx.z * CP_ROWS + warp;
    const bool live = FAST || (x < g.w && y < g.h);
    const int nv = FAST ? 4 : (live ? min(4, g.w - x) : 0);
    const bool vec = FAST || (vec_ok && nv == 4);
    const size_t p = live ? (size_t)y * g.w + x : 0;
    const size_t fs = (size_t)g.W * g.H, np = (size_t)g.w * g.h;
    // every global load of the thread is issued before the first barrier
    float v[CP_FB][4];
    {
        const uint16_t* src = raw + (size_t)k0 * fs + (live ? (size_t)(y + g.y0) * g.W + g.x0 + x : 0);
#pragma unroll
        for (int j = 0; j < CP_FB; ++j) {
#pragma unroll
            for (int i = 0; i < 4; ++i) v[j][i] = 0.f;
            if (FAST && j < NKF) {
                const unsigned int* q = reinterpret_cast<const unsigned int*>(src + (size_t)j * fs);
                const unsigned int a = __ldcs(q), b = __ldcs(q + 1);
                v[j][0] = (float)(a & 0xffffu); v[j][1] = (float)(a >> 16);
                v[j][2] = (float)(b & 0xffffu); v[j][3] = (float)(b >> 16);
            } else if (!FAST && j < nk && live) {
                load4_u16(src + (size_t)j * fs, nv, v[j]);
            }
        }
    }
    float mb[4], ms[4], inv[4];
    if (vec) {
        const float4 a = __ldg(reinterpret_cast<const float4*>(MB + p));
        const float4 b = __ldg(reinterpret_cast<const float4*>(MD + p));
        const float4 c = __ldg(reinterpret_cast<const float4*>(MF + p));
        mb[0] = a.x; mb[1] = a.y; mb[2] = a.z; mb[3] = a.w;
        ms[0] = b.x; ms[1] = b.y; ms[2] = b.z; ms[3] = b.w;
        inv[0] = c.x; inv[1] = c.y; inv[2] = c.z; inv[3] = c.w;
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            mb[i] = i < nv ? MB[p + i] : 0.f; ms[i] = i < nv ? MD[p + i] : 0.f; inv[i] = i < nv ? MF[p + i] : 0.f;
        }
    }
    unsigned okm = 0xfu;          // bit i: pixel i counts in the profiles (bad-pixel mask, O4)
    if (MASK) {
        if (vec) {
            const uchar4 b = __ldg(reinterpret_cast<const uchar4*>(bad + p));
            okm = (b.x ? 0u : 1u) | (b.y ? 0u : 2u) | (b.z ? 0u : 4u) | (b.w ? 0u : 8u);
        } else {
            okm = 0u;
            for (int i = 0; i < nv; ++i) okm |= __ldg(bad + p + i) ? 0u : (1u << i);
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        mb[i] = fmaf(dark_scale, ms[i], mb[i]);
        const float f = inv[i];
        // MUFU.RCP (1 ulp) instead of the IEEE division sequence, which was 11 % of the instructions and 22 % of the
        // stall samples of this kernel; the product differs from the quotient by < 2.5e-7 relative
        inv[i] = (f > 0.f && f <= 3.402823466e+38f) ? __fdividef(1.0f, f) : 0.f;     // dead lanes: 0, so they add nothing
    }
    float* dst = out + (size_t)k0 * np + p;
    float rsum[CP_FB];
#pragma unroll
    for (int j = 0; j < CP_FB; ++j) rsum[j] = 0.f;
#pragma unroll
    for (int j = 0; j < CP_FB; ++j) {
        if (j >= nk) break;                     // block-uniform
        const float L = s_level[j];
        float r[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) r[i] = ((v[j][i] - L) - mb[i]) * inv[i];
        if (vec) __stcg(reinterpret_cast<float4*>(dst + (size_t)j * np), make_float4(r[0], r[1], r[2], r[3]));
        else for (int i = 0; i < nv; ++i) dst[(size_t)j * np + i] = r[i];
        if (MASK && okm != 0xfu) {  // masked pixels are written like any other but stay out of the profiles
#pragma unroll
            for (int i = 0; i < 4; ++i) r[i] = ((okm >> i) & 1u) ? r[i] : 0.f;
        }
        *reinterpret_cast<float4*>(&s_col[j][warp][4 * lane]) = make_float4(r[0], r[1], r[2], r[3]);
        rsum[j] = (r[0] + r[1]) + (r[2] + r[3]);
    }
    {
        // row-segment sums of the 4 frames in ONE butterfly: the first two steps halve the number of frames a lane carries
        // (it keeps two, then one, and hands the others to its partner), the last three are a plain 8-lane sum: 6 shuffles
        // instead of 20, the same pairing order as four separate warp sums (so the same bits), and lanes 0, 8, 16, 24 end up
        // with the totals of frames 0, 1, 2, 3: one atomic instruction for all four
        static_assert(CP_FB == 4, "the transposing reduction is written for 4 frames per block");
        const bool h16 = lane & 16, h8 = lane & 8;
        float ka = h16 ? rsum[2] : rsum[0], kb = h16 ? rsum[3] : rsum[1];
        ka += __shfl_xor_sync(0xffffffffu, h16 ? rsum[0] : rsum[2], 16);
        kb += __shfl_xor_sync(0xffffffffu, h16 ? rsum[1] : rsum[3], 16);
        float kk = h8 ? kb : ka;
        kk += __shfl_xor_sync(0xffffffffu, h8 ? ka : kb, 8);
        kk += __shfl_xor_sync(0xffffffffu, kk, 4);
        kk += __shfl_xor_sync(0xffffffffu, kk, 2);
        kk += __shfl_xor_sync(0xffffffffu, kk, 1);
        const int jf = (h16 ? 2 : 0) + (h8 ? 1 : 0);
        if ((lane & 7) == 0 && jf < nk && (FAST || y < g.h))
            atomicAdd(reinterpret_cast<unsigned long long*>(rowsum) + (size_t)(k0 + jf) * g.h + y, (unsigned long long)__float2ll_rn(kk * PROF_FIX));
    }
    __syncthreads();
    // thread = (frame, column): the tile's rows in a fixed order
    for (int jc = threadIdx.x; jc < CP_FB * CP_COLS; jc += CP_THREADS) {
        const int j = jc >> 7, c = jc & (CP_COLS - 1);
        const int cx = blockIdx.y * CP_COLS + c;
        if (FAST ? (j < NKF) : (j < nk && cx < g.w)) {
            float t = 0.f;
#pragma unroll
            for (int rr = 0; rr < CP_ROWS; ++rr) t += s_col[j][rr][c];
            atomicAdd(reinterpret_cast<unsigned long long*>(colsum) + (size_t)(k0 + j) * g.w + cx, (unsigned long long)__float2ll_rn(t * PROF_FIX));
        }
    }
}

__global__ void __launch_bounds__(CP_THREADS, 1536 / CP_THREADS) k_calibrate_prof(const uint16_t* __restrict__ raw, Geom g, int n,
                                                           float dark_scale, const float* __restrict__ MB,
                                                           const float* __restrict__ MD, const float* __restrict__ MF,
                                                           float* __restrict__ out, const unsigned long long* __restrict__ os_part,
                                                           int nos, const uint8_t* __restrict__ bad, long long* __restrict__ colsum,
                                                           long long* __restrict__ rowsum, int vec_ok, int pair_ok)
{
    __shared__ float s_level[CP_FB];
    __shared__ __align__(16) float s_col[CP_FB][CP_ROWS][CP_COLS];
    const bool fast = vec_ok && pair_ok && (int)(blockIdx.y + 1) * CP_COLS <= g.w && (int)(blockIdx.z + 1) * CP_ROWS <= g.h;
    const int nkf = fast ? min(CP_FB, n - (int)blockIdx.x * CP_FB) : 0;      // block-uniform
#define MRED_CP_BODY(N)                                                                                                                   \
    do {                                                                                                                                  \
        if (bad) calibrate_prof_body<N, true>(raw, g, n, dark_scale, MB, MD, MF, out, os_part, nos, bad, colsum, rowsum, vec_ok, s_level, s_col);  \
        else calibrate_prof_body<N, false>(raw, g, n, dark_scale, MB, MD, MF, out, os_part, nos, bad, colsum, rowsum, vec_ok, s_level, s_col);   \
    } while (0)
    switch (nkf) {
        case 4: MRED_CP_BODY(4); break;
        case 3: MRED_CP_BODY(3); break;
        case 2: MRED_CP_BODY(2); break;
        case 1: MRED_CP_BODY(1); break;
        default: MRED_CP_BODY(0); break;
    }
#undef MRED_CP_BODY
}

// frames per chunk: enough chunks to fill the machine, at most 8 frames per thread, chunks of equal size
static int chunk_frames(int n)
{
    const int nch = (n + 7) / 8;
    return (n + nch - 1) / nch;
}

int launch_calibrate_prof(const uint16_t* raw, const Geom& g, int n, float dark_scale, const float* MB, const float* MD,
                          const float* MF, float* out, const unsigned long long* os_part, const uint8_t* bad,
                          long long* colsum, long long* rowsum, cudaStream_t st)
{
    const int tx = (g.w + CP_COLS - 1) / CP_COLS, ty = (g.h + CP_ROWS - 1) / CP_ROWS;
    if (tx > 65535 || ty > 65535) return MRED_EINVAL;
    dim3 grid((unsigned)((n + CP_FB - 1) / CP_FB), (unsigned)tx, (unsigned)ty);
    const int vec_ok = (g.w % 4 == 0) ? 1 : 0;
    const int pair_ok = (g.W % 2 == 0 && g.x0 % 2 == 0) ? 1 : 0;     // raw rows of the image rectangle start 4-byte aligned
    k_calibrate_prof<<<grid, CP_THREADS, 0, st>>>(raw, g, n, dark_scale, MB, MD, MF, out, os_part, frame_sums_parts(g), bad, colsum, rowsum, vec_ok, pair_ok);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

int launch_calibrate(const uint16_t* raw, const Geom& g, int n, float dark_scale, const float* MB, const float* MD,
                     const float* MF, float* out, double* level_out, const unsigned long long* os_part, cudaStream_t st)
{
    const int w4 = (g.w + 3) / 4;
    const long long groups = (long long)g.h * w4;
    const int fc = chunk_frames(n);
    if ((n + fc - 1) / fc > 65535) return MRED_EINVAL;          // gridDim.y; n <= 524 280 (include/mred.h)
    dim3 grid((unsigned)((groups + 255) / 256), (unsigned)((n + fc - 1) / fc));
    const int vec_ok = (g.w % 4 == 0) ? 1 : 0;
    k_calibrate<<<grid, 256, 0, st>>>(raw, g, n, fc, dark_scale, MB, MD, MF, out, os_part, frame_sums_parts(g), level_out, vec_ok);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
