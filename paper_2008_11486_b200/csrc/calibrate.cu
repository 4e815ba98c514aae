// calibrate.cu -- overscan level (O1) and the fused trim + level + bias/dark + flat pass (O3).
// PAPER.md L63 / L99: overscan cutout, bias subtraction, dark subtraction, flat fielding.
//
// HBM roofline: per science pixel 2 B (uint16) in + 4 B (float32) out; the three master planes
// (12 B/px) are loaded ONCE per thread and kept in registers while the thread walks FC frames, so
// they cost 12/FC B/px of L2 traffic instead of 12 (which would make the pass L2-bound).
#include "common.cuh"

namespace mred {

// ---------------------------------------------------------------------------------------------
// Exact integer sums: overscan columns of every frame, optionally the image rectangle as well
// (used for <F_k> of the flats).  Integer atomics -> order-independent, bit-exact.
// grid (row_chunks, n), block 256; each warp takes rows r0 + warp, r0 + warp + 8, ...
// ---------------------------------------------------------------------------------------------
// grid (ceil(H/256), n), block 256: one thread per row of the overscan strip
__global__ void __launch_bounds__(256) k_frame_sums(const uint16_t* __restrict__ raw, Geom g, int n,
                                                    unsigned long long* __restrict__ os_sum)
{
    const int k = blockIdx.y;
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long s = 0;
    if (r < g.H) s = overscan_row_sum(raw + (size_t)k * g.W * g.H, g.W, g.os_x0, g.os_x1, r);
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0 && s) atomicAdd(os_sum + k, s);
}

int launch_frame_sums(const uint16_t* raw, const Geom& g, int n, unsigned long long* os_sum,
                      unsigned long long* /*img_sum*/, cudaStream_t st)
{
    MRED_CUDA_TRY(cudaMemsetAsync(os_sum, 0, sizeof(unsigned long long) * n, st));
    if (g.os_x1 <= g.os_x0) return MRED_OK;
    dim3 grid((g.H + 255) / 256, n);
    k_frame_sums<<<grid, 256, 0, st>>>(raw, g, n, os_sum);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
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
                                                   float* __restrict__ out, const unsigned long long* __restrict__ os_sum,
                                                   double* __restrict__ level_out, int vec_ok)
{
    __shared__ float s_level[CAL_MAXFC];
    const int k0 = blockIdx.y * fc, k1 = min(k0 + fc, n);
    if (threadIdx.x < k1 - k0) {
        const long long cnt = (long long)(g.os_x1 - g.os_x0) * g.H;
        const double L = cnt > 0 ? (double)os_sum[k0 + threadIdx.x] / (double)cnt : 0.0;
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
        inv[i] = (f > 0.f && f <= 3.402823466e+38f) ? 1.0f / f : 0.f;
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

int launch_calibrate(const uint16_t* raw, const Geom& g, int n, float dark_scale, const float* MB, const float* MD,
                     const float* MF, float* out, double* level_out, const unsigned long long* os_sum,
                     double* /*prof_ws*/, cudaStream_t st)
{
    const int w4 = (g.w + 3) / 4;
    const long long groups = (long long)g.h * w4;
    // frames per chunk: enough chunks to fill the machine, at most CAL_MAXFC frames per thread
    int fc = n < 8 ? n : 8;
    if (fc > CAL_MAXFC) fc = CAL_MAXFC;
    dim3 grid((unsigned)((groups + 255) / 256), (unsigned)((n + fc - 1) / fc));
    const int vec_ok = (g.w % 4 == 0) ? 1 : 0;
    k_calibrate<<<grid, 256, 0, st>>>(raw, g, n, fc, dark_scale, MB, MD, MF, out, os_sum, level_out, vec_ok);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
