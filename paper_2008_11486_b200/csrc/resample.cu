// resample.cu -- sub-pixel shift by bicubic-spline interpolation (O5; PAPER.md L63,
// L107, L164, L266).  The per-CTA program is in resample_block.cuh; this file is the kernel shell
// (shared memory, barriers, per-frame parameters) and the launcher.
#include "common.cuh"
#include "resample_block.cuh"

namespace mred {

using namespace rs;

template <int TW>
__global__ void __launch_bounds__(TW) k_resample(const float* __restrict__ in, int n, int w, int h,
                                                 const __grid_constant__ HostShifts hs,
                                                 const double* __restrict__ dshift, float fill,
                                                 float* __restrict__ out, int4* __restrict__ fp_dev, int BH)
{
    typedef BlockCfg<TW> Cfg;
    __shared__ float s_tile[Cfg::TILE_FLOATS];
    __shared__ float s_T[Cfg::T_FLOATS];
    const int k = blockIdx.z;
    // (sx, sy): by value from the host call, or minus the estimated content displacement (device)
    const double sx = dshift ? -dshift[2 * k] : hs.s[k][0];
    const double sy = dshift ? -dshift[2 * k + 1] : hs.s[k][1];
    const size_t np = (size_t)w * h;
    BlockCtx c;
    block_setup<TW>(c, in + (size_t)k * np, out + (size_t)k * np, w, h, sx, sy, blockIdx.x, blockIdx.y, BH, fill,
                    s_tile, s_T);
    if (fp_dev && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0)
        fp_dev[k] = make_int4(c.ax.lo, c.ax.hi, c.ay.lo, c.ay.hi);
    YState st;
    y_state_init(st);
    for (int j = 0; j < c.nblocks; ++j) {
        const int rb = c.r_begin + j * R;
        load_phase<TW>(c, threadIdx.x, TW, rb);
        __syncthreads();
        x_phase<TW>(c, threadIdx.x, TW);
        __syncthreads();
        y_phase<TW>(c, st, threadIdx.x, rb, j == 0);
        __syncthreads();
    }
}

int launch_resample(const float* in, int n, int w, int h, const double* sx_host, const double* sy_host,
                    const double* dshift_dev, float fill, float* out, int32_t* fp_dev, cudaStream_t st)
{
    HostShifts hs;
    if (!dshift_dev)
        for (int k = 0; k < n; ++k) { hs.s[k][0] = sx_host[k]; hs.s[k][1] = sy_host[k]; }
    constexpr int TW = 128;
    const int strips = (w + TW - 1) / TW;
    // band height: full columns when there are enough (frame, strip) pairs to fill the machine,
    // else split in y (each band pays one warm-up block of R rows)
    int BH = h;
    const long long ctas_full = (long long)strips * n;
    if (ctas_full < 148 * 6) {
        long long bands = (148 * 6 + ctas_full - 1) / ctas_full;
        BH = (int)((h + bands - 1) / bands);
        BH = ((BH + R - 1) / R) * R;
        if (BH < 4 * R) BH = 4 * R;
        if (BH > h) BH = h;
    }
    const int bands = (h + BH - 1) / BH;
    dim3 grid(strips, bands, n);
    k_resample<TW><<<grid, TW, 0, st>>>(in, n, w, h, hs, dshift_dev, fill, out, reinterpret_cast<int4*>(fp_dev), BH);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
