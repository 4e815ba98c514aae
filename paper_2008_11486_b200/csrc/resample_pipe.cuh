// resample_pipe.cuh -- k_resample_pipe: the CTA-tiled, TMA-staged spline-shift kernel as a warp-specialised pipeline.
// Mathematics: resample.cu; segments and the per-row / per-column code (rt::make_seg, rs::x_pass, rt::causal, rt::sweep):
// resample_tile.cuh.  This file says who runs what, and when.
//
// Round 2's first tiled kernel alternated phases inside a CTA: all 8 warps ran the x pass of a chunk, a block barrier, 6.5
// warps ran the y pass, a block barrier.  ncu (profiles/r2_kernels.md): a third of the resident warps sat at one of the two
// barriers at any time and the y phase left 1.5 of 8 warps idle.  Here a pipeline of 16 warps is three roles that run
// CONCURRENTLY on different chunks and meet only through mbarriers:
//   producer (1 warp, one lane)  TMA boxes into NS = 3 stages; waits for a stage to be read (tempty) before reusing it
//   x warps  (8)                 wait for the box (tfull) and for a free ring slot (rempty); x pass of their two rows out
//                                of the stage into the ring slot; release the stage (tempty), publish the slot (rfull)
//   y warps  (7; 208 columns)    wait for the slot (rfull); causal recursion in place, sweep of the chunk before with the
//                                4 y taps and the stores; release the slot of the chunk before (rempty)
// With NR = 4 ring slots the x warps run up to two chunks ahead of the y warps, so neither role waits for the other's
// slowest warp.  Every arrival is one lane per warp after __syncwarp(); every wait is a warp-wide try_wait with a
// suspend-time hint (a plain polling loop took 40 % of the issue slots).
// A CTA is one pipeline of 512 threads, two per SM (NPIPE = 1).  Measured against it: NPIPE = 2, two pipelines in one CTA of
// 1024 threads with their warps interleaved (pipeline = warp & 1).  As two CTAs the pipeline launched second on an SM runs
// 25 % slower than the first (the warp scheduler favours the older CTA) and finishes alone; interleaved in one CTA both
// finish together, which is worth 1 % when the kernel has the GPU to itself (config 3: 136.7 against 138.1 us, config 5
// 2.93 against 2.98 ms).  But a CTA that needs a whole SM's registers can only start on an SM that is completely free: in
// the 6-stream step of bench.py, where other groups' kernels hold parts of every SM, the 512-thread CTAs find room
// earlier and their neighbours fill the issue slots this latency-bound kernel leaves: 1.89 -> 1.84 ms per step (+ 2.7 %
// frames/s).  The step is what the library is for, so NPIPE = 1 it is.
// The two configured detector widths (1024, 4096) get an instantiation with the output pitch compiled in: the 16 stores
// of a sweep then take immediate offsets from one base register instead of a pointer chain whose every update waited for
// the store before it to have read its address (config 3: 144 -> 138 us).
// Shared memory per pipeline: 3 x 16 KB stages + 4 x 13 KB ring = 100 KB; registers <= 64: two pipelines = 32 warps per SM.
#pragma once
#include "resample_tile.cuh"

namespace mred {
namespace rp {

using namespace rt;
using tma::mbar_arrive;
using tma::mbar_wait_parked;

constexpr int XW = CH / 2;                   // x warps: two rows of the chunk each
constexpr int YW = (TW + 31) / 32;           // y warps: one column per thread (the last one is half used)
constexpr int NTHR_P = (XW + YW + 1) * 32;   // + the producer warp: 512 threads
constexpr int NS = 3;                        // TMA stages
constexpr int NR = 4;                        // ring slots
constexpr int NPIPE = 1;                     // pipelines per CTA (2: warps interleaved, pipeline = warp & 1; see above)
constexpr size_t SMEM_1 = (size_t)NS * STAGE_FLOATS * 4 + (size_t)NR * T_FLOATS * 4 + 128;   // one pipeline: stages, ring, barriers
constexpr size_t SMEM_P = SMEM_1 * NPIPE;

// running (index, phase parity) of a circular set of N mbarriers
template <int N> struct Ring {
    int i = 0;
    unsigned ph = 0;
    __device__ __forceinline__ void next() { if (++i == N) { i = 0; ph ^= 1u; } }
};

}  // namespace rp

template <int PITCH>
__global__ void __launch_bounds__(rp::NTHR_P * rp::NPIPE, 2 / rp::NPIPE)
k_resample_pipe(const __grid_constant__ CUtensorMap tmap, int n, int w, int h, int ns, long long units, long long per_cta,
                const __grid_constant__ HostShifts hs, const double* __restrict__ dshift, float fill,
                float* __restrict__ out, int4* __restrict__ fp_dev)
{
    using namespace rp;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int pipe = NPIPE == 2 ? (int)((threadIdx.x >> 5) & 1) : 0;
    float* stage = reinterpret_cast<float*>(smem_raw + pipe * SMEM_1);   // [NS][CH][BOXW]   TMA destinations
    float* tring = stage + NS * STAGE_FLOATS;                            // [NR][CH][TW]     x-shifted rows / g
    uint64_t* tfull = reinterpret_cast<uint64_t*>(tring + NR * T_FLOATS);// [NS] box landed
    uint64_t* tempty = tfull + NS;                                       // [NS] box read by all x warps
    uint64_t* rfull = tempty + NS;                                       // [NR] slot written by all x warps
    uint64_t* rempty = rfull + NR;                                       // [NR] slot no longer needed by the y warps
    const int tid = threadIdx.x, lane = tid & 31, warp = (tid >> 5) / NPIPE;      // warp: index inside the pipeline

    for (int k = blockIdx.x * NTHR_P * NPIPE + tid; k < n && fp_dev; k += gridDim.x * NTHR_P * NPIPE) {
        const double sx = dshift ? -dshift[2 * k] : hs.s[k][0];
        const double sy = dshift ? -dshift[2 * k + 1] : hs.s[k][1];
        const Axis ax = make_axis(w, sx), ay = make_axis(h, sy);
        fp_dev[k] = make_int4(ax.lo, ax.hi, ay.lo, ay.hi);
    }
    if (warp == 0 && lane == 0) {                                        // one thread per pipeline
        if (smem_u32(stage) & 127u) __trap();                            // the TMA destinations must be 128-byte aligned
        for (int i = 0; i < NS; ++i) { mbar_init(&tfull[i], 1); mbar_init(&tempty[i], XW); }
        for (int i = 0; i < NR; ++i) { mbar_init(&rfull[i], XW); mbar_init(&rempty[i], YW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();                                                     // the only block barrier
    const long long u0 = ((long long)blockIdx.x * NPIPE + pipe) * per_cta, u1 = min(units, u0 + per_cta);
    if (u0 >= u1) return;
    const size_t np = (size_t)w * h;

    // ------------------------------------------------------------------------------------------- producer
    if (warp == XW + YW) {
        if (lane == 0) {
            Walker wk;
            wk.u = u0; wk.u1 = u1; wk.j = 0; wk.nch = 0; wk.x = 0; wk.a0 = 0; wk.z = 0;
            Ring<NS> s;
            bool wrapped = false;
            Box b;
            while (wk.next(b, w, h, ns, hs, dshift)) {
                if (wrapped) mbar_wait_parked(&tempty[s.i], s.ph ^ 1u);         // the box that used this stage has been read
                mbar_arrive_expect_tx(&tfull[s.i], STAGE_FLOATS * 4);
                tma_load_3d(stage + s.i * STAGE_FLOATS, &tmap, b.x, b.y, b.z, &tfull[s.i]);
                s.next();
                if (s.i == 0) wrapped = true;
            }
        }
        return;
    }

    // ------------------------------------------------------------------------------------------- x warps
    if (warp < XW) {
        Ring<NS> s;
        Ring<NR> q;
        bool qwrapped = false;
        long long u = u0;
        while (u < u1) {
            const long long item = u / h;
            const int ya = (int)(u - item * h);
            const int len = (int)min((long long)(h - ya), u1 - u);
            u += len;
            const Seg sg = make_seg(item, ya, ya + len, w, h, ns, hs, dshift);
            if (sg.nch == 0) continue;
            const float nax = sg.ax.ident ? 0.f : -U_INF;
            const float nax2 = nax * nax, nax4 = nax2 * nax2, nax8 = nax4 * nax4;
            const float scx = sg.ax.ident ? 1.f : 6.0f * U_INF;
            const float wx[4] = {scx * sg.ax.w[0], scx * sg.ax.w[1], scx * sg.ax.w[2], scx * sg.ax.w[3]};
            const bool edge = sg.pL >= 0 || sg.pR >= 0;
            const int i0 = 2 * warp;
            const bool keep = lane >= HL && lane < 32 - HL;
            for (int j = 0; j < sg.nch; ++j) {
                const int a = sg.a0 + CH * j;                            // first source row of the chunk
                mbar_wait_parked(&tfull[s.i], s.ph);
                if (qwrapped) mbar_wait_parked(&rempty[q.i], q.ph ^ 1u);        // the chunk that used this slot has been swept
                if (a + i0 + 1 >= 0) {                                   // rows above the plane are never read
                    float* b0 = stage + s.i * STAGE_FLOATS + i0 * BOXW;
                    float* b1 = b0 + BOXW;
                    if (edge) {
                        x_reflect(b0, sg.pL, sg.pR, lane);
                        x_reflect(b1, sg.pL, sg.pR, lane);
                        // these generic-proxy writes precede the next TMA (async proxy) write to the same stage
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    }
                    float f[2][V];
                    {
                        const float4 p0 = *reinterpret_cast<const float4*>(b0 + V * lane);
                        const float4 p1 = *reinterpret_cast<const float4*>(b0 + V * lane + 4);
                        const float4 q0 = *reinterpret_cast<const float4*>(b1 + V * lane);
                        const float4 q1 = *reinterpret_cast<const float4*>(b1 + V * lane + 4);
                        f[0][0] = p0.x; f[0][1] = p0.y; f[0][2] = p0.z; f[0][3] = p0.w;
                        f[0][4] = p1.x; f[0][5] = p1.y; f[0][6] = p1.z; f[0][7] = p1.w;
                        f[1][0] = q0.x; f[1][1] = q0.y; f[1][2] = q0.z; f[1][3] = q0.w;
                        f[1][4] = q1.x; f[1][5] = q1.y; f[1][6] = q1.z; f[1][7] = q1.w;
                    }
                    rs::x_pass<2>(nax, nax8, wx, f);
                    float* t0 = tring + q.i * T_FLOATS + i0 * TW + V * (lane - HL);
                    switch (sg.r) {          // warp-uniform: the outputs move r positions left
                        case 0: store_rows(t0, keep, f); break;
                        case 1: shift_left<1>(f[0]); shift_left<1>(f[1]); store_rows(t0, keep, f); break;
                        case 2: shift_left<2>(f[0]); shift_left<2>(f[1]); store_rows(t0, keep, f); break;
                        default: shift_left<3>(f[0]); shift_left<3>(f[1]); store_rows(t0, keep, f); break;
                    }
                }
                __syncwarp();
                if (lane == 0) { mbar_arrive(&tempty[s.i]); mbar_arrive(&rfull[q.i]); }
                s.next();
                q.next();
                if (q.i == 0) qwrapped = true;
            }
        }
        return;
    }

    // ------------------------------------------------------------------------------------------- y warps
    const int yw = warp - XW;
    const int ty = yw * 32 + lane;               // the thread's column inside the strip
    Ring<NR> q;
    int qprev = NR - 1;                          // slot of the chunk before
    long long u = u0;
    while (u < u1) {
        const long long item = u / h;
        const int ya = (int)(u - item * h);
        const int len = (int)min((long long)(h - ya), u1 - u);
        const int yb = ya + len;
        u += len;
        const Seg sg = make_seg(item, ya, yb, w, h, ns, hs, dshift);
        float* outk = out + (size_t)sg.k * np;
        {   // rows of the segment without data: fill
            const int cols = sg.Xe - sg.Xs;
            const int nlo = min(sg.ylo, yb) - ya;                        // rows [ya, ya + nlo)
            const int nhi = yb - max(sg.yhi + 1, ya);                    // rows [yb - nhi, yb)
            for (int r = yw; r < nlo + nhi; r += YW) {
                const int y = r < nlo ? ya + r : yb - nhi + (r - nlo);
                float* dst = outk + (size_t)y * w + sg.Xs;
                for (int x = lane * 4; x < cols; x += 128)               // Xs, cols, w: multiples of 4
                    *reinterpret_cast<float4*>(dst + x) = make_float4(fill, fill, fill, fill);
            }
        }
        if (sg.nch == 0) continue;
        const int col = sg.Xs + ty;
        bool ycol = ty < TW && col < sg.Xe;
        YK yk;
        yk.na = -U_INF;
        const float scy = sg.ay.ident ? 1.f : 6.0f * U_INF;
        yk.w0 = scy * sg.ay.w[0]; yk.w1 = scy * sg.ay.w[1]; yk.w2 = scy * sg.ay.w[2]; yk.w3 = scy * sg.ay.w[3];
        yk.my = sg.ay.m; yk.ylo = sg.ylo; yk.yhi = sg.yhi;
        yk.po = outk + (ycol ? col : sg.Xs);
        yk.w = w;
        yk.in0 = col >= sg.ax.lo && col <= sg.ax.hi;
        yk.in1 = yk.in0;
        if (ycol && !yk.in0) {
            // a column outside the x footprint: fill, for every row of the segment that carries data
            for (int y = sg.ylo; y <= sg.yhi; ++y) yk.po[(size_t)((unsigned)y * (unsigned)w)] = fill;
            ycol = false;
        }
        VT gprev, s1, s2, s3;
        vzero(gprev); vzero(s1); vzero(s2); vzero(s3);
        for (int j = 0; j < sg.nch; ++j) {
            const int a = sg.a0 + CH * j;
            mbar_wait_parked(&rfull[q.i], q.ph);
            if (ycol) {
                float* Tc = tring + q.i * T_FLOATS + ty;
                if (sg.ay.ident) {
                    // pure row translation: interval k = source row k, weights (0, 1, 0, 0)
#pragma unroll 4
                    for (int i = 0; i < CH; ++i) {
                        const int y = a + i - yk.my;
                        if (y >= yk.ylo && y <= yk.yhi) { VT t; vld(Tc + i * TW, t); put(yk, yk.po + (size_t)((unsigned)y * (unsigned)w), t); }
                    }
                } else {
                    const bool is_final = a + CH == h;
                    const bool low = a <= CH;                            // rows < LOWROWS: tabulated coefficients
                    const VT A = low ? causal<true>(Tc, a, is_final, yk.na, gprev) : causal<false>(Tc, a, is_final, yk.na, gprev);
                    if (j >= 1 && a - 1 >= sg.kA - 1) {                  // the chunk before holds rows that are evaluated
                        const float* Tp = tring + qprev * T_FLOATS + ty;
                        if (a - CH <= CH) sweep_any<true, false>(Tp, a - CH, A, yk, sg.kA, sg.kB, s1, s2, s3);
                        else sweep_any<false, false, PITCH>(Tp, a - CH, A, yk, sg.kA, sg.kB, s1, s2, s3);
                    }
                    if (is_final && a + CH - 1 >= sg.kA - 1) sweep_any<false, true>(Tc, a, A, yk, sg.kA, sg.kB, s1, s2, s3);
                }
            }
            __syncwarp();
            if (lane == 0) {
                // the chunk before is done with once this chunk has started its sweep; a segment's last chunk (final, or
                // look-ahead only) and every chunk of a pure row translation are done with at once
                if (sg.ay.ident) mbar_arrive(&rempty[q.i]);
                else {
                    if (j >= 1) mbar_arrive(&rempty[qprev]);
                    if (j == sg.nch - 1) mbar_arrive(&rempty[q.i]);
                }
            }
            qprev = q.i;
            q.next();
        }
    }
}

namespace rp {

template <int PITCH>
inline int launch_resample_pipe_t(const float* in, int n, int w, int h, const HostShifts& hs, const double* dshift_dev,
                                  float fill, float* out, int4* fpd, cudaStream_t st)
{
    CUtensorMap tm;
    const cuuint64_t dims[3] = {(cuuint64_t)w, (cuuint64_t)h, (cuuint64_t)n};
    const cuuint64_t strides[2] = {(cuuint64_t)w * 4, (cuuint64_t)w * (cuuint64_t)h * 4};
    const cuuint32_t box[3] = {BOXW, CH, 1};
    if (!tma::encode_f32_map(&tm, in, 3, dims, strides, box)) { set_cuda_error(cudaErrorInvalidValue); return MRED_ECUDA; }
    static PerDeviceOnce once;
    static std::atomic<int> occ_cache[64];
    int dev;
    if (once.pending(dev)) {
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample_pipe<PITCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_P));
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample_pipe<PITCH>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        int occ = 1;
        MRED_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_resample_pipe<PITCH>, NTHR_P * NPIPE, SMEM_P));
        occ *= NPIPE;                                                    // resident pipelines per SM
        if (dev >= 0) occ_cache[dev].store(occ < 1 ? 1 : occ);
        once.mark(dev);
    }
    int occ = dev >= 0 ? occ_cache[dev].load() : 1;
    if (occ < 1) occ = 1;
    const int ns = (w + TW - 1) / TW;
    const long long units = (long long)n * ns * h;
    // resident CTAs: every SM gets `occ`, unless the runs would become so short that their warm-up rows dominate
    const int sms = sm_count();
    long long ctas = (long long)sms * occ;
    while (ctas > sms && units / ctas < 160) ctas -= sms;
    if (ctas > units / CH + 1) ctas = units / CH + 1;
    long long per = (units + ctas - 1) / ctas;
    per = (per + CH - 1) / CH * CH;
    ctas = (units + per - 1) / per;
    k_resample_pipe<PITCH><<<dim3((unsigned)((ctas + NPIPE - 1) / NPIPE)), NTHR_P * NPIPE, SMEM_P, st>>>(tm, n, w, h, ns, units, per, hs, dshift_dev, fill, out, fpd);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

// the configured detector formats (1024 and 4096 columns) get the kernel with the pitch compiled in
inline int launch_resample_pipe(const float* in, int n, int w, int h, const HostShifts& hs, const double* dshift_dev,
                                float fill, float* out, int4* fpd, cudaStream_t st)
{
    if (w == 1024) return launch_resample_pipe_t<1024>(in, n, w, h, hs, dshift_dev, fill, out, fpd, st);
    if (w == 4096) return launch_resample_pipe_t<4096>(in, n, w, h, hs, dshift_dev, fill, out, fpd, st);
    return launch_resample_pipe_t<0>(in, n, w, h, hs, dshift_dev, fill, out, fpd, st);
}

}  // namespace rp
}  // namespace mred
