// coadd_stream.cuh -- mean / k-sigma-clipped mean along the stack axis as a streaming pass plus a compacted clip pass
// (O6; "sigma-clipped-mean algorithm", L182).
//
// Why: a thread that keeps its pixel's whole N-frame column in registers and runs up to three clip passes over it issues
// ~27 instructions per value; at N = 60 that is issue-bound at about a third of the HBM rate, with 200+ registers per
// thread and 8 warps per SM.  But a clip pass only matters for the pixels where it rejects something.  So:
//   stage   a block owns 128 consecutive pixels.  Warp 0 issues one 512-byte bulk copy (cp.async.bulk, completion on an
//           mbarrier) per frame: the [N][128] tile lands in shared memory with no register staging, and with 7 blocks per
//           SM at N = 60 some 200 KB per SM are in flight.
//   pass A  thread = pixel, ONE sweep down its column in shared memory with O(1) state: moments about a provisional
//           centre (the median of the first three frames), minimum and maximum.  6 instructions per value, ~30 registers.
//           From these: the mean, the population sigma, and whether the first clip pass would reject anything at all
//           (max |v - mu| > k sigma).  If not -- most pixels -- the result is the mean of everything, exactly what O6 says.
//   pass B  the "dirty" pixels of the block (15-20 % at N = 60, 3 sigma) are compacted into the first ceil(d/32) warps,
//           each thread re-reading one column from shared memory and running the full clip loop (the same float operations
//           as combine_mean_clip, combine.cuh); rejected entries become NaN in shared memory, from which the rejection
//           mask is read off.  Without compaction every warp would run three masked passes for its few dirty lanes.
// Frames whose footprint does not cover the whole tile take the general branch of pass A (per-pixel test, absent = NaN).
// HBM traffic: N * 4 B read + 4 + 2 (+ 4 ceil(N/32)) B written per pixel; requires w * h % 4 == 0 (16-byte aligned tiles).
#pragma once
#include "tma.cuh"

namespace mred {
namespace cs {

constexpr int TP = 128;            // pixels per tile = threads per block

__device__ __forceinline__ float median3(float a, float b, float c)
{
    return fmaxf(fminf(a, b), fminf(fmaxf(a, b), c));
}

// rejection-mask words of one pixel from the NaN entries (absent or rejected) of its column
__device__ __forceinline__ void mask_from_nan(const float* col, int n, uint32_t* __restrict__ rejmask, size_t np, size_t p)
{
    const int words = (n + 31) >> 5;
    for (int wd = 0; wd < words; ++wd) {
        uint32_t bits = 0u;
        const int k0 = 32 * wd, k1 = min(n, k0 + 32);
        for (int k = k0; k < k1; ++k) {
            const float v = col[k * TP];
            if (!(v == v)) bits |= 1u << (k - k0);
        }
        rejmask[(size_t)wd * np + p] = bits;
    }
}

}  // namespace cs

// grid (ceil(np / 128)), block 128, dynamic shared memory n * 512 bytes
__global__ void __launch_bounds__(cs::TP) k_coadd_stream(const float* __restrict__ stack, int n, int w, int h,
                                                         const int4* __restrict__ fp_dev, int use_fp,
                                                         const __grid_constant__ HostFootprints hfp, int clip, float ksigma,
                                                         int max_iter, float* __restrict__ out, uint16_t* __restrict__ count,
                                                         uint32_t* __restrict__ rejmask)
{
    using namespace cs;
    extern __shared__ __align__(128) float vals[];          // [n][TP]
    __shared__ __align__(8) uint64_t s_bar;
    __shared__ unsigned char s_cls[MRED_MAX_STACK + 1];     // 0: frame misses the tile, 1: covers it, 2: covers part of it
    __shared__ short s_list[TP];
    __shared__ int s_nall, s_nnone, s_nd;
    const int tid = threadIdx.x, lane = tid & 31;
    const size_t np = (size_t)w * h;
    const size_t p0 = (size_t)blockIdx.x * TP;
    const int tp = (int)min((size_t)TP, np - p0);           // pixels of this tile (a multiple of 4)
    if (tid == 0) {
        s_nall = 0; s_nnone = 0; s_nd = 0;
        tma::mbar_init(&s_bar, 1);
        tma::fence_mbar_init();
    }
    __syncthreads();
    // classify every frame against the tile's pixels [p0, p0 + tp)
    {
        const size_t p1 = p0 + tp - 1;
        const int ya = (int)((unsigned)p0 / (unsigned)w), yb = (int)((unsigned)p1 / (unsigned)w);      // w * h < 2^31
        const int xa = (int)(p0 - (size_t)ya * w), xb = (int)(p1 - (size_t)yb * w);
        for (int k = tid; k < n; k += TP) {
            int cls = 1;
            if (use_fp) {
                const int4 f = fp_dev ? fp_dev[k] : hfp.fp[k];
                const bool rows_in = ya >= f.z && yb <= f.w, rows_out = yb < f.z || ya > f.w || f.x > f.y;
                if (ya == yb) {
                    const bool cols_in = xa >= f.x && xb <= f.y, cols_out = xb < f.x || xa > f.y;
                    cls = (rows_in && cols_in) ? 1 : ((rows_out || cols_out) ? 0 : 2);
                } else {
                    cls = (rows_in && f.x <= 0 && f.y >= w - 1) ? 1 : (rows_out ? 0 : 2);
                }
            }
            s_cls[k] = (unsigned char)cls;
            if (cls == 1) atomicAdd(&s_nall, 1);
            if (cls == 0) atomicAdd(&s_nnone, 1);
        }
    }
    __syncthreads();
    // stage the tile: one bulk copy per frame that touches it
    if (tid < 32) {
        if (lane == 0) tma::mbar_arrive_expect_tx(&s_bar, (uint32_t)(n - s_nnone) * (uint32_t)tp * 4u);
        __syncwarp();
        for (int k = lane; k < n; k += 32)
            if (s_cls[k]) tma::bulk_load(vals + k * TP, stack + (size_t)k * np + p0, (uint32_t)tp * 4u, &s_bar);
    }
    const bool live = tid < tp;
    const size_t p = p0 + tid;
    float* col = vals + tid;
    const bool fast = s_nall == n;                          // block-uniform: every frame covers every pixel of the tile
    tma::mbar_wait(&s_bar, 0);

    // ---- pass A
    float c0 = 0.f, s1 = 0.f, s2 = 0.f, mn = CUDART_INF_F, mx = -CUDART_INF_F;
    int m = 0;
    if (live) {
        if (fast) {
            c0 = n >= 3 ? median3(col[0], col[TP], col[2 * TP]) : col[0];
#pragma unroll 8
            for (int k = 0; k < n; ++k) {
                const float d = col[k * TP] - c0;
                s1 += d;
                s2 = fmaf(d, d, s2);
                mn = fminf(mn, d);
                mx = fmaxf(mx, d);
            }
            m = n;
        } else {
            const int y = (int)((unsigned)p / (unsigned)w), x = (int)((unsigned)p - (unsigned)y * (unsigned)w);
            for (int k = 0; k < n; ++k) {
                const int cls = s_cls[k];
                bool ok = cls == 1;
                if (cls == 2) {
                    const int4 f = fp_dev ? fp_dev[k] : hfp.fp[k];
                    ok = x >= f.x && x <= f.y && y >= f.z && y <= f.w;
                }
                if (!ok) { col[k * TP] = CUDART_NAN_F; continue; }       // absent: NaN, like a rejected value
                const float v = col[k * TP];
                if (m == 0) c0 = v;
                const float d = v - c0;
                s1 += d;
                s2 = fmaf(d, d, s2);
                mn = fminf(mn, d);
                mx = fmaxf(mx, d);
                ++m;
            }
        }
    }
    bool dirty = false;
    if (live) {
        float value = 0.f;
        if (m > 0) {
            const float mean = s1 / (float)m;
            const float S = fmaxf(s2 - mean * s1, 0.f);
            value = c0 + mean;
            if (clip && max_iter > 0) {
                const float thr = fmaf(ksigma, sqrtf(S / (float)m), 1e-10f * fabsf(value));
                // the first pass would reject something, or the provisional centre sits so far from the mean (it was
                // an outlier itself) that the one-sweep sigma has lost digits: pass B works it out from the values
                dirty = (mx - mean > thr) || (mean - mn > thr) || (mean * mean * (float)m > 16.0f * S);
            }
        }
        if (!dirty) {
            out[p] = value;
            if (count) count[p] = (uint16_t)m;
            if (rejmask) {
                if (fast) {
                    const int words = (n + 31) >> 5;
                    for (int wd = 0; wd < words; ++wd) rejmask[(size_t)wd * np + p] = 0u;
                } else {
                    mask_from_nan(col, n, rejmask, np, p);
                }
            }
        }
    }
    // ---- compaction of the dirty pixels into the first warps
    {
        const unsigned b = __ballot_sync(0xffffffffu, dirty);
        int base = 0;
        if (lane == 0 && b) base = atomicAdd(&s_nd, __popc(b));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (dirty) s_list[base + __popc(b & ((1u << lane) - 1u))] = (short)tid;
    }
    __syncthreads();
    if (tid >= s_nd) return;
    // ---- pass B: the clip loop of combine_mean_clip (combine.cuh) on one column in shared memory; NaN = not used
    {
        const int q = s_list[tid];
        const size_t pq = p0 + q;
        float* cq = vals + q;
        float sum = 0.f;
        int mq = 0;
        for (int k = 0; k < n; ++k) { const float v = cq[k * TP]; if (v == v) { sum += v; ++mq; } }
        const float c = sum / (float)mq;                     // mq > 0: a pixel without values is never dirty
        float t1 = 0.f, t2 = 0.f;
        for (int k = 0; k < n; ++k) { const float d = cq[k * TP] - c; if (d == d) { t1 += d; t2 = fmaf(d, d, t2); } }
        int cnt = mq;
        float mean = t1 / (float)cnt;
        float S = fmaxf(t2 - mean * t1, 0.f);
        for (int it = 0; it < max_iter; ++it) {
            const float thr = fmaf(ksigma, sqrtf(S / (float)cnt), 1e-10f * fabsf(c));
            float n1 = 0.f, n2 = 0.f;
            int ncnt = 0;
            for (int k = 0; k < n; ++k) {
                const float v = cq[k * TP];
                const float t = (v - c) - mean;
                if (fabsf(t) <= thr) { ++ncnt; n1 += t; n2 = fmaf(t, t, n2); }
                else if (v == v) cq[k * TP] = CUDART_NAN_F;
            }
            if (ncnt == cnt) break;
            cnt = ncnt;
            if (cnt == 0) break;
            const float dm = n1 / (float)cnt;
            mean += dm;
            S = fmaxf(n2 - dm * n1, 0.f);
            if (dm * dm * (float)cnt > 0.25f * S) {          // a large outlier left: second moment about the new mean
                float q1 = 0.f, q2 = 0.f;
                for (int k = 0; k < n; ++k) { const float t = (cq[k * TP] - c) - mean; if (t == t) { q1 += t; q2 = fmaf(t, t, q2); } }
                const float dq = q1 / (float)cnt;
                mean += dq;
                S = fmaxf(q2 - dq * q1, 0.f);
            }
        }
        out[pq] = cnt > 0 ? c + mean : 0.f;
        if (count) count[pq] = (uint16_t)cnt;
        if (rejmask) mask_from_nan(cq, n, rejmask, np, pq);
    }
}

}  // namespace mred
