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
//   pass B  the "dirty" pixels of the block (15-20 % at N = 60, 3 sigma) are compacted, and L lanes share each of them
//           (L = 128 / dirty count, a power of two: frames k = sub, sub + L, ..), so the block's threads stay busy and the
//           serial chains are L times shorter.  A clip pass is a sweep of 4 instructions per value (load, two subtractions,
//           compare); only a REJECTED value does more: it is marked NaN in shared memory and taken out of the running
//           count, sum and sum of squares, from which the next mean and sigma follow (sum_kept (t - dm)^2 = S - sum_rej t^2
//           - cnt dm^2, all terms of order N sigma^2; when one outlier carries a quarter of S the moments are taken again
//           in a sweep of their own, so nothing cancels).  The passes start from pass A's statistics.  The rejection mask
//           is read off the NaN marks.  Without compaction every warp would run three masked passes for its few dirty lanes.
// Frames whose footprint does not cover the whole tile take the general branch of pass A (per-pixel test, absent = NaN).
// HBM traffic: N * 4 B read + 4 + 2 (+ 4 ceil(N/32)) B written per pixel; requires w * h % 4 == 0 (16-byte aligned tiles).
#pragma once
#include "tma.cuh"

namespace mred {
namespace cs {

constexpr int TP = 128;            // pixels per tile = threads per block
constexpr int TPS = 132;           // row pitch of the staged tile in floats: 528 B (a multiple of 16 for the bulk copies);
                                   // 132 = 4 (mod 32), so the lanes that share one pixel's column in pass B (frames k, k+1, ..)
                                   // hit different banks, and pass A (consecutive pixels of one frame) is conflict-free anyway

__device__ __forceinline__ float median3(float a, float b, float c)
{
    return fmaxf(fminf(a, b), fminf(fmaxf(a, b), c));
}

// sum over the L lanes (L a power of two, lanes aligned to L) that share a pixel; every lane gets the total
__device__ __forceinline__ float group_sum(float v, int L, unsigned gmask)
{
    for (int o = L >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(gmask, v, o);
    return v;
}
__device__ __forceinline__ int group_sum(int v, int L, unsigned gmask)
{
    for (int o = L >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(gmask, v, o);
    return v;
}

}  // namespace cs

// grid (ceil(np / 128)), block 128, dynamic shared memory n * 528 bytes
__global__ void __launch_bounds__(cs::TP) k_coadd_stream(const float* __restrict__ stack, int n, int w, int h,
                                                         const int4* __restrict__ fp_dev, int use_fp,
                                                         const __grid_constant__ HostFootprints hfp, int clip, float ksigma,
                                                         int max_iter, float* __restrict__ out, uint16_t* __restrict__ count,
                                                         uint32_t* __restrict__ rejmask)
{
    using namespace cs;
    extern __shared__ __align__(128) float vals[];          // [n][TPS]
    __shared__ __align__(8) uint64_t s_bar;
    __shared__ unsigned char s_cls[MRED_MAX_STACK + 1];     // 0: frame misses the tile, 1: covers it, 2: covers part of it
    __shared__ short s_list[TP];
    __shared__ float s_c0[TP], s_mean[TP], s_S[TP];         // pass A's statistics of the dirty pixels, for pass B
    __shared__ short s_m[TP];                               // values in the column; negative: statistics unusable (recentre)
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
            if (s_cls[k]) tma::bulk_load(vals + k * TPS, stack + (size_t)k * np + p0, (uint32_t)tp * 4u, &s_bar);
    }
    const bool live = tid < tp;
    const size_t p = p0 + tid;
    float* col = vals + tid;
    const bool fast = s_nall == n;                          // block-uniform: every frame covers every pixel of the tile
    const bool do_clip = clip && max_iter > 0;
    const int words = (n + 31) >> 5;
    // one warp polls the mbarrier, the others sleep at the block barrier (128 polling threads took a fifth of all issue
    // slots away from the blocks that had their data); the barrier carries the copies' visibility on to them
    if (tid < 32) tma::mbar_wait(&s_bar, 0);
    __syncthreads();

    // ---- pass A
    bool dirty = false;
    if (live) {
        float value = 0.f;
        int m = 0;
        if (!fast) {
            // frames that do not cover this pixel become NaN in the staged column: absent, like a rejected value
            const int y = (int)((unsigned)p / (unsigned)w), x = (int)((unsigned)p - (unsigned)y * (unsigned)w);
            for (int k = 0; k < n; ++k) {
                const int cls = s_cls[k];
                if (cls == 1) continue;                      // block-uniform
                bool ok = false;
                if (cls == 2) {
                    const int4 f = fp_dev ? fp_dev[k] : hfp.fp[k];
                    ok = x >= f.x && x <= f.y && y >= f.z && y <= f.w;
                }
                if (!ok) col[k * TPS] = CUDART_NAN_F;
            }
        }
        if (!do_clip) {
            // plain mean, compensated: the sum, then the sum of the residuals about the float32 mean (what the first
            // sum lost to rounding next to a 60000-ADU outlier comes back with the second)
            float sum = 0.f;
            if (fast) {
#pragma unroll 8
                for (int k = 0; k < n; ++k) sum += col[k * TPS];
                m = n;
            } else {
                for (int k = 0; k < n; ++k) { const float v = col[k * TPS]; if (v == v) { sum += v; ++m; } }
            }
            if (m > 0) {
                const float c = sum / (float)m;
                float r1 = 0.f;
                if (fast) {
#pragma unroll 8
                    for (int k = 0; k < n; ++k) r1 += col[k * TPS] - c;
                } else {
                    for (int k = 0; k < n; ++k) { const float d = col[k * TPS] - c; if (d == d) r1 += d; }
                }
                value = c + r1 / (float)m;
            }
        } else {
            // one sweep with O(1) state: moments about a provisional centre, minimum and maximum
            float c0 = 0.f, s1 = 0.f, s2 = 0.f, mn = CUDART_INF_F, mx = -CUDART_INF_F;
            if (fast) {
                c0 = n >= 3 ? median3(col[0], col[TPS], col[2 * TPS]) : col[0];
#pragma unroll 8
                for (int k = 0; k < n; ++k) {
                    const float d = col[k * TPS] - c0;
                    s1 += d;
                    s2 = fmaf(d, d, s2);
                    mn = fminf(mn, d);
                    mx = fmaxf(mx, d);
                }
                m = n;
            } else {
                int k0 = 0;
                while (k0 < n && !(col[k0 * TPS] == col[k0 * TPS])) ++k0;      // first frame that covers the pixel
                c0 = k0 < n ? col[k0 * TPS] : 0.f;
#pragma unroll 4
                for (int k = 0; k < n; ++k) {                // branch-free: fminf / fmaxf skip NaN by themselves
                    const float d = col[k * TPS] - c0;
                    const bool ok = d == d;
                    const float dz = ok ? d : 0.f;
                    s1 += dz;
                    s2 = fmaf(dz, dz, s2);
                    mn = fminf(mn, d);
                    mx = fmaxf(mx, d);
                    m += ok ? 1 : 0;
                }
            }
            if (m > 0) {
                const float mean = s1 / (float)m;
                const float S = fmaxf(s2 - mean * s1, 0.f);
                value = c0 + mean;
                const float thr = fmaf(ksigma, sqrtf(S / (float)m), 1e-10f * fabsf(value));
                // the provisional centre sits far from the mean (it was an outlier itself): the one-sweep sigma has lost
                // digits, pass B takes the moments again about the mean
                const bool recentre = mean * mean * (float)m > 16.0f * S;
                dirty = (mx - mean > thr) || (mean - mn > thr) || recentre;      // the first pass would reject something
                if (dirty) { s_c0[tid] = c0; s_mean[tid] = mean; s_S[tid] = S; s_m[tid] = (short)(recentre ? -m : m); }
            }
        }
        if (!dirty) {
            out[p] = value;
            if (count) count[p] = (uint16_t)m;
            if (rejmask) {
                for (int wd = 0; wd < words; ++wd) {
                    uint32_t bits = 0u;
                    if (!fast) {
                        const int k0 = 32 * wd, k1 = min(n, k0 + 32);
                        for (int k = k0; k < k1; ++k) { const float v = col[k * TPS]; if (!(v == v)) bits |= 1u << (k - k0); }
                    }
                    rejmask[(size_t)wd * np + p] = bits;
                }
            }
        }
    }
    // ---- compaction of the dirty pixels
    {
        const unsigned b = __ballot_sync(0xffffffffu, dirty);
        int base = 0;
        if (lane == 0 && b) base = atomicAdd(&s_nd, __popc(b));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (dirty) s_list[base + __popc(b & ((1u << lane) - 1u))] = (short)tid;
    }
    __syncthreads();
    const int nd = s_nd;
    if (nd == 0) return;
    // ---- pass B: the clip loop (same float operations as combine_mean_clip, combine.cuh) on the dirty columns, L lanes per
    // column (L = the largest power of two that lets the block take all of them at once): each lane owns frames
    // sub, sub + L, ..; the three sums of a pass are reduced over the group by shuffles.  NaN = not used.
    int L = 1;
    while (L < 32 && 2 * L * nd <= TP && 2 * L <= n) L <<= 1;
    const int sub = tid & (L - 1);
    const unsigned gmask = (L == 32) ? 0xffffffffu : (((1u << L) - 1u) << (lane & ~(L - 1)));
    for (int gi = tid / L; gi < nd; gi += TP / L) {
        const int q = s_list[gi];
        const size_t pq = p0 + q;
        float* cq = vals + q;
        int cnt = s_m[q];
        float c = s_c0[q], mean = s_mean[q], S = s_S[q];
        if (cnt < 0) {                                       // take the moments again about the mean
            cnt = -cnt;
            float sum = 0.f;
            for (int k = sub; k < n; k += L) { const float v = cq[k * TPS]; if (v == v) sum += v; }
            c = group_sum(sum, L, gmask) / (float)cnt;
            float t1 = 0.f, t2 = 0.f;
            for (int k = sub; k < n; k += L) { const float d = cq[k * TPS] - c; if (d == d) { t1 += d; t2 = fmaf(d, d, t2); } }
            t1 = group_sum(t1, L, gmask);
            t2 = group_sum(t2, L, gmask);
            mean = t1 / (float)cnt;
            S = fmaxf(t2 - mean * t1, 0.f);
        }
        // mean, S: mean and centred sum of squares of the cnt survivors, both about c (sum of (v - c) - mean over them = 0)
        for (int it = 0; it < max_iter; ++it) {
            const float thr = fmaf(ksigma, sqrtf(S / (float)cnt), 1e-10f * fabsf(c));
            float r1 = 0.f, r2 = 0.f;                        // sum and sum of squares of what this pass rejects
            int rc = 0;
            for (int k = sub; k < n; k += L) {
                const float t = (cq[k * TPS] - c) - mean;
                if (fabsf(t) > thr) {                        // false for NaN (absent / rejected before)
                    cq[k * TPS] = CUDART_NAN_F;
                    ++rc; r1 += t; r2 = fmaf(t, t, r2);
                }
            }
            rc = group_sum(rc, L, gmask);
            if (rc == 0) break;                              // group-uniform: nothing rejected
            r1 = group_sum(r1, L, gmask);
            r2 = group_sum(r2, L, gmask);
            cnt -= rc;
            if (cnt == 0) break;
            const float dm = -r1 / (float)cnt;               // the survivors' deviations summed to -r1: their mean moves by dm
            mean += dm;
            if (r2 > 0.25f * S) {
                // what left carried a good part of S (a cosmic ray, a hot column): S - r2 would cancel, so the second moment
                // of the survivors is taken again, about the new mean, in a sweep of its own (q1 mops up what dm lost
                // to rounding next to the outlier)
                float q1 = 0.f, q2 = 0.f;
                for (int k = sub; k < n; k += L) { const float t = (cq[k * TPS] - c) - mean; if (t == t) { q1 += t; q2 = fmaf(t, t, q2); } }
                q1 = group_sum(q1, L, gmask);
                q2 = group_sum(q2, L, gmask);
                const float dq = q1 / (float)cnt;
                mean += dq;
                S = fmaxf(q2 - dq * q1, 0.f);
            } else {
                S = fmaxf((S - r2) - dm * dm * (float)cnt, 0.f);
            }
        }
        if (sub == 0) {
            out[pq] = cnt > 0 ? c + mean : 0.f;
            if (count) count[pq] = (uint16_t)cnt;
        }
        if (rejmask) {
            __syncwarp(gmask);                               // the NaN marks of the other lanes of the group
            for (int wd = 0; wd < words; ++wd) {
                uint32_t bits = 0u;
                const int k0 = 32 * wd, k1 = min(n, k0 + 32);
                for (int k = k0 + sub; k < k1; k += L) { const float v = cq[k * TPS]; if (!(v == v)) bits |= 1u << (k - k0); }
                for (int o = L >> 1; o > 0; o >>= 1) bits |= __shfl_xor_sync(gmask, bits, o);
                if (sub == 0) rejmask[(size_t)wd * np + pq] = bits;
            }
        }
    }
}

}  // namespace mred
