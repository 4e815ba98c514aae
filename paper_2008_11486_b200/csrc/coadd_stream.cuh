// coadd_stream.cuh -- mean / k-sigma-clipped mean along the stack axis as a streaming pass plus a compacted clip pass
// (O6; "sigma-clipped-mean algorithm", L182).
//
// Why: a thread that keeps its pixel's whole N-frame column in registers and runs up to three clip passes over it issues
// ~27 instructions per value; at N = 60 that is issue-bound at about a third of the HBM rate, with 200+ registers per
// thread and 8 warps per SM.  But a clip pass only matters for the pixels where it rejects something.  So:
//   stage   a block owns 128 consecutive pixels.  One cp.async.bulk.tensor box (132 pixels x N frames through a 2-D tensor
//           map over the [N][w*h] stack, completion on an mbarrier) brings the whole tile into shared memory with no
//           register staging; with 6 blocks per SM at N = 60 some 190 KB per SM are in flight.
//   pass A  thread = pixel, ONE sweep down its column in shared memory with O(1) state: moments about a provisional
//           centre (the median of the first three frames), minimum and maximum.  6 instructions per value, ~30 registers.
//           From these: the mean, the population sigma, and whether the first clip pass would reject anything at all
//           (max |v - mu| > k sigma).  If not -- most pixels -- the result is the mean of everything, exactly what O6 says.
//   pass B  the "dirty" pixels of the block (15-20 % at N = 60, 3 sigma) are compacted, and L lanes share each of them
//           (L = 128 / dirty count, a power of two: frames k = sub, sub + L, ..), so the block's threads stay busy and the
//           serial chains are L times shorter.  A clip pass is one branch-free sweep (cs::clip_dirty); what it rejects is
//           marked NaN in shared memory and its count, sum and sum of squares give the next mean and sigma (sum_kept
//           (t - dm)^2 = S - sum_rej t^2 - cnt dm^2, all terms of order N sigma^2; when one outlier carries a quarter of S
//           the second moment is taken again in a sweep of its own, so nothing cancels).  The passes start from pass A's
//           statistics.  The rejection mask is read off the NaN marks.  Without compaction every warp would run three
//           masked passes for its few dirty lanes.
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

struct ClipArgs {
    float* vals; const short* list; const float *c0, *mean, *S; const short* m;
    int n, nd; float ksigma; int max_iter; size_t p0, np;
    float* out; uint16_t* count; uint32_t* rejmask;
};

template <int L>
__device__ __forceinline__ float gsum(float v, unsigned gmask)
{
#pragma unroll
    for (int o = L >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(gmask, v, o);
    return v;
}
template <int L>
__device__ __forceinline__ int gsum(int v, unsigned gmask)
{
#pragma unroll
    for (int o = L >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(gmask, v, o);
    return v;
}

// The clip loop of O6 on the dirty columns.  L lanes share a column: lane `sub` owns frames sub, sub + L, ...  A pass is
// ONE branch-free sweep (per value: load, two subtractions, compare, select, two accumulates, a predicated count and a
// predicated store of the NaN mark): with 16 columns per warp some lane rejects at almost every step, so a branch around
// the "rare" rejection would be taken all the time.  The survivors' moments are accumulated about the column's provisional
// centre c (pass A: the median of three frames, within a sigma of the survivors' mean whatever the outliers are), NOT about
// the mean that is being clipped against, which still holds the outliers: so mean' = m1 / cnt and S' = m2 - mean' m1 do
// not cancel even when a 60000-ADU hit has just left, and no second sweep is needed.  Only a centre that was an outlier
// itself (|mean'| > 4 sigma) is moved and the moments taken again.  NaN = not used.
template <int L>
__device__ __forceinline__ void clip_dirty(const ClipArgs& a, int tid)
{
    const int lane = tid & 31, sub = tid & (L - 1);
    const unsigned gmask = (L == 32) ? 0xffffffffu : (((1u << L) - 1u) << (lane & ~(L - 1)));
    const int n = a.n;
    constexpr int STEP = L * TPS;                            // this lane's next frame is L rows on
    for (int gi = tid / L; gi < a.nd; gi += TP / L) {
        const int q = a.list[gi];
        const size_t pq = a.p0 + q;
        float* cq = a.vals + q + sub * TPS;
        const int nk = (n - sub + L - 1) / L;                // frames of this lane
        int cnt = a.m[q];
        float c = a.c0[q], mean = a.mean[q], S = a.S[q];
        bool recentre = cnt < 0;
        cnt = recentre ? -cnt : cnt;
        for (int it = 0; it < a.max_iter; ++it) {
            if (recentre) {                                  // group-uniform, rare: centre on the survivors' mean
                c += mean;
                float t1 = 0.f, t2 = 0.f;
#pragma unroll 4
                for (int i = 0; i < nk; ++i) { float d = cq[i * STEP] - c; d = (d == d) ? d : 0.f; t1 += d; t2 = fmaf(d, d, t2); }
                t1 = gsum<L>(t1, gmask);
                t2 = gsum<L>(t2, gmask);
                mean = t1 / (float)cnt;
                S = fmaxf(t2 - mean * t1, 0.f);
            }
            const float thr = fmaf(a.ksigma, sqrtf(S / (float)cnt), 1e-10f * fabsf(c));
            float m1 = 0.f, m2 = 0.f;                        // survivors: sum and sum of squares of v - c
            int ncnt = 0;
#pragma unroll 4
            for (int i = 0; i < nk; ++i) {
                const float u = cq[i * STEP] - c;
                const bool keep = fabsf(u - mean) <= thr;    // false for NaN (absent / rejected before)
                const float uk = keep ? u : 0.f;
                m1 += uk;
                m2 = fmaf(uk, uk, m2);
                ncnt += keep ? 1 : 0;
                if (!keep) cq[i * STEP] = CUDART_NAN_F;      // a predicated store
            }
            ncnt = gsum<L>(ncnt, gmask);
            if (ncnt == cnt) break;                          // group-uniform: nothing rejected
            cnt = ncnt;
            if (cnt == 0) break;
            m1 = gsum<L>(m1, gmask);
            m2 = gsum<L>(m2, gmask);
            mean = m1 / (float)cnt;
            S = fmaxf(m2 - mean * m1, 0.f);
            recentre = mean * mean * (float)cnt > 16.0f * S;
        }
        if (sub == 0) {
            a.out[pq] = cnt > 0 ? c + mean : 0.f;
            if (a.count) a.count[pq] = (uint16_t)cnt;
        }
        if (a.rejmask) {
            // mask words from the NaN marks; L divides 32, so word wd holds this lane's frames i in [wd 32/L, (wd+1) 32/L)
            constexpr int PER = 32 / L;
            const int words = (n + 31) >> 5;
            for (int wd = 0; wd < words; ++wd) {
                uint32_t bits = 0u;
#pragma unroll
                for (int j = 0; j < PER; ++j) {
                    const int i = wd * PER + j;
                    if (i < nk) { const float v = cq[i * STEP]; if (!(v == v)) bits |= 1u << (sub + j * L); }
                }
#pragma unroll
                for (int o = L >> 1; o > 0; o >>= 1) bits |= __shfl_xor_sync(gmask, bits, o);
                if (sub == 0) a.rejmask[(size_t)wd * a.np + pq] = bits;
            }
        }
    }
}

}  // namespace cs

// grid (ceil(np / 128)), block 128, dynamic shared memory n * 528 bytes; tmap: dims {w*h, n}, box {132, n}
__global__ void __launch_bounds__(cs::TP) k_coadd_stream(const __grid_constant__ CUtensorMap tmap, int n, int w, int h,
                                                         const int4* __restrict__ fp_dev, int use_fp,
                                                         const __grid_constant__ HostFootprints hfp, int mode, float ksigma,
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
    __shared__ unsigned char s_nfl[MRED_MAX_STACK + 1];     // the frames that do not cover the whole tile (any order)
    __shared__ int s_nall, s_nnone, s_nd, s_nnf;
    const int tid = threadIdx.x, lane = tid & 31;
    const size_t np = (size_t)w * h;
    const size_t p0 = (size_t)blockIdx.x * TP;
    const int tp = (int)min((size_t)TP, np - p0);           // pixels of this tile (a multiple of 4)
    // stage the tile: ONE tensor copy, a box of TPS pixels x n frames out of the [n][w*h] stack, issued before anything else
    // so that the classification of the frames below runs under the copy.  (One 512-byte bulk copy per frame, 60 per tile,
    // held the whole kernel at 3.5 TB/s: the copy engine takes a copy every ~40 cycles per SM whatever its size.)  The box
    // is 4 pixels wider than the tile, so the rows land with the 132-float pitch that keeps pass B free of bank conflicts;
    // pixels beyond the plane arrive as zeros and are never looked at.
    if (tid == 0) {
        s_nall = 0; s_nnone = 0; s_nd = 0; s_nnf = 0;
        tma::mbar_init(&s_bar, 1);
        tma::fence_mbar_init();
        tma::mbar_arrive_expect_tx(&s_bar, (uint32_t)n * (uint32_t)TPS * 4u);
        tma::tma_load_2d(vals, &tmap, (int)p0, 0, &s_bar);
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
            else s_nfl[atomicAdd(&s_nnf, 1)] = (unsigned char)k;
            if (cls == 0) atomicAdd(&s_nnone, 1);
        }
    }
    __syncthreads();
    const bool live = tid < tp;
    const size_t p = p0 + tid;
    float* col = vals + tid;
    const bool fast = s_nall == n;                          // block-uniform: every frame covers every pixel of the tile
    const bool do_clip = mode == MRED_SIGCLIP && max_iter > 0;
    const bool minmax = mode == MRED_MINMAX;
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
            const int nnf = s_nnf;
            for (int i = 0; i < nnf; ++i) {                  // only the frames that miss part of the tile
                const int k = s_nfl[i];
                const int4 f = fp_dev ? fp_dev[k] : hfp.fp[k];
                const bool ok = (unsigned)(x - f.x) <= (unsigned)(f.y - f.x) && (unsigned)(y - f.z) <= (unsigned)(f.w - f.z) &&
                                f.x <= f.y && f.z <= f.w;
                if (!ok) col[k * TPS] = CUDART_NAN_F;
            }
        }
        bool nan_marks = !fast;              // the column holds NaN marks (absent frames, minmax rejects) for the mask
        if (minmax) {
            // NEXT-2 variant (Q26): one minimum and one maximum (first occurrences in frame order) are left out,
            // mean of the rest; fewer than 3 values: plain mean.  Compensated like the plain mean below.
            float sum = 0.f, mn = CUDART_INF_F, mx = -CUDART_INF_F;
            int imn = -1, imx = -1;
            for (int k = 0; k < n; ++k) {
                const float v = col[k * TPS];
                if (!(v == v)) continue;
                sum += v; ++m;
                if (v < mn) { mn = v; imn = k; }
                if (v > mx) { mx = v; imx = k; }
            }
            if (m >= 3) {
                if (imx == imn) {            // every value equal: the maximum is the first entry other than the minimum
                    imx = -1;
                    for (int k = 0; k < n && imx < 0; ++k) { const float v = col[k * TPS]; if (v == v && k != imn) imx = k; }
                }
                const float c = sum / (float)m;
                float r1 = 0.f;
                for (int k = 0; k < n; ++k) { const float d = col[k * TPS] - c; if (d == d) r1 += d; }
                value = c + ((r1 - (mn - c)) - (mx - c)) / (float)(m - 2);
                col[imn * TPS] = CUDART_NAN_F;
                col[imx * TPS] = CUDART_NAN_F;
                m -= 2;
                nan_marks = true;
            } else if (m > 0) {
                value = sum / (float)m;
            }
        } else if (!do_clip) {
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
                    if (nan_marks) {
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
    // ---- pass B on the compacted dirty columns, L lanes per column (the largest power of two that lets the block take all
    // of them at once)
    int L = 1;
    while (L < 32 && 2 * L * nd <= TP && 2 * L <= n) L <<= 1;
    const ClipArgs ca{vals, s_list, s_c0, s_mean, s_S, s_m, n, nd, ksigma, max_iter, p0, np, out, count, rejmask};
    switch (L) {
        case 1: clip_dirty<1>(ca, tid); break;
        case 2: clip_dirty<2>(ca, tid); break;
        case 4: clip_dirty<4>(ca, tid); break;
        case 8: clip_dirty<8>(ca, tid); break;
        case 16: clip_dirty<16>(ca, tid); break;
        default: clip_dirty<32>(ca, tid); break;
    }
}

}  // namespace mred
