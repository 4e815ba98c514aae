// estimate.cu -- per-frame offset estimation from marginal profiles (O4, reading Q10).
// The paper obtains relative positions from FITS WCS headers on the CPU;
// with no headers here the north star asks for an image-based estimate.
//
//   k_profiles : one streaming pass over the frames (the only HBM traffic, N*4wh B): fixed-point (int64) column
//                partial sums per 32-row band and complete row sums, valid-pixel counts.
//   k_estimate : per (frame, axis): mean from the integer sums, median by a bitonic sort (registers + shuffles inside
//                a warp, shared memory across warps), subtract; C(l) = sum_j a[j] b[j+l], l in [-R, R] against the
//                reference profile; argmax with ties to the smaller |l| then smaller l; 3-point parabola.
// No float atomics: every sum has a fixed order, so the integer result is reproducible.
#include "common.cuh"

namespace mred {

constexpr int PROF_BR = 32;        // rows per band
constexpr int RIF = 4;             // rows in flight per thread in k_profiles
constexpr float FIX = PROF_FIX;    // fixed-point scale of the profile sums (common.cuh)
constexpr int PROF_MAXLEN = MRED_MAX_PROFILE;  // longest profile the finalize kernel holds in shared memory

struct EstimateWs {
    long long* colpart;  // [n][w]   fixed-point column sums (value * FIX), accumulated with integer atomics by the bands
    int* colcnt;      // [n][w]   valid rows per column (contiguous after colpart: zeroed together; used with a mask only)
    unsigned int* ticket;  // [n][2] flags of k_estimate (contiguous after colcnt: zeroed by the same memset)
    long long* rowsum;   // [n][h]
    int* rowcnt;      // [n][h]
    double* prof;     // [n][2][plen]  median-subtracted profiles (x then y)
    double* corr;     // [n][2][2*MRED_MAX_LAG+1]  C(l) of every lag
    size_t zero_bytes, bytes;
    int nbands, plen;
};

static EstimateWs carve_est(void* ws, int w, int h, int n)
{
    EstimateWs e;
    char* p = static_cast<char*>(ws);
    auto take = [&](size_t b) { char* q = p; p += align_up(b, 16); return q; };
    e.nbands = (h + PROF_BR - 1) / PROF_BR;
    e.plen = w > h ? w : h;
    e.colpart = reinterpret_cast<long long*>(take(8 * (size_t)n * w));
    e.colcnt = reinterpret_cast<int*>(take(4 * (size_t)n * w));
    e.ticket = reinterpret_cast<unsigned int*>(take(4 * (size_t)n * 2));
    e.rowsum = reinterpret_cast<long long*>(take(8 * (size_t)n * h));
    e.rowcnt = reinterpret_cast<int*>(take(4 * (size_t)n * h));
    e.zero_bytes = (size_t)(p - static_cast<char*>(ws));    // everything up to here is an accumulator: cleared per call
    e.prof = reinterpret_cast<double*>(take(8 * (size_t)n * 2 * e.plen));
    e.corr = reinterpret_cast<double*>(take(8 * (size_t)n * 2 * (2 * MRED_MAX_LAG + 1)));
    e.bytes = (size_t)(p - static_cast<char*>(ws));
    return e;
}

size_t estimate_ws_bytes(int w, int h, int n) { return carve_est(nullptr, w, h, n).bytes; }

void estimate_accumulators(void* ws, int w, int h, int n, void** zero, size_t* zero_bytes, long long** colsum, long long** rowsum)
{
    const EstimateWs e = carve_est(ws, w, h, n);
    *zero = e.colpart; *zero_bytes = e.zero_bytes; *colsum = e.colpart; *rowsum = e.rowsum;
}

__global__ void __launch_bounds__(256) k_profiles(const float* __restrict__ frames, int w, int h,
                                                  const uint8_t* __restrict__ bad, EstimateWs e, int vec_ok)
{
    __shared__ long long s_row[PROF_BR][8];
    __shared__ int s_cnt[PROF_BR][8];
    const int band = blockIdx.x, k = blockIdx.y;
    const int y0 = band * PROF_BR, y1 = min(y0 + PROF_BR, h);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const float* f = frames + (size_t)k * w * h;
    for (int i = threadIdx.x; i < PROF_BR * 8; i += blockDim.x) { (&s_row[0][0])[i] = 0; (&s_cnt[0][0])[i] = 0; }
    __syncthreads();
    for (int xc = 0; xc < w; xc += 1024) {
        const int x = xc + 4 * threadIdx.x;
        const int nv = max(0, min(4, w - x));
        long long cs[4] = {0, 0, 0, 0};
        int cc[4] = {0, 0, 0, 0};
        for (int yb = y0; yb < y1; yb += RIF) {     // RIF rows in flight per thread
            float v[RIF][4];
            bool ok[RIF][4];
#pragma unroll
            for (int u = 0; u < RIF; ++u) {
#pragma unroll
                for (int i = 0; i < 4; ++i) { v[u][i] = 0.f; ok[u][i] = false; }
                const int y = yb + u;
                if (y >= y1) continue;
                const size_t p = (size_t)y * w + x;
                if (nv == 4 && vec_ok) {
                    const float4 t = __ldcs(reinterpret_cast<const float4*>(f + p));
                    v[u][0] = t.x; v[u][1] = t.y; v[u][2] = t.z; v[u][3] = t.w;
                    ok[u][0] = ok[u][1] = ok[u][2] = ok[u][3] = true;
                    if (bad) {
                        const uchar4 b = __ldg(reinterpret_cast<const uchar4*>(bad + p));
                        ok[u][0] = !b.x; ok[u][1] = !b.y; ok[u][2] = !b.z; ok[u][3] = !b.w;
                    }
                } else {
                    for (int i = 0; i < nv; ++i) { v[u][i] = __ldcs(f + p + i); ok[u][i] = bad ? !__ldg(bad + p + i) : true; }
                }
            }
            // No float64 in the streaming loop: RIF rows are summed in
            // float32 (relative error 6e-8 of an 8-value sum), then accumulated as 64-bit fixed point (value * 2^14):
            // integer adds are exact and order-independent, so the profile is reproducible bit for bit.
            float c4[4] = {0.f, 0.f, 0.f, 0.f}, rs[RIF];
            int rc[RIF];
#pragma unroll
            for (int u = 0; u < RIF; ++u) { rs[u] = 0.f; rc[u] = 0; }
#pragma unroll
            for (int u = 0; u < RIF; ++u)
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (ok[u][i]) { c4[i] += v[u][i]; ++cc[i]; rs[u] += v[u][i]; ++rc[u]; }
#pragma unroll
            for (int i = 0; i < 4; ++i) cs[i] += __float2ll_rn(c4[i] * FIX);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int u = 0; u < RIF; ++u) { rs[u] += __shfl_xor_sync(0xffffffffu, rs[u], o); rc[u] += __shfl_xor_sync(0xffffffffu, rc[u], o); }
            if (lane == 0) {
#pragma unroll
                for (int u = 0; u < RIF; ++u)
                    if (yb + u < y1) { s_row[yb + u - y0][warp] += __float2ll_rn(rs[u] * FIX); s_cnt[yb + u - y0][warp] += rc[u]; }
            }
        }
        for (int i = 0; i < nv; ++i) {
            // integer atomics: exact and order-independent, so no per-band partials have to be kept and re-read
            atomicAdd(reinterpret_cast<unsigned long long*>(e.colpart) + (size_t)k * w + x + i, (unsigned long long)cs[i]);
            if (bad) atomicAdd(e.colcnt + (size_t)k * w + x + i, cc[i]);
        }
    }
    __syncthreads();
    for (int r = threadIdx.x; r < y1 - y0; r += blockDim.x) {
        long long t = 0;
        int c = 0;
        for (int i = 0; i < 8; ++i) { t += s_row[r][i]; c += s_cnt[r][i]; }
        e.rowsum[(size_t)k * h + y0 + r] = t;
        if (bad) e.rowcnt[(size_t)k * h + y0 + r] = c;
    }
}

// Valid-pixel counts per column and per row of the bad-pixel mask, into the count arrays of frame 0 (the mask is the
// same for every frame of a stack, so the chained path counts once and k_estimate reads frame 0's counts for all frames).
// grid (nbands), block 256; the arrays must be zero on entry.
__global__ void __launch_bounds__(256) k_mask_counts(const uint8_t* __restrict__ bad, int w, int h, EstimateWs e)
{
    const int y0 = blockIdx.x * PROF_BR, y1 = min(y0 + PROF_BR, h);
    const int lane = threadIdx.x & 31;
    for (int xc = 0; xc < w; xc += 1024) {
        const int x = xc + 4 * threadIdx.x;
        const int nv = max(0, min(4, w - x));
        int cc[4] = {0, 0, 0, 0};
        for (int y = y0; y < y1; ++y) {
            int rc = 0;
            for (int i = 0; i < nv; ++i) { const int ok = !__ldg(bad + (size_t)y * w + x + i); cc[i] += ok; rc += ok; }
            rc = warp_sum(rc);
            if (lane == 0 && rc) atomicAdd(e.rowcnt + y, rc);
        }
        for (int i = 0; i < nv; ++i)
            if (cc[i]) atomicAdd(e.colcnt + x + i, cc[i]);
    }
}

// order-preserving map double -> uint64
__device__ __forceinline__ unsigned long long key_of(double v)
{
    const unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u >> 63) ? ~u : (u | 0x8000000000000000ULL);
}
__device__ __forceinline__ double val_of(unsigned long long k)
{
    const unsigned long long u = (k >> 63) ? (k & 0x7fffffffffffffffULL) : ~k;
    return __longlong_as_double((long long)u);
}

// Ascending bitonic sort of keys[0..P) in shared memory, P a power of two (block-wide call).
// P <= blockDim.x: one key per thread in a register; the 40 of 55 exchange steps whose partner sits in the same warp are two
// shuffles, only the 15 cross-warp steps go through shared memory (two barriers each).  Larger P: pairs in shared memory.
// A data-independent ~3 us, where the 8-pass radix select it replaces spent ~20 us in barriers and same-bin atomics.
__device__ void block_sort(unsigned long long* keys, int P)
{
    if (P <= (int)blockDim.x) {
        const int i = threadIdx.x;
        unsigned long long v = i < P ? keys[i] : ~0ULL;
        for (int k = 2; k <= P; k <<= 1) {
            for (int j = k >> 1; j > 0; j >>= 1) {
                unsigned long long o;
                if (j >= 32) {
                    __syncthreads();
                    if (i < P) keys[i] = v;
                    __syncthreads();
                    o = i < P ? keys[i ^ j] : v;
                } else {
                    o = __shfl_xor_sync(0xffffffffu, v, j);
                }
                const bool takemin = (((i & j) == 0) == ((i & k) == 0));
                v = takemin ? (o < v ? o : v) : (o > v ? o : v);
            }
        }
        __syncthreads();
        if (i < P) keys[i] = v;
        __syncthreads();
        return;
    }
    for (int k = 2; k <= P; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            __syncthreads();
            for (int t = threadIdx.x; t < (P >> 1); t += blockDim.x) {
                const int i = 2 * t - (t & (j - 1)), l = i + j;
                const unsigned long long a = keys[i], b = keys[l];
                if ((a > b) == ((i & k) == 0)) { keys[i] = b; keys[l] = a; }
            }
        }
    }
    __syncthreads();
}

// Median-subtracted mean profile of frame k along `axis` into dst[0..len) (shared memory); keys[0..P) is scratch
// for the sort (invalid lines get the +inf key, which sorts last).  All threads of the block call it.
__device__ void block_profile(const EstimateWs& e, int w, int h, int k, int axis, int len, int P, int has_bad,
                              double* dst, unsigned long long* keys, int* s_m)
{
    const double INF = __longlong_as_double(0x7ff0000000000000LL);
    if (threadIdx.x == 0) *s_m = 0;
    __syncthreads();
    int mine = 0;
    for (int i = threadIdx.x; i < P; i += blockDim.x) {
        double v = INF;
        if (i < len) {
            long long s = 0;
            int c = axis == 0 ? h : w;         // without a bad-pixel mask every line is complete
            if (axis == 0) {
                s = __ldcg(e.colpart + (size_t)k * w + i);
                if (has_bad) c = __ldcg(e.colcnt + (size_t)(has_bad == 2 ? 0 : k) * w + i);
            } else {
                s = __ldcg(e.rowsum + (size_t)k * h + i);
                if (has_bad) c = __ldcg(e.rowcnt + (size_t)(has_bad == 2 ? 0 : k) * h + i);
            }
            if (c > 0) { v = (double)s / ((double)FIX * (double)c); ++mine; }
            dst[i] = v;
        }
        keys[i] = key_of(v);
    }
    mine = warp_sum(mine);                     // one shared-memory atomic per warp, not per thread:
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(s_m, mine);   // 1024 same-address atomics cost ~15 us
    __syncthreads();
    const int m = *s_m;
    double med = 0.0;
    if (m > 0) {
        block_sort(keys, P);
        med = val_of(keys[(m - 1) >> 1]);
        if (!(m & 1)) med = 0.5 * (med + val_of(keys[m >> 1]));
    }
    for (int i = threadIdx.x; i < len; i += blockDim.x) {
        const double v = dst[i];
        dst[i] = (v == INF) ? 0.0 : v - med;
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------
// k_estimate: profile finishing AND lag search of one (frame, axis) per block (round 1 had two kernels, k_finalize and
// k_correlate: 28-36 us of dependent latency per stack).  grid (n, 2), block 512 (1024 threads, one sort key each, are no
// faster alone -- 30.4 against 30.8 us -- and a 1024-thread block waits longer for room on an SM that other streams' kernels
// share: bench.py's 6-stream step 1.790 -> 1.777 ms; 256 threads: 1.771 ms but 36.6 us alone).  Block x = 0 takes the REFERENCE frame:
// it writes its median-subtracted profile to e.prof and raises a flag (the zeroed ticket of (ref, axis)); every other block
// finishes its own profile (the bitonic sort is the long part, and runs in parallel with the reference's), then waits for
// the flag -- a block only ever waits for the block with x = 0 of its own axis, which precedes it in dispatch order, the
// decoupled look-back pattern -- stages the reference profile in the shared memory the sort no longer needs, and takes
//   C(l) = sum_j a[j] b[j+l], l in [-R, R]   (float64, one lag per warp at a time), the argmax with ties to the smaller |l|
// then the smaller l, and the 3-point (log-)parabola.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_estimate(int w, int h, int n, int ref, int R, int peak, int has_bad, EstimateWs e,
                                                   int32_t* __restrict__ ishift, double* __restrict__ shift)
{
    extern __shared__ double s_dyn[];     // own profile b[P], then sort keys[P] / reference profile a[len]
    __shared__ int s_m;
    __shared__ double sC[2 * MRED_MAX_LAG + 1];
    const int axis = blockIdx.y;
    const int bx = blockIdx.x;
    const int k = bx == 0 ? ref : (bx <= ref ? bx - 1 : bx);
    const int len = axis == 0 ? w : h;
    int P = 1;
    while (P < len) P <<= 1;
    double* b = s_dyn;
    unsigned long long* keys = reinterpret_cast<unsigned long long*>(s_dyn + P);
    block_profile(e, w, h, k, axis, len, P, has_bad, b, keys, &s_m);
    double* gref = e.prof + ((size_t)ref * 2 + axis) * e.plen;
    unsigned int* flag = e.ticket + 2 * ref + axis;
    if (k == ref) {
        for (int i = threadIdx.x; i < len; i += blockDim.x) gref[i] = b[i];
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            atomicExch(flag, 1u);
            ishift[2 * k + axis] = 0;
            shift[2 * k + axis] = 0.0;
        }
        return;
    }
    if (threadIdx.x == 0) {
        while (atomicAdd(flag, 0u) == 0u) __nanosleep(200);
        __threadfence();
    }
    __syncthreads();
    double* a = reinterpret_cast<double*>(keys);          // the sort is done: its scratch holds the reference profile
    for (int i = threadIdx.x; i < len; i += blockDim.x) a[i] = __ldcg(gref + i);
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int q = warp; q <= 2 * R; q += (int)(blockDim.x >> 5)) {
        const int l = q - R;
        const int j0 = max(0, -l), j1 = min(len, len - l);
        double s = 0.0;
        for (int j = j0 + lane; j < j1; j += 32) s = fma(a[j], b[j + l], s);
        s = warp_sum(s);
        if (lane == 0) sC[q] = s;
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    int best = 0;
    for (int l = -R; l <= R; ++l) {
        const double c = sC[l + R], cb = sC[best + R];
        const int al = l < 0 ? -l : l, ab = best < 0 ? -best : best;
        if (c > cb || (c == cb && (al < ab || (al == ab && l < best)))) best = l;
    }
    double delta = 0.0;
    const int ab = best < 0 ? -best : best;
    if (ab < R) {
        double cm = sC[best - 1 + R], c0 = sC[best + R], cp = sC[best + 1 + R];
        if (peak == 1 && cm > 0.0 && c0 > 0.0 && cp > 0.0) { cm = log(cm); c0 = log(c0); cp = log(cp); }   // Gaussian peak (Q27)
        const double den = cm - 2.0 * c0 + cp;
        if (den < 0.0) {
            delta = 0.5 * (cm - cp) / den;
            delta = delta > 0.5 ? 0.5 : (delta < -0.5 ? -0.5 : delta);
        }
    }
    ishift[2 * k + axis] = best;
    shift[2 * k + axis] = (double)best + delta;
}

int launch_mask_counts(const uint8_t* bad, int w, int h, int n, void* ws, cudaStream_t st)
{
    const EstimateWs e = carve_est(ws, w, h, n);
    k_mask_counts<<<dim3(e.nbands), 256, 0, st>>>(bad, w, h, e);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

int launch_estimate(const float* frames, int n, int w, int h, int ref, int max_lag, const uint8_t* bad,
                    int32_t* ishift, double* shift, void* ws, int flags, int peak, cudaStream_t st)
{
    const EstimateWs e = carve_est(ws, w, h, n);
    const int vec_ok = (w % 4 == 0) ? 1 : 0;
    if (!(flags & EST_ZEROED)) MRED_CUDA_TRY(cudaMemsetAsync(e.colpart, 0, e.zero_bytes, st));
    if (!(flags & EST_HAVE_SUMS)) {
        k_profiles<<<dim3(e.nbands, n), 256, 0, st>>>(frames, w, h, bad, e, vec_ok);
        MRED_LAUNCH_CHECK();
    }
    int P = 1;
    while (P < (w > h ? w : h)) P <<= 1;
    static PerDeviceOnce once;
    int dev;
    if (once.pending(dev)) {
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_estimate, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * PROF_MAXLEN * (int)sizeof(double)));
        once.mark(dev);
    }
    k_estimate<<<dim3(n, 2), 512, 2 * (size_t)P * sizeof(double), st>>>(w, h, n, ref, max_lag, peak,
                                                                        bad ? ((flags & EST_SHARED_COUNTS) ? 2 : 1) : 0, e, ishift, shift);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

// ---------------------------------------------------------------------------------------------
// mred_estimate_shifts_static: the scratch of the estimate kernels in a file-scope device array instead of a caller's
// workspace, for callers that cannot allocate (include/mred.h).  Every device that loads the library holds the
// MRED_STATIC_SCRATCH_BYTES of it until the process exits.  In HOST code the array's name is only a handle of the host
// side, not a device address, so the address the kernels get is looked up with cudaGetSymbolAddress, once per device
// with that device current, and kept.  All calls share the array: launch_estimate clears the accumulators and the
// flags at its top (cudaMemsetAsync on the stream), and calls that overlap on the GPU would race on it.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_estimate_scratch[MRED_STATIC_SCRATCH_BYTES];

int launch_estimate_static(const float* frames, int n, int w, int h, int ref, int max_lag, const uint8_t* bad,
                           int32_t* ishift, double* shift, int peak, cudaStream_t st)
{
    if (estimate_ws_bytes(w, h, n) > (size_t)MRED_STATIC_SCRATCH_BYTES) return MRED_ELIMIT;
    static std::atomic<void*> addr[64];
    int dev = -1;
    MRED_CUDA_TRY(cudaGetDevice(&dev));
    void* p = (dev >= 0 && dev < 64) ? addr[dev].load(std::memory_order_acquire) : nullptr;
    if (!p) {
        MRED_CUDA_TRY(cudaGetSymbolAddress(&p, g_estimate_scratch));
        if (!p) { set_cuda_error(cudaErrorInvalidSymbol); return MRED_ECUDA; }
        if (dev >= 0 && dev < 64) addr[dev].store(p, std::memory_order_release);
    }
    return launch_estimate(frames, n, w, h, ref, max_lag, bad, ishift, shift, p, 0, peak, st);
}

}  // namespace mred
