// fill.cu -- bad-pixel fill (O7, reading Q25; "bad pixel masking", Table 6).
//
// Every masked pixel is replaced by a linear interpolation between the nearest good pixels of the original frame along
// the axis with the shorter gap (ties: x), else by the nearest one-sided good neighbour (order xl, xr, yl, yu), else 0.
// The mask is the same for every frame of a stack, so the work splits in two:
//   k_fill_plan   once per call, mask only: one thread per pixel; a masked pixel searches its row and its column for the
//                 nearest good pixels and appends (pixel, source a, source b, weight of b) to a list in the workspace
//                 (a block gathers its entries in shared memory and reserves room with one atomic).
//                 The four searches advance together and stop as soon as the shorter axis is decided (a hot column: one round).
//   k_fill_apply  per stack: (frame, list entry) -> out[p] = f[a] + (f[b] - f[a]) wb.  Sources are good pixels, targets
//                 masked ones, so the update is in place without hazards.  Traffic: 3 x 4 B per masked pixel and frame
//                 (1 % of the pixels in config 4): 22 us for 64 frames, mostly scattered 4-byte accesses.
#include "common.cuh"

namespace mred {

// The list is kept as FILL_NSUB sub-lists, each with its own counter on its own 128-byte line: a block of the plan kernel
// collects its entries in shared memory and reserves room in sub-list (block % FILL_NSUB) with ONE atomic.  (One global
// counter bumped once per masked pixel -- 10 000 same-address atomics for ten hot columns -- took 246 us, 24 ns each: ten
// times the rest of the fill.)
constexpr int FILL_NSUB = 32;      // sub-lists
constexpr int FILL_BPS = 4;        // blocks of the apply kernel per sub-list and frame
constexpr int FILL_CSTRIDE = 32;   // ints between two counters (128 bytes)

struct FillWs {
    int* count;      // [FILL_NSUB] entries of each sub-list, at count[s * FILL_CSTRIDE] (zeroed by the launch sequence)
    int4* list;      // [FILL_NSUB][cap] {pixel, a, b, float_as_int(wb)}; a = -1: value 0
    size_t cap;      // entries a sub-list can hold: the pixels of the blocks that feed it
    size_t bytes;
};

static FillWs carve_fill(void* ws, int w, int h)
{
    FillWs f;
    char* p = static_cast<char*>(ws);
    const size_t np = (size_t)w * h, nblk = (np + 255) / 256;
    f.count = reinterpret_cast<int*>(p);
    f.list = reinterpret_cast<int4*>(p + (size_t)FILL_NSUB * FILL_CSTRIDE * 4);
    f.cap = (nblk + FILL_NSUB - 1) / FILL_NSUB * 256;
    f.bytes = (size_t)FILL_NSUB * FILL_CSTRIDE * 4 + 16 * (size_t)FILL_NSUB * f.cap;
    return f;
}

size_t fill_ws_bytes(int w, int h) { return carve_fill(nullptr, w, h).bytes; }

__global__ void __launch_bounds__(256) k_fill_plan(const uint8_t* __restrict__ bad, int w, int h, int* __restrict__ count,
                                                   int4* __restrict__ list, size_t cap)
{
    __shared__ int s_n, s_base;
    __shared__ int4 s_e[256];
    if (threadIdx.x == 0) s_n = 0;
    __syncthreads();
    const size_t np = (size_t)w * h;
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < np && bad[p]) {
        const int y = (int)((unsigned)p / (unsigned)w), x = (int)((unsigned)p - (unsigned)y * (unsigned)w);
        const uint8_t* row = bad + (size_t)y * w;
        // The four searches (left, right, below, above) advance together, one step each per round (four independent
        // loads), and stop as soon as the answer cannot change: an axis with both neighbours found wins when the other
        // axis, whatever it still finds, cannot have a shorter gap (x wins ties).  So a hot-column pixel beside another
        // masked pixel (x gap 3) looks 2 rows up and down, not down the whole masked column -- searched one after the
        // other, two such pixels held the kernel for 250 us (1024 dependent loads each).  Only a pixel with no pair on
        // either axis walks to the borders (the one-sided rule needs all four distances).
        int xl = x, xr = x, yl = y, yu = y;
        bool rxl = false, rxr = false, ryl = false, ryu = false;      // resolved: a good pixel found there, or the border passed
        bool hx = false, hy = false;
        while (true) {
            if (!rxl) { --xl; rxl = xl < 0 || !row[xl]; }
            if (!rxr) { ++xr; rxr = xr >= w || !row[xr]; }
            if (!ryl) { --yl; ryl = yl < 0 || !bad[(size_t)yl * w + x]; }
            if (!ryu) { ++yu; ryu = yu >= h || !bad[(size_t)yu * w + x]; }
            hx = rxl && rxr && xl >= 0 && xr < w;
            hy = ryl && ryu && yl >= 0 && yu < h;
            const bool nox = (rxl && xl < 0) || (rxr && xr >= w);     // this axis can have no pair
            const bool noy = (ryl && yl < 0) || (ryu && yu >= h);
            const int gx = (xr - xl) + (rxl ? 0 : 1) + (rxr ? 0 : 1); // the gap is at least this
            const int gy = (yu - yl) + (ryl ? 0 : 1) + (ryu ? 0 : 1);
            if (hx && (hy || noy || gy >= xr - xl)) break;            // x pair known; y is known, impossible, or cannot be shorter
            if (hy && (nox || gx > yu - yl)) break;                   // y pair known; x impossible or certainly longer
            if (nox && noy && rxl && rxr && ryl && ryu) break;        // no pair at all: every one-sided distance is known
        }
        int a = -1, b = -1;
        float wb = 0.f;
        if (hx && (!hy || xr - xl <= yu - yl)) {
            a = y * w + xl; b = y * w + xr;
            wb = (float)((double)(x - xl) / (double)(xr - xl));
        } else if (hy) {
            a = yl * w + x; b = yu * w + x;
            wb = (float)((double)(y - yl) / (double)(yu - yl));
        } else {
            int dist = 0;
            if (xl >= 0) { a = y * w + xl; dist = x - xl; }
            if (xr < w && (a < 0 || xr - x < dist)) { a = y * w + xr; dist = xr - x; }
            if (yl >= 0 && (a < 0 || y - yl < dist)) { a = yl * w + x; dist = y - yl; }
            if (yu < h && (a < 0 || yu - y < dist)) { a = yu * w + x; dist = yu - y; }
            b = a;
        }
        s_e[atomicAdd(&s_n, 1)] = make_int4((int)p, a, b, __float_as_int(wb));   // the order of the entries does not matter
    }
    __syncthreads();
    const int nb = s_n;
    if (nb == 0) return;                             // block-uniform
    const int sub = blockIdx.x % FILL_NSUB;
    if (threadIdx.x == 0) s_base = atomicAdd(count + sub * FILL_CSTRIDE, nb);
    __syncthreads();
    if ((int)threadIdx.x < nb) list[(size_t)sub * cap + s_base + threadIdx.x] = s_e[threadIdx.x];
}

// grid (FILL_NSUB * FILL_BPS, n): FILL_BPS blocks stride over each sub-list, whose length is only known on the device
__global__ void __launch_bounds__(256) k_fill_apply(float* __restrict__ frames, size_t np, const int* __restrict__ count,
                                                    const int4* __restrict__ list, size_t cap)
{
    float* f = frames + (size_t)blockIdx.y * np;
    const int sub = blockIdx.x / FILL_BPS, j = blockIdx.x % FILL_BPS;
    const int cnt = count[sub * FILL_CSTRIDE];
    const int4* l = list + (size_t)sub * cap;
    for (int i = j * blockDim.x + threadIdx.x; i < cnt; i += FILL_BPS * blockDim.x) {
        const int4 e = l[i];
        float v = 0.f;
        if (e.y >= 0) {
            const float va = f[e.y], vb = f[e.z];
            v = fmaf(vb - va, __int_as_float(e.w), va);
        }
        f[e.x] = v;
    }
}

int launch_fill_bad(float* frames, int n, int w, int h, const uint8_t* bad, void* ws, cudaStream_t st)
{
    const FillWs f = carve_fill(ws, w, h);
    const size_t np = (size_t)w * h;
    MRED_CUDA_TRY(cudaMemsetAsync(f.count, 0, (size_t)FILL_NSUB * FILL_CSTRIDE * 4, st));
    k_fill_plan<<<dim3((unsigned)((np + 255) / 256)), 256, 0, st>>>(bad, w, h, f.count, f.list, f.cap);
    MRED_LAUNCH_CHECK();
    k_fill_apply<<<dim3((unsigned)(FILL_NSUB * FILL_BPS), (unsigned)n), 256, 0, st>>>(frames, np, f.count, f.list, f.cap);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
