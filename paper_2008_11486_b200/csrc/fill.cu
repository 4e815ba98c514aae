// fill.cu -- bad-pixel fill (O7, reading Q25; "bad pixel masking", Table 6).
//
// Every masked pixel is replaced by a linear interpolation between the nearest good pixels of the original frame along
// the axis with the shorter gap (ties: x), else by the nearest one-sided good neighbour (order xl, xr, yl, yu), else 0.
// The mask is the same for every frame of a stack, so the work splits in two:
//   k_fill_plan   once per call, mask only: one thread per pixel; a masked pixel searches its row and its column for the
//                 nearest good pixels and appends (pixel, source a, source b, weight of b) to a list in the workspace.
//                 A hot column costs two steps per pixel in x and no search in y (a gap of 2 cannot be beaten).
//   k_fill_apply  per stack: (frame, list entry) -> out[p] = f[a] + (f[b] - f[a]) wb.  Sources are good pixels, targets
//                 masked ones, so the update is in place without hazards.  Traffic: 3 x 4 B per masked pixel and frame
//                 (1 % of the pixels in config 4): a few microseconds, bound by launch latency.
#include "common.cuh"

namespace mred {

struct FillWs {
    int* count;      // [1] entries in the list (zeroed by the plan kernel's launch sequence)
    int4* list;      // [np] {pixel, a, b, float_as_int(wb)}; a = -1: value 0
    size_t bytes;
};

static FillWs carve_fill(void* ws, int w, int h)
{
    FillWs f;
    char* p = static_cast<char*>(ws);
    f.count = reinterpret_cast<int*>(p);
    f.list = reinterpret_cast<int4*>(p + 16);
    f.bytes = 16 + 16 * (size_t)w * h;
    return f;
}

size_t fill_ws_bytes(int w, int h) { return carve_fill(nullptr, w, h).bytes; }

__global__ void __launch_bounds__(256) k_fill_plan(const uint8_t* __restrict__ bad, int w, int h, int* __restrict__ count,
                                                   int4* __restrict__ list)
{
    const size_t np = (size_t)w * h;
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np || !bad[p]) return;
    const int y = (int)((unsigned)p / (unsigned)w), x = (int)((unsigned)p - (unsigned)y * (unsigned)w);
    const uint8_t* row = bad + (size_t)y * w;
    int xl = x - 1, xr = x + 1;
    while (xl >= 0 && row[xl]) --xl;
    while (xr < w && row[xr]) ++xr;
    const bool hx = xl >= 0 && xr < w;
    int yl = y - 1, yu = y + 1;
    bool hy = false;
    if (!(hx && xr - xl == 2)) {                 // a gap of 2 along x is the shortest there is: no need to look along y
        while (yl >= 0 && bad[(size_t)yl * w + x]) --yl;
        while (yu < h && bad[(size_t)yu * w + x]) ++yu;
        hy = yl >= 0 && yu < h;
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
    const int at = atomicAdd(count, 1);          // the order of the entries does not matter: they are independent
    list[at] = make_int4((int)p, a, b, __float_as_int(wb));
}

// grid (blocks, n): grid-stride over the list, whose length is only known on the device
__global__ void __launch_bounds__(256) k_fill_apply(float* __restrict__ frames, size_t np, const int* __restrict__ count,
                                                    const int4* __restrict__ list)
{
    float* f = frames + (size_t)blockIdx.y * np;
    const int cnt = *count;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < cnt; i += gridDim.x * blockDim.x) {
        const int4 e = list[i];
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
    MRED_CUDA_TRY(cudaMemsetAsync(f.count, 0, 16, st));
    k_fill_plan<<<dim3((unsigned)((np + 255) / 256)), 256, 0, st>>>(bad, w, h, f.count, f.list);
    MRED_LAUNCH_CHECK();
    int blocks = (int)((np / 64 + 255) / 256);   // enough threads for a mask of ~1.5 % of the pixels in one sweep
    if (blocks < 1) blocks = 1;
    if (blocks > 4 * sm_count()) blocks = 4 * sm_count();
    k_fill_apply<<<dim3((unsigned)blocks, (unsigned)n), 256, 0, st>>>(frames, np, f.count, f.list);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace mred
