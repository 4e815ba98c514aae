// resample_tile.cuh -- the CTA-tiled, TMA-staged spline-shift kernel (the route for planes with 16-byte-aligned rows,
// w >= 256, h >= 64: every configured detector format).  Mathematics: resample.cu; O5 (PAPER.md L63, L107, L164,
// L266).
//
// A CTA (256 threads) owns a run of (frame, strip of 208 output columns, output rows [ya, yb)) segments; the runs are an
// even split of all n * strips * h strip-rows over the resident CTAs, so no wave is left half empty.  It walks a segment
// in chunks of 16 source rows:
//   TMA      one cp.async.bulk.tensor box of 256 columns x 16 rows per chunk, 3 chunks in flight per CTA, completion on an
//            mbarrier.  Columns / rows outside the plane arrive as zeros.  The box must start on a 16-byte boundary
//            (an unaligned inner coordinate raises an illegal-instruction fault on sm_100a), so it starts r = 0..3 columns
//            left of the source column the strip needs; the x pass works at the box's alignment and moves its OUTPUT
//            r columns (r register renames + r shuffles per row, a warp-uniform switch over r).
//   x pass   warp = 2 rows of the chunk out of shared memory, lane = 8 consecutive samples: the constant-coefficient
//            causal / anti-causal recursions inside the lane, lane-to-lane carries by shuffle (rs::x_pass), the 4 x taps;
//            the 208 kept columns go to a shared-memory ring.  Strips that touch an image edge first write the
//            point-reflected halo (f(-i) = 2 f(0) - f(i)) into the staged rows.
//   y pass   thread = one column, streaming down the chunks: causal recursion in place in the ring, the look-ahead sum that
//            starts the anti-causal sweep of the chunk before (16 rows: a^16 = 7e-10), the sweep with the 4 y taps, one
//            coalesced 128-byte store per warp and row.  The first rows of a plane use the EXACT elimination coefficients
//            of the natural-spline system (u_0 = 0, u_i = 1 / (4 - u_{i-1}), c_0 = f_0) and the last row c_{h-1} = f_{h-1},
//            with the virtual c_{-1} = 2 c_0 - c_1, c_h = 2 c_{h-1} - c_{h-2}: no rows beyond the plane are ever needed.
// Shared memory: 3 x 16 KB stages + 2 x 13 KB ring = 74.8 KB, three CTAs (24 warps) per SM.
// HBM traffic: 4 B read (x 256/208 through L2 for the strip halos) + 4 B written per pixel; a segment that starts inside a
// plane re-reads 17-32 rows of warm-up.
#pragma once
#include "tma.cuh"

namespace mred {
namespace rt {

using rs::Axis;
using rs::make_axis;
using rs::U_INF;
using rs::V;

constexpr int CH = 16;                  // source rows per chunk
constexpr int BOXW = 256;               // source columns per chunk row (32 lanes x 8)
constexpr int TW = rs::OUTCOLS;         // 208 output columns per strip
constexpr int HL = rs::HALO_L;          // 3 halo lanes on either side
constexpr int NSTAGE = 3;               // TMA boxes in flight per CTA
constexpr int NTHR = 256;
constexpr int LOWROWS = 32;             // rows whose elimination coefficients differ from their limit a (to float32: ~12)
constexpr int STAGE_FLOATS = CH * BOXW; // 16 KB
constexpr int T_FLOATS = CH * TW;       // 13 KB
constexpr int MIN_W = BOXW, MIN_H = 64; // smaller planes take the warp kernels of resample_warp.cuh

template <int NT> constexpr size_t smem_bytes()
{
    return (size_t)NSTAGE * STAGE_FLOATS * 4 + (size_t)NT * T_FLOATS * 4 + NSTAGE * 8;
}

// Natural-spline elimination from the first row (O5): u_0 = 0, u_i = 1 / (4 - u_{i-1}) -> a = 2 - sqrt(3).  In
// units of c' = c / 6a the forward pass is g_i = p_i f_i - u_i g_{i-1} with p_0 = 1 / 6a, p_i = u_i / a, and the back
// substitution c'_i = g_i - u_i c'_{i+1}.  Beyond row ~12 the coefficients equal their limits to float32.
struct LowTab { float u[LOWROWS], p[LOWROWS]; };
__host__ __device__ constexpr LowTab make_low()
{
    LowTab t{};
    const double a = 0.26794919243112270647;
    double u = 0.0;
    for (int i = 0; i < LOWROWS; ++i) {
        if (i > 0) u = 1.0 / (4.0 - u);
        t.u[i] = (float)u;
        t.p[i] = (float)(i == 0 ? 1.0 / (6.0 * a) : u / a);
    }
    return t;
}
__constant__ LowTab c_low = make_low();

struct PowTab { float v[CH]; };
__host__ __device__ constexpr PowTab make_pow()
{
    PowTab t{};
    double p = 1.0;
    for (int i = 0; i < CH; ++i) { t.v[i] = (float)p; p *= -(double)U_INF; }
    return t;
}

using tma::smem_u32;
using tma::mbar_init;
using tma::mbar_arrive_expect_tx;
using tma::mbar_wait;
using tma::tma_load_3d;

// ---- one segment: output rows [ya, yb) of strip s of frame k ---------------------------------------------------------
struct Seg {
    int k, Xs, Xe;        // frame; kept output columns [Xs, Xe)
    int xsrc0;            // source column under warp position 0 (may be negative; a multiple of 4: TMA boxes start 16-byte aligned)
    int r;                // 0..3: the strip's outputs sit r positions to the right of the box alignment
    int ylo, yhi;         // output rows of the segment that carry data (inclusive; ylo > yhi: none)
    int a0, nch;          // first source row of chunk 0 (may be negative), number of chunks
    int kA, kB;           // first and last interval (source row index) evaluated
    int pL, pR;           // warp position of image column 0 / w-1 when the box reaches beyond that edge, else -1
    Axis ax, ay;
};

// largest row g <= v on the chunk grid g = h (mod 16): chunks never straddle the last row of a plane
__device__ __forceinline__ int grid_floor(int v, int h)
{
    int r = (v - h) % CH;
    if (r < 0) r += CH;
    return v - r;
}

__device__ __forceinline__ Seg make_seg(long long item, int ya, int yb, int w, int h, int ns, const HostShifts& hs,
                                        const double* __restrict__ dshift)
{
    Seg g;
    g.k = (int)(item / ns);
    const int s = (int)(item - (long long)g.k * ns);
    const double sx = dshift ? -dshift[2 * g.k] : hs.s[g.k][0];
    const double sy = dshift ? -dshift[2 * g.k + 1] : hs.s[g.k][1];
    g.ax = make_axis(w, sx);
    g.ay = make_axis(h, sy);
    g.Xs = TW * s;
    g.Xe = min(g.Xs + TW, w);
    const int xs = g.Xs - V * HL + g.ax.m;                    // source column under the strip's first halo position
    g.r = xs & 3;                                             // two's complement: also right for negative xs
    g.xsrc0 = xs - g.r;
    const bool x_any = max(g.Xs, g.ax.lo) <= min(g.Xe - 1, g.ax.hi);
    g.ylo = max(ya, g.ay.lo);
    g.yhi = min(yb - 1, g.ay.hi);
    if (!x_any) { g.ylo = yb; g.yhi = yb - 1; }
    g.a0 = 0; g.nch = 0; g.kA = 0; g.kB = -1;
    g.pL = (g.xsrc0 < 0 && -g.xsrc0 <= BOXW - 1) ? -g.xsrc0 : -1;
    const int pr = (w - 1) - g.xsrc0;
    g.pR = (pr >= 0 && pr < BOXW - 1) ? pr : -1;
    if (g.ylo > g.yhi) return g;
    const int kA = g.ylo + g.ay.m, kB = g.yhi + g.ay.m;       // intervals [kA, kB], inside [0, h-2] (identity axis: [0, h-1])
    g.kA = kA; g.kB = kB;
    if (g.ay.ident) {                                         // pure row translation: rows [kA, kB] are copied
        g.a0 = grid_floor(kA, h);
        g.nch = (kB - g.a0) / CH + 1;
        return g;
    }
    int a0 = grid_floor(kA - 1 - CH, h);                      // >= 16 rows of causal warm-up before c'[kA - 1] ...
    if (a0 < CH) a0 = grid_floor(0, h);                       // ... or the exact start at row 0
    const int last = min(kB + 2, h - 1);                      // last row whose c' is evaluated
    const int jl = (last - a0) / CH;
    const bool jl_final = a0 + CH * (jl + 1) == h;
    g.a0 = a0;
    g.nch = jl_final ? jl + 1 : jl + 2;                       // + the look-ahead chunk that starts jl's sweep
    return g;
}

// ---- y pass: a thread owns CY adjacent columns.  CY = 2 (64-bit shared-memory and global accesses, half the load / store /
// address instructions per pixel) was MEASURED SLOWER than CY = 1: config 3 192 us against 153 us, config 5 3.81 ms against
// 3.10 ms -- the y phase then runs in 3.25 warps per CTA instead of 6.5 and its dependent chains are no longer hidden.
constexpr int CY = 1;
struct F2 { float x, y; };
template <int C> struct ValT { using type = float; };
template <> struct ValT<2> { using type = F2; };
using VT = ValT<CY>::type;

__device__ __forceinline__ float vfma(float s, float a, float b) { return fmaf(s, a, b); }
__device__ __forceinline__ F2 vfma(float s, F2 a, F2 b) { return F2{fmaf(s, a.x, b.x), fmaf(s, a.y, b.y)}; }
__device__ __forceinline__ float vmul(float s, float a) { return s * a; }
__device__ __forceinline__ F2 vmul(float s, F2 a) { return F2{s * a.x, s * a.y}; }
__device__ __forceinline__ float vext(float c0, float c1) { return fmaf(2.0f, c0, -c1); }            // 2 c0 - c1
__device__ __forceinline__ F2 vext(F2 c0, F2 c1) { return F2{fmaf(2.0f, c0.x, -c1.x), fmaf(2.0f, c0.y, -c1.y)}; }
__device__ __forceinline__ void vzero(float& v) { v = 0.f; }
__device__ __forceinline__ void vzero(F2& v) { v.x = 0.f; v.y = 0.f; }
__device__ __forceinline__ void vld(const float* p, float& v) { v = *p; }
__device__ __forceinline__ void vld(const float* p, F2& v) { const float2 t = *reinterpret_cast<const float2*>(p); v.x = t.x; v.y = t.y; }
__device__ __forceinline__ void vst(float* p, float v) { *p = v; }
__device__ __forceinline__ void vst(float* p, F2 v) { *reinterpret_cast<float2*>(p) = make_float2(v.x, v.y); }

// y-pass constants of one segment, per thread
struct YK {
    float na;            // -a
    float w0, w1, w2, w3;// the four weights times 6a
    int my, ylo, yhi;    // interval k -> output row k - my, stored when in [ylo, yhi]
    float* po;           // output plane + the thread's first column
    int w;
    bool in0, in1;       // CY = 2: which of the two columns lie in the x footprint (at least one does)
};

__device__ __forceinline__ void put(const YK& c, float* p, float v) { *p = v; }
__device__ __forceinline__ void put(const YK& c, float* p, F2 v)
{
    if (c.in0 && c.in1) *reinterpret_cast<float2*>(p) = make_float2(v.x, v.y);      // all but the two columns at a footprint edge
    else if (c.in0) p[0] = v.x;
    else p[1] = v.y;
}

// One output value = the 4 y taps.  FULL: the caller has established that every interval of the sweep is stored, and
// walks `ptr` down the rows itself (two integer instructions per value instead of the guard, the multiplication by the
// pitch and the 64-bit address of the general form: the store address arithmetic was 17 % of all instructions issued).
template <bool FULL>
__device__ __forceinline__ void emit(const YK& c, float*& ptr, int k, VT a0, VT a1, VT a2, VT a3)
{
    if (FULL) {
        put(c, ptr, vfma(c.w3, a3, vfma(c.w2, a2, vfma(c.w1, a1, vmul(c.w0, a0)))));
        ptr -= c.w;
    } else {
        const int y = k - c.my;
        if (y < c.ylo || y > c.yhi) return;          // block-uniform
        put(c, c.po + (size_t)((unsigned)y * (unsigned)c.w), vfma(c.w3, a3, vfma(c.w2, a2, vfma(c.w1, a1, vmul(c.w0, a0)))));
    }
}

// Anti-causal sweep of one chunk (rows a .. a+15 of the ring columns at Tc, row stride TW) with the 4 y taps.
//   REGULAR: cstart = c'[a+16] from the look-ahead of the chunk that follows; evaluates intervals a-2 .. a+13, the three
//            that reach into the chunk before with the values s1..s3 = c'[a-1], c'[a-2], c'[a-3] that chunk left.
//   FINAL:   the chunk ends with the last row of the plane: c'[h-1] is stored in the ring (exact end condition), the
//            virtual c'[h] = 2 c'[h-1] - c'[h-2]; evaluates up to interval h-2.
//   LOW:     rows below LOWROWS: elimination coefficients from the table, rows < -1 do not exist, row -1 is the virtual
//            c'[-1] = 2 c'[0] - c'[1].
template <bool LOW, bool FINAL, bool FULL>
__device__ __forceinline__ void sweep(const float* Tc, int a, VT cstart, const YK& yk, VT& s1, VT& s2, VT& s3)
{
    constexpr int ITOP = FINAL ? CH - 2 : CH - 1;
    constexpr int IEMIT = FINAL ? CH - 3 : CH - 4;          // first (highest) row of the sweep that completes an interval
    VT c0 = cstart, c1, c2, c3, n1, n2, n3;
    if (FINAL) vld(Tc + (CH - 1) * TW, c0);
    vzero(c1); vzero(c2); vzero(c3); vzero(n2); vzero(n3);
    n1 = c0;
    float* ptr = yk.po;
    if (FULL) ptr += (size_t)((unsigned)(a + IEMIT + 1 - yk.my) * (unsigned)yk.w);     // row of the highest interval
#pragma unroll
    for (int i = ITOP; i >= 0; --i) {
        const int row = a + i;
        VT cn;
        if (!LOW || row >= 0) {
            VT g;
            vld(Tc + i * TW, g);
            cn = LOW ? vfma(-c_low.u[row], c0, g) : vfma(yk.na, c0, g);
        } else if (row == -1) {
            cn = vext(c0, c1);
        } else {
            vzero(cn);
        }
        c3 = c2; c2 = c1; c1 = c0; c0 = cn;
        if (FINAL && i == CH - 2) c2 = vext(c1, c0);
        if (i == CH - 1) n1 = c0;
        if (i == CH - 2) n2 = c0;
        if (i == CH - 3) n3 = c0;
        if (i <= IEMIT) emit<FULL>(yk, ptr, row + 1, c0, c1, c2, c3);
    }
    if (LOW && a == 0) s1 = vext(c0, c1);                  // c'[-1] when row 0 opens the chunk
    emit<FULL>(yk, ptr, a, s1, c0, c1, c2);
    emit<FULL>(yk, ptr, a - 1, s2, s1, c0, c1);
    emit<FULL>(yk, ptr, a - 2, s3, s2, s1, c0);
    s1 = n1; s2 = n2; s3 = n3;
}

// block-uniform dispatch: FULL when every interval the sweep evaluates (a-2 .. top) is stored
template <bool LOW, bool FINAL>
__device__ __forceinline__ void sweep_any(const float* Tc, int a, VT cstart, const YK& yk, int kA, int kB, VT& s1, VT& s2,
                                          VT& s3)
{
    const int ktop = a + (FINAL ? CH - 2 : CH - 3);
    if (a - 2 >= kA && ktop <= kB) sweep<LOW, FINAL, true>(Tc, a, cstart, yk, s1, s2, s3);
    else sweep<LOW, FINAL, false>(Tc, a, cstart, yk, s1, s2, s3);
}

// Causal pass of one chunk in place (T -> g) and the look-ahead sum A = c'[a] seen from the chunk before.
template <bool LOW>
__device__ __forceinline__ VT causal(float* Tc, int a, bool is_final, float na, VT& gprev)
{
    constexpr PowTab PW = make_pow();
    const float inv6a = 1.0f / (6.0f * U_INF);
    VT A;
    vzero(A);
    float om = 1.f;
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        const int row = a + i;
        if (LOW && row < 0) continue;                       // block-uniform
        VT t, g;
        vld(Tc + i * TW, t);
        if (LOW) {
            const float u = c_low.u[row];
            g = vfma(-u, gprev, vmul(c_low.p[row], t));
            A = vfma(om, g, A);
            om *= -u;
        } else {
            g = vfma(na, gprev, t);
            A = vfma(PW.v[i], g, A);
        }
        gprev = g;
        vst(Tc + i * TW, (i == CH - 1 && is_final) ? vmul(inv6a, t) : g);     // last row of the plane: c'[h-1] = f[h-1] / 6a
    }
    return A;
}

// f[j] <- element j + R of (own 8 values, the next lane's 8 values): R register renames and R shuffles
template <int R>
__device__ __forceinline__ void shift_left(float (&f)[V])
{
    if (R == 0) return;
    float nx[R > 0 ? R : 1];
#pragma unroll
    for (int j = 0; j < R; ++j) nx[j] = __shfl_down_sync(0xffffffffu, f[j], 1);
#pragma unroll
    for (int j = 0; j + R < V; ++j) f[j] = f[j + R];
#pragma unroll
    for (int j = 0; j < R; ++j) f[V - R + j] = nx[j];
}

__device__ __forceinline__ void store_rows(float* t0, bool keep, const float (&f)[2][V])
{
    if (!keep) return;
    *reinterpret_cast<float4*>(t0) = make_float4(f[0][0], f[0][1], f[0][2], f[0][3]);
    *reinterpret_cast<float4*>(t0 + 4) = make_float4(f[0][4], f[0][5], f[0][6], f[0][7]);
    *reinterpret_cast<float4*>(t0 + TW) = make_float4(f[1][0], f[1][1], f[1][2], f[1][3]);
    *reinterpret_cast<float4*>(t0 + TW + 4) = make_float4(f[1][4], f[1][5], f[1][6], f[1][7]);
}

// The reflected halo of one staged row: positions left of image column 0 (at warp position pL) and right of column
// w-1 (at pR) get 2 f(edge) - f(mirror); 24 samples suffice (a^24 = 2e-14).  One warp, its own row.
__device__ __forceinline__ void x_reflect(float* buf, int pL, int pR, int lane)
{
    const int d = lane + 1;
    if (lane < V * HL) {
        if (pL >= 0) {
            const int p = pL - d, q = pL + d;
            if (p >= 0 && q < BOXW) buf[p] = fmaf(2.0f, buf[pL], -buf[q]);
        }
        if (pR >= 0) {
            const int p = pR + d, q = pR - d;
            if (p < BOXW && q >= 0) buf[p] = fmaf(2.0f, buf[pR], -buf[q]);
        }
    }
    __syncwarp();
}

// what the producer needs to know about a chunk
struct Box { int x, y, z; };

// enumerates, in order, the chunks of the units [u, u1) of one CTA
struct Walker {
    long long u, u1;
    int j, nch, x, a0, z;
    __device__ __forceinline__ bool next(Box& b, int w, int h, int ns, const HostShifts& hs, const double* __restrict__ dshift)
    {
        while (true) {
            if (j < nch) { b.x = x; b.y = a0 + CH * j; b.z = z; ++j; return true; }
            if (u >= u1) return false;
            const long long item = u / h;
            const int ya = (int)(u - item * h);
            const int len = (int)min((long long)(h - ya), u1 - u);
            const Seg g = make_seg(item, ya, ya + len, w, h, ns, hs, dshift);
            u += len;
            j = 0; nch = g.nch; x = g.xsrc0; a0 = g.a0; z = g.k;
        }
    }
};

}  // namespace rt

template <int NT>
__global__ void __launch_bounds__(rt::NTHR, NT == 2 ? 3 : 2)
k_resample_tile(const __grid_constant__ CUtensorMap tmap, int n, int w, int h, int ns, long long units, long long per_cta,
                const __grid_constant__ HostShifts hs, const double* __restrict__ dshift, float fill,
                float* __restrict__ out, int4* __restrict__ fp_dev)
{
    using namespace rt;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* stage = reinterpret_cast<float*>(smem_raw);                   // [NSTAGE][CH][BOXW]   TMA destinations (128-byte aligned)
    float* tring = stage + NSTAGE * STAGE_FLOATS;                        // [NT][CH][TW]         x-shifted rows / g
    uint64_t* full = reinterpret_cast<uint64_t*>(tring + NT * T_FLOATS); // [NSTAGE]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    for (int k = blockIdx.x * NTHR + tid; k < n && fp_dev; k += gridDim.x * NTHR) {
        const double sx = dshift ? -dshift[2 * k] : hs.s[k][0];
        const double sy = dshift ? -dshift[2 * k + 1] : hs.s[k][1];
        const Axis ax = make_axis(w, sx), ay = make_axis(h, sy);
        fp_dev[k] = make_int4(ax.lo, ax.hi, ay.lo, ay.hi);
    }
    if (tid == 0) {
        if (smem_u32(smem_raw) & 127u) __trap();                         // the TMA destinations must be 128-byte aligned
        for (int i = 0; i < NSTAGE; ++i) mbar_init(&full[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const long long u0 = (long long)blockIdx.x * per_cta, u1 = min(units, u0 + per_cta);
    if (u0 >= u1) return;

    // The last warp has no column in the y pass (208 columns = 6.5 warps): its first lane is the producer (NSTAGE chunks
    // ahead of the consumers), and the warp is the only one that polls an mbarrier; everybody else learns that a chunk
    // has landed from the block barrier that follows (256 polling threads cost issue slots the other CTAs could use).
    constexpr int PW = NTHR / 32 - 1;
    Walker wk;
    wk.u = u0; wk.u1 = u1; wk.j = 0; wk.nch = 0; wk.x = 0; wk.a0 = 0; wk.z = 0;
    int total = 0;                               // chunks of this CTA
    for (long long uu = u0; uu < u1;) {
        const long long item = uu / h;
        const int ya = (int)(uu - item * h);
        const int len = (int)min((long long)(h - ya), u1 - uu);
        total += make_seg(item, ya, ya + len, w, h, ns, hs, dshift).nch;
        uu += len;
    }
    if (warp == PW) {
        if (lane == 0) {
            for (int i = 0; i < NSTAGE; ++i) {
                Box b;
                if (!wk.next(b, w, h, ns, hs, dshift)) break;
                mbar_arrive_expect_tx(&full[i], STAGE_FLOATS * 4);
                tma_load_3d(stage + i * STAGE_FLOATS, &tmap, b.x, b.y, b.z, &full[i]);
            }
        }
        __syncwarp();
        if (total > 0) mbar_wait(&full[0], 0);
    }
    __syncthreads();
    int done = 0;                                // chunks consumed

    const size_t np = (size_t)w * h;
    int st = 0;                                  // stage of the next chunk and the parity of its mbarrier phase
    unsigned ph = 0;
    long long u = u0;
    while (u < u1) {
        const long long item = u / h;
        const int ya = (int)(u - item * h);
        const int len = (int)min((long long)(h - ya), u1 - u);
        const int yb = ya + len;
        u += len;
        const Seg sg = make_seg(item, ya, yb, w, h, ns, hs, dshift);
        float* outk = out + (size_t)sg.k * np;
        // rows of the segment without data: fill
        {
            const int cols = sg.Xe - sg.Xs;
            const int nlo = min(sg.ylo, yb) - ya;                        // rows [ya, ya + nlo)
            const int nhi = yb - max(sg.yhi + 1, ya);                    // rows [yb - nhi, yb)
            for (int r = warp; r < nlo + nhi; r += NTHR / 32) {
                const int y = r < nlo ? ya + r : yb - nhi + (r - nlo);
                float* dst = outk + (size_t)y * w + sg.Xs;
                for (int x = lane * 4; x < cols; x += 128)               // Xs, cols, w: multiples of 4
                    *reinterpret_cast<float4*>(dst + x) = make_float4(fill, fill, fill, fill);
            }
        }
        if (sg.nch == 0) continue;

        // x-pass constants
        const float nax = sg.ax.ident ? 0.f : -U_INF;
        const float nax2 = nax * nax, nax4 = nax2 * nax2, nax8 = nax4 * nax4;
        const float scx = sg.ax.ident ? 1.f : 6.0f * U_INF;
        const float wx[4] = {scx * sg.ax.w[0], scx * sg.ax.w[1], scx * sg.ax.w[2], scx * sg.ax.w[3]};
        const bool edge = sg.pL >= 0 || sg.pR >= 0;
        // y-pass constants of this thread's CY columns
        const int col = sg.Xs + CY * tid;
        bool ycol = CY * tid < TW && col < sg.Xe;           // Xe - Xs is a multiple of 4: a pair never straddles the strip's end
        YK yk;
        yk.na = -U_INF;
        const float scy = sg.ay.ident ? 1.f : 6.0f * U_INF;
        yk.w0 = scy * sg.ay.w[0]; yk.w1 = scy * sg.ay.w[1]; yk.w2 = scy * sg.ay.w[2]; yk.w3 = scy * sg.ay.w[3];
        yk.my = sg.ay.m; yk.ylo = sg.ylo; yk.yhi = sg.yhi;
        yk.po = outk + (ycol ? col : sg.Xs);
        yk.w = w;
        yk.in0 = col >= sg.ax.lo && col <= sg.ax.hi;
        yk.in1 = CY == 2 ? (col + 1 >= sg.ax.lo && col + 1 <= sg.ax.hi) : yk.in0;
        if (ycol && !(yk.in0 && yk.in1)) {
            // columns outside the x footprint: fill, for every row of the segment that carries data
            for (int y = sg.ylo; y <= sg.yhi; ++y) {
                float* q = yk.po + (size_t)((unsigned)y * (unsigned)w);
                if (!yk.in0) q[0] = fill;
                if (CY == 2 && !yk.in1) q[1] = fill;
            }
            if (!yk.in0 && !yk.in1) ycol = false;            // nothing else to do for this thread
        }
        VT gprev, s1, s2, s3;
        vzero(gprev); vzero(s1); vzero(s2); vzero(s3);

        for (int j = 0; j < sg.nch; ++j) {
            const int a = sg.a0 + CH * j;                               // first source row of the chunk
            float* T = tring + (j % NT) * T_FLOATS;      // (the chunk's box has landed: see the end of the iteration before)
            // ---------------- x pass: warp = rows 2 warp, 2 warp + 1
            {
                const int i0 = 2 * warp;
                if (a + i0 + 1 >= 0) {                                  // rows above the plane are never read again
                    float* b0 = stage + st * STAGE_FLOATS + i0 * BOXW;
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
                    float* t0 = T + i0 * TW + V * (lane - HL);
                    const bool keep = lane >= HL && lane < 32 - HL;
                    switch (sg.r) {          // warp-uniform: the outputs move r positions left (each case stores by itself:
                                             // a common store after the switch would cost 16 register moves per pair of rows)
                        case 0: store_rows(t0, keep, f); break;
                        case 1: shift_left<1>(f[0]); shift_left<1>(f[1]); store_rows(t0, keep, f); break;
                        case 2: shift_left<2>(f[0]); shift_left<2>(f[1]); store_rows(t0, keep, f); break;
                        default: shift_left<3>(f[0]); shift_left<3>(f[1]); store_rows(t0, keep, f); break;
                    }
                }
            }
            __syncthreads();                    // the chunk's x-shifted rows are complete; its stage is free again
            if (warp == PW) {
                if (lane == 0) {
                    Box b;
                    if (wk.next(b, w, h, ns, hs, dshift)) {
                        mbar_arrive_expect_tx(&full[st], STAGE_FLOATS * 4);
                        tma_load_3d(stage + st * STAGE_FLOATS, &tmap, b.x, b.y, b.z, &full[st]);
                    }
                }
                __syncwarp();
                if (done + 1 < total) {             // wait for the next chunk while the other warps run the y pass
                    const int nst = st + 1 == NSTAGE ? 0 : st + 1;
                    mbar_wait(&full[nst], nst == 0 ? ph ^ 1u : ph);
                }
            }
            // ---------------- y pass: thread = column
            if (ycol) {
                float* Tc = T + CY * tid;
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
                        const float* Tp = tring + ((j - 1) % NT) * T_FLOATS + CY * tid;
                        if (a - CH <= CH) sweep_any<true, false>(Tp, a - CH, A, yk, sg.kA, sg.kB, s1, s2, s3);
                        else sweep_any<false, false>(Tp, a - CH, A, yk, sg.kA, sg.kB, s1, s2, s3);
                    }
                    if (is_final && a + CH - 1 >= sg.kA - 1) sweep_any<false, true>(Tc, a, A, yk, sg.kA, sg.kB, s1, s2, s3);
                }
            }
            __syncthreads();                    // the next chunk has landed (seen by the last warp); with NT == 2 also: the
                                                // ring slot of chunk j-1 is written again by the x pass of chunk j+1
            ++done;
            if (++st == NSTAGE) { st = 0; ph ^= 1u; }
        }
    }
}

namespace rt {

inline bool tile_route(int w, int h) { return (w % 4 == 0) && w >= MIN_W && h >= MIN_H; }

constexpr int TILE_NT = 2;

inline int launch_resample_tile(const float* in, int n, int w, int h, const HostShifts& hs, const double* dshift_dev,
                                float fill, float* out, int4* fpd, cudaStream_t st)
{
    CUtensorMap tm;
    const cuuint64_t dims[3] = {(cuuint64_t)w, (cuuint64_t)h, (cuuint64_t)n};
    const cuuint64_t strides[2] = {(cuuint64_t)w * 4, (cuuint64_t)w * (cuuint64_t)h * 4};
    const cuuint32_t box[3] = {BOXW, CH, 1};
    if (!tma::encode_f32_map(&tm, in, 3, dims, strides, box)) { set_cuda_error(cudaErrorInvalidValue); return MRED_ECUDA; }
    constexpr size_t smem = smem_bytes<TILE_NT>();
    static PerDeviceOnce once;
    static std::atomic<int> occ_cache[64];
    int dev;
    if (once.pending(dev)) {
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample_tile<TILE_NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        MRED_CUDA_TRY(cudaFuncSetAttribute(k_resample_tile<TILE_NT>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        int occ = 1;
        MRED_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_resample_tile<TILE_NT>, NTHR, smem));
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
    k_resample_tile<TILE_NT><<<dim3((unsigned)ctas), NTHR, smem, st>>>(tm, n, w, h, ns, units, per, hs, dshift_dev, fill, out, fpd);
    MRED_LAUNCH_CHECK();
    return MRED_OK;
}

}  // namespace rt
}  // namespace mred
