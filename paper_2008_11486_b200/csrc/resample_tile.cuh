// resample_tile.cuh -- the per-row and per-column code of the CTA-tiled, TMA-staged spline-shift kernel (the route for
// planes with 16-byte-aligned rows, w >= 256, h >= 64: every configured detector format): segments, the x pass of a staged
// row pair, the causal pass and the anti-causal sweep of a column.  The kernel that runs them (k_resample_pipe, a
// warp-specialised pipeline) is in resample_pipe.cuh.  Mathematics: resample.cu; O5 (PAPER.md L63, L107, L164,
// L266).
//
// A pipeline owns a run of (frame, strip of 208 output columns, output rows [ya, yb)) segments; the runs are an even split
// of all n * strips * h strip-rows over the resident pipelines, so no wave is left half empty.  It walks a segment in
// chunks of 16 source rows:
//   TMA      one cp.async.bulk.tensor box of 256 columns x 16 rows per chunk, completion on an mbarrier.  Columns / rows
//            outside the plane arrive as zeros.  The box must start on a 16-byte boundary (an unaligned inner coordinate
//            raises an illegal-instruction fault on sm_100a), so it starts r = 0..3 columns left of the source column the
//            strip needs; the x pass works at the box's alignment and moves its OUTPUT r columns (r register renames + r
//            shuffles per row, a warp-uniform switch over r).
//   x pass   warp = 2 rows of the chunk out of shared memory, lane = 8 consecutive samples: the constant-coefficient
//            causal / anti-causal recursions inside the lane, lane-to-lane carries by shuffle (rs::x_pass), the 4 x taps;
//            the 208 kept columns go to a shared-memory ring.  Strips that touch an image edge first write the
//            point-reflected halo (f(-i) = 2 f(0) - f(i)) into the staged rows.
//   y pass   thread = one column, streaming down the chunks: causal recursion in place in the ring, the look-ahead sum that
//            starts the anti-causal sweep of the chunk before (16 rows: a^16 = 7e-10), the sweep with the 4 y taps, one
//            coalesced 128-byte store per warp and row.  The first rows of a plane use the EXACT elimination coefficients
//            of the natural-spline system (u_0 = 0, u_i = 1 / (4 - u_{i-1}), c_0 = f_0) and the last row c_{h-1} = f_{h-1},
//            with the virtual c_{-1} = 2 c_0 - c_1, c_h = 2 c_{h-1} - c_{h-2}: no rows beyond the plane are ever needed.
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
constexpr int LOWROWS = 32;             // rows whose elimination coefficients differ from their limit a (to float32: ~12)
constexpr int STAGE_FLOATS = CH * BOXW; // 16 KB
constexpr int T_FLOATS = CH * TW;       // 13 KB
constexpr int MIN_W = BOXW, MIN_H = 64; // smaller planes take the warp kernels of resample_warp.cuh

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
// PITCH > 0: the row pitch of the output plane (floats) is known at compile time, so the stores of a FULL sweep take
// immediate offsets from one base register (no pointer chain, whose updates wait for the stores in flight to have read
// their address); PITCH == 0: the pitch is c.w.
template <bool FULL, int PITCH = 0>
__device__ __forceinline__ void emit(const YK& c, float*& ptr, int k, VT a0, VT a1, VT a2, VT a3)
{
    if (FULL) {
        put(c, ptr, vfma(c.w3, a3, vfma(c.w2, a2, vfma(c.w1, a1, vmul(c.w0, a0)))));
        ptr -= PITCH > 0 ? PITCH : c.w;
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
template <bool LOW, bool FINAL, bool FULL, int PITCH = 0>
__device__ __forceinline__ void sweep(const float* Tc, int a, VT cstart, const YK& yk, VT& s1, VT& s2, VT& s3)
{
    constexpr int ITOP = FINAL ? CH - 2 : CH - 1;
    constexpr int IEMIT = FINAL ? CH - 3 : CH - 4;          // first (highest) row of the sweep that completes an interval
    VT c0 = cstart, c1, c2, c3, n1, n2, n3;
    if (FINAL) vld(Tc + (CH - 1) * TW, c0);
    vzero(c1); vzero(c2); vzero(c3); vzero(n2); vzero(n3);
    n1 = c0;
    float* ptr = yk.po;
    if (FULL) ptr += (size_t)((unsigned)(a + IEMIT + 1 - yk.my) * (unsigned)(PITCH > 0 ? PITCH : yk.w));     // row of the highest interval
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
        if (i <= IEMIT) emit<FULL, PITCH>(yk, ptr, row + 1, c0, c1, c2, c3);
    }
    if (LOW && a == 0) s1 = vext(c0, c1);                  // c'[-1] when row 0 opens the chunk
    emit<FULL, PITCH>(yk, ptr, a, s1, c0, c1, c2);
    emit<FULL, PITCH>(yk, ptr, a - 1, s2, s1, c0, c1);
    emit<FULL, PITCH>(yk, ptr, a - 2, s3, s2, s1, c0);
    s1 = n1; s2 = n2; s3 = n3;
}

// block-uniform dispatch: FULL when every interval the sweep evaluates (a-2 .. top) is stored
template <bool LOW, bool FINAL, int PITCH = 0>
__device__ __forceinline__ void sweep_any(const float* Tc, int a, VT cstart, const YK& yk, int kA, int kB, VT& s1, VT& s2,
                                          VT& s3)
{
    const int ktop = a + (FINAL ? CH - 2 : CH - 3);
    if (a - 2 >= kA && ktop <= kB) sweep<LOW, FINAL, true, PITCH>(Tc, a, cstart, yk, s1, s2, s3);
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

namespace rt {

inline bool tile_route(int w, int h) { return (w % 4 == 0) && w >= MIN_W && h >= MIN_H; }

}  // namespace rt
}  // namespace mred
