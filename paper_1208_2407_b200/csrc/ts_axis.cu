// ts_axis.cu -- axis-split evolution for steps WITHOUT a potential (a flat potential
// drops the diagonal factor; the step is then the four kinetic parts only).
//
// A horizontal sweep acts inside rows, a vertical sweep along columns, both with scalar
// coefficients, so every X sweep commutes with every Y sweep (tensor-product structure; pinned on
// the oracle by test_xy_regrouping and on dense matrices by test_stage_order...).  A chain of n
// second-order sub-steps therefore factorises EXACTLY,
//
//     U2(c_{n-1}) ... U2(c_0)  =  [X-chain along every row]  (x)  [Y-chain along every column],
//     axis chain = E(h_0) O(f_0) E(h_0 + h_1) O(f_1) ... O(f_{n-1}) E(h_{n-1}),
//
// E / O = even / odd pair sweep along the axis, h = half angle, f = full angle (adjacent half
// sweeps of chained sub-steps merged).  Only the rounding differs from the literal stage order.
// The two chains are independent 1-D problems, and each gets the decomposition that suits it:
//
//   line_kernel   a warp holds a WHOLE line (row or column) of up to 32 * NS sites in registers,
//                 NS consecutive sites per lane, and applies the complete chain -- all n sub-steps
//                 -- in one launch: in-thread pairs are plain FMAs, one pair per lane and odd sweep
//                 crosses lanes by shuffle.  No halo, no pass structure, no shared memory; the
//                 state is read once and written once.  Longer ROWS are cut into windows of
//                 32 * NS sites with a halo of 2 sites per sub-step and side that is recomputed
//                 and discarded, n <= 16 sub-steps per pass, rows prefetched into a
//                 second register set.
//   ycol_kernel   long COLUMNS: the streaming register pipeline of ts_stream.cu reduced to its
//                 vertical sweeps -- a warp walks down a strip of 64 columns, two sites per lane,
//                 S <= 16 chained sub-steps in flight, rows brought in by bulk async copies (TMA)
//                 into a per-warp shared-memory ring.  No x halo at all.
//
// Against the fused 2-D kernel (128-site strips with a 2S halo in x AND the y pipeline in the same
// registers) the split removes the x-halo recomputation (1.23x at S = 6) and lets a pass chain
// twice as many sub-steps, at the price of two passes over HBM instead of one.
#include <math.h>

#include <atomic>
#include <type_traits>

#include "ts_internal.h"
#include "ts_rows.cuh"
#include "ts_tma.cuh"

namespace ts {
namespace {

using namespace tma;

constexpr int kMaxPeriod = 8;     // longest pattern of distinct sub-steps (ts_evolve 1, ts_evolve_u4 5)
constexpr int kMaxChain = 16;     // sub-steps per windowed / pipelined pass

// ---------------------------------------------------------------------------------------------
// line kernel
// ---------------------------------------------------------------------------------------------
template <typename T>
struct LineParams {
    const T* src_re;
    const T* src_im;
    T* dst_re;
    T* dst_im;
    int64_t line_stride;    // elements between consecutive lines
    int64_t site_stride;    // elements between consecutive sites of a line (1: rows)
    int n_lines, n_sites;
    int n_lanes;            // lanes that hold sites (resident lines shorter than 32 * NS)
    int n_win, wi, halo;    // windows per line (1: the whole line is resident), interior, halo
    int lines_per_warp;
    int periodic;
    int64_t n_sub;          // sub-steps of this pass
    int period, phase0;     // pattern of distinct sub-steps; index of this pass's first sub-step
    int resc_every;         // deferred cosines are multiplied in every resc_every sub-steps ...
    T resc;                 // ... by this factor (keeps the scaled amplitudes in range)
    T final_scale;          // the rest of the deferred cosines, applied at the store
    T te_first, te_last;    // tangents: opening and closing even half sweep
    T te_mid[kMaxPeriod];   // even sweep merged from entry k's closing and entry k+1's opening half
    T to[kMaxPeriod];       // odd sweep of pattern entry k
    T sec_o[kMaxPeriod];    // 1 / cos of it (unpaired sites at closed ends)
};

template <typename T, int NS>
struct Line {
    T re[NS];
    T im[NS];
};

template <typename T, int NS>
__device__ __forceinline__ void line_even(Line<T, NS>& L, T t) {
#pragma unroll
    for (int k = 0; k < NS; k += 2) rows::rot(L.re[k], L.im[k], L.re[k + 1], L.im[k + 1], t);
}
#ifndef TS_SCALAR_F32
template <int NS>
__device__ __forceinline__ void line_even(Line<float, NS>& L, float t) {
#pragma unroll
    for (int k = 0; k < NS; k += 2) {
        float nr0, nr1, ni0, ni1;
        rows::fma2(nr0, nr1, -t, L.im[k + 1], L.im[k], L.re[k], L.re[k + 1]);
        rows::fma2(ni0, ni1, t, L.re[k + 1], L.re[k], L.im[k], L.im[k + 1]);
        L.re[k] = nr0; L.re[k + 1] = nr1; L.im[k] = ni0; L.im[k + 1] = ni1;
    }
}
#endif

// odd sweep: pairs (1,2), (3,4), ... in-thread; (NS-1, 0 of the next lane) by shuffle, both lanes
// computing their own side.  EDGE: the cross-lane pair may be cut (closed end, ghost lanes): the
// coupling is then 0 and the unpaired real site takes 1/cos instead (ts_rows.cuh).
template <typename T, int NS, bool EDGE>
__device__ __forceinline__ void line_odd(Line<T, NS>& L, T t, T sec, int up_src, int dn_src,
                                         bool cut_up, bool cut_dn) {
    const T up_re = __shfl_sync(0xffffffffu, L.re[NS - 1], up_src);
    const T up_im = __shfl_sync(0xffffffffu, L.im[NS - 1], up_src);
    const T dn_re = __shfl_sync(0xffffffffu, L.re[0], dn_src);
    const T dn_im = __shfl_sync(0xffffffffu, L.im[0], dn_src);
#pragma unroll
    for (int k = 1; k + 1 < NS; k += 2) rows::rot(L.re[k], L.im[k], L.re[k + 1], L.im[k + 1], t);
    T r0 = L.re[0], i0 = L.im[0], r3 = L.re[NS - 1], i3 = L.im[NS - 1];
    T t_up = t, t_dn = t;
    if (EDGE) {
        const T c0 = cut_up ? sec : T(1), c3 = cut_dn ? sec : T(1);
        t_up = cut_up ? T(0) : t;
        t_dn = cut_dn ? T(0) : t;
        r0 *= c0; i0 *= c0; r3 *= c3; i3 *= c3;
    }
    L.re[0] = fma(-t_up, up_im, r0);
    L.im[0] = fma(t_up, up_re, i0);
    L.re[NS - 1] = fma(-t_dn, dn_im, r3);
    L.im[NS - 1] = fma(t_dn, dn_re, i3);
}

template <typename T, int NS>
__device__ __forceinline__ void line_scale(Line<T, NS>& L, T s) {
#pragma unroll
    for (int k = 0; k < NS; ++k) { L.re[k] *= s; L.im[k] *= s; }
}
#ifndef TS_SCALAR_F32
template <int NS>
__device__ __forceinline__ void line_scale(Line<float, NS>& L, float s) {
#pragma unroll
    for (int k = 0; k < NS; k += 2) {
        rows::mul2v(L.re[k], L.re[k + 1], L.re[k], L.re[k + 1], s, s);
        rows::mul2v(L.im[k], L.im[k + 1], L.im[k], L.im[k + 1], s, s);
    }
}
#endif

// 16-byte (or, for NS = 2 in fp32, 8-byte) pieces of a contiguous run
template <typename T>
struct Piece {
    static constexpr int n = 16 / sizeof(T);
};

__device__ __forceinline__ void ld_piece(const float* p, float* v, int n) {
    if (n == 4) {
        const float4 q = __ldg(reinterpret_cast<const float4*>(p));
        v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
    } else {
        const float2 q = __ldg(reinterpret_cast<const float2*>(p));
        v[0] = q.x; v[1] = q.y;
    }
}
__device__ __forceinline__ void ld_piece(const double* p, double* v, int) {
    const double2 q = __ldg(reinterpret_cast<const double2*>(p));
    v[0] = q.x; v[1] = q.y;
}
__device__ __forceinline__ void st_piece(float* p, const float* v, int n) {
    if (n == 4) *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    else *reinterpret_cast<float2*>(p) = make_float2(v[0], v[1]);
}
__device__ __forceinline__ void st_piece(double* p, const double* v, int) {
    *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
}

// COL = false: rows (site stride 1, vector accesses, 4 warps per block, each warp a window of a
// block of consecutive rows, the next row prefetched while the current one is computed);
// COL = true: columns (site stride = pitch, scalar accesses; the 8 warps of a block take 8
// adjacent columns at the same time, so that the 32-byte sectors they share are fetched once).
template <typename T, int NS, bool EDGE, bool COL>
__global__ void __launch_bounds__(COL ? 256 : 128, COL ? 1 : (sizeof(T) * NS >= 128 ? 2 : 4))
line_kernel(const __grid_constant__ LineParams<T> p) {
    constexpr int PW = (Piece<T>::n < NS) ? Piece<T>::n : NS;     // sites per vector access
    const int lane = threadIdx.x & 31;
    const int wpb = COL ? 8 : 4;
    const int wg = blockIdx.x * wpb + (threadIdx.x >> 5);
    int win, line0, line1;
    if (COL) {
        win = 0; line0 = wg; line1 = min(wg + 1, p.n_lines);
    } else {
        win = wg % p.n_win;
        line0 = (wg / p.n_win) * p.lines_per_warp;
        line1 = min(line0 + p.lines_per_warp, p.n_lines);
    }
    if (line0 >= p.n_lines) return;

    const int xs = win * p.wi - p.halo;          // first site of the window (may be < 0)
    const int xl = xs + NS * lane;               // first site of the lane
    const bool active = lane < p.n_lanes;
    // the ring of lanes that hold sites: a resident periodic line closes on itself; in a window
    // the wrap-around partners of lanes 0 / 31 only reach the halo, which is discarded
    const int up_src = lane == 0 ? p.n_lanes - 1 : lane - 1;
    const int dn_src = lane == p.n_lanes - 1 ? 0 : lane + 1;
    bool cut_up = false, cut_dn = false;
    if (EDGE) {
        // lanes beyond the line (ghosts: zeros that must stay zero) and, on a closed line, the
        // lanes on either side of each of its two ends
        const bool closed = !p.periodic;
        cut_up = !active || (closed && (xl == 0 || xl == p.n_sites));
        cut_dn = !active || (closed && (xl + NS == p.n_sites || xl + NS == 0));
    }
    // interior of the window: what this warp stores
    const int st_lo = win * p.wi;
    const int st_hi = min(st_lo + p.wi, p.n_sites);

    auto load = [&](int line, Line<T, NS>& L) {
        const int64_t base = (int64_t)line * p.line_stride;
        if (COL) {
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                const int64_t off = base + (int64_t)(xl + k) * p.site_stride;
                L.re[k] = active ? __ldg(p.src_re + off) : T(0);
                L.im[k] = active ? __ldg(p.src_im + off) : T(0);
            }
        } else {
#pragma unroll
            for (int k = 0; k < NS; k += PW) {
                int x = xl + k;
                bool ok = active;
                if (p.periodic) x = rows::wrap_index(x, p.n_sites);
                else ok = ok && x >= 0 && x < p.n_sites;
                if (ok) {
                    ld_piece(p.src_re + base + x, &L.re[k], PW);
                    ld_piece(p.src_im + base + x, &L.im[k], PW);
                } else {
#pragma unroll
                    for (int i = 0; i < PW; ++i) { L.re[k + i] = T(0); L.im[k + i] = T(0); }
                }
            }
        }
    };
    auto store = [&](int line, Line<T, NS>& L) {
        const int64_t base = (int64_t)line * p.line_stride;
        line_scale(L, p.final_scale);
        if (COL) {
            if (!active) return;
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                const int64_t off = base + (int64_t)(xl + k) * p.site_stride;
                p.dst_re[off] = L.re[k];
                p.dst_im[off] = L.im[k];
            }
        } else {
#pragma unroll
            for (int k = 0; k < NS; k += PW) {
                const int x = xl + k;
                if (active && x >= st_lo && x < st_hi) {
                    st_piece(p.dst_re + base + x, &L.re[k], PW);
                    st_piece(p.dst_im + base + x, &L.im[k], PW);
                }
            }
        }
    };
    // E(h_0) O(f_0) E(h_0 + h_1) ... O(f_{n-1}) E(h_{n-1}); pattern entry k = (phase0 + s) mod period
    auto chain = [&](Line<T, NS>& L) {
        line_even(L, p.te_first);
        int k = p.phase0, since = 0;
#pragma unroll 1
        for (int64_t s = 0; s < p.n_sub; ++s) {
            line_odd<T, NS, EDGE>(L, p.to[k], p.sec_o[k], up_src, dn_src, cut_up, cut_dn);
            line_even(L, s + 1 == p.n_sub ? p.te_last : p.te_mid[k]);
            if (++k == p.period) k = 0;
            if (++since == p.resc_every) { since = 0; line_scale(L, p.resc); }
        }
    };

    if (COL) {
        Line<T, NS> A;
        load(line0, A);
        chain(A);
        store(line0, A);
    } else {
        Line<T, NS> A, B;
        load(line0, A);
#pragma unroll 1
        for (int line = line0; line < line1; line += 2) {
            const bool two = line + 1 < line1;
            if (two) load(line + 1, B);
            chain(A);
            store(line, A);
            if (two) {
                if (line + 2 < line1) load(line + 2, A);
                chain(B);
                store(line + 1, B);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// column pipeline kernel
// ---------------------------------------------------------------------------------------------
constexpr int kYWarps = 4;
constexpr int kYCols = 64;        // columns per warp: 2 sites per lane

template <typename T>
struct YcolParams {
    const T* src_re;
    const T* src_im;
    T* dst_re;
    T* dst_im;
    int nx, ny;
    int n_strips, seg_rows, nst;
    int periodic_y;
    T te[kMaxChain + 1];     // even sweeps: opening half, S-1 merged, closing half
    T to[kMaxChain];         // odd sweep of sub-step j (the caller's full-angle coefficients)
    T sec_o[kMaxChain];
    T out_scale;
};

template <typename T>
struct Row2 {
    T re[2];
    T im[2];
};

template <typename T>
__device__ __forceinline__ void ypair2(Row2<T>& a, Row2<T>& b, T t) {
#pragma unroll
    for (int i = 0; i < 2; ++i) rows::rot(a.re[i], a.im[i], b.re[i], b.im[i], t);
}
#ifndef TS_SCALAR_F32
__device__ __forceinline__ void ypair2(Row2<float>& a, Row2<float>& b, float t) {
    float ar0, ar1, ai0, ai1, br0, br1, bi0, bi1;
    rows::fma2(ar0, ar1, -t, b.im[0], b.im[1], a.re[0], a.re[1]);
    rows::fma2(ai0, ai1, t, b.re[0], b.re[1], a.im[0], a.im[1]);
    rows::fma2(br0, br1, -t, a.im[0], a.im[1], b.re[0], b.re[1]);
    rows::fma2(bi0, bi1, t, a.re[0], a.re[1], b.im[0], b.im[1]);
    a.re[0] = ar0; a.re[1] = ar1; a.im[0] = ai0; a.im[1] = ai1;
    b.re[0] = br0; b.re[1] = br1; b.im[0] = bi0; b.im[1] = bi1;
}
#endif
template <typename T>
__device__ __forceinline__ void scale2(Row2<T>& r, T s) {
    r.re[0] *= s; r.re[1] *= s; r.im[0] *= s; r.im[1] *= s;
}
template <typename T>
__device__ __forceinline__ void zero2(Row2<T>& r) {
    r.re[0] = r.re[1] = r.im[0] = r.im[1] = T(0);
}

__device__ __forceinline__ void lds2(uint32_t addr, float (&v)[2]) {
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v[0]), "=f"(v[1]) : "r"(addr));
}
__device__ __forceinline__ void lds2(uint32_t addr, double (&v)[2]) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v[0]), "=d"(v[1]) : "r"(addr));
}
__device__ __forceinline__ void st2(float* p, const float (&v)[2], float s) {
    float a, b;
    rows::mul2v(a, b, v[0], v[1], s, s);
    *reinterpret_cast<float2*>(p) = make_float2(a, b);
}
__device__ __forceinline__ void st2(double* p, const double (&v)[2], double s) {
    *reinterpret_cast<double2*>(p) = make_double2(v[0] * s, v[1] * s);
}

// stages 0..S-1 of one iteration.  Stage J holds the row pair that still waits for its odd
// partner below; the incoming pair (x0, x1) = rows (y - 2J, y - 2J + 1) gets the even sweep that
// opens sub-step J (merged with the one that closed sub-step J-1), then the odd sweep couples
// the waiting pair's lower row with x0, and the waiting pair moves on to stage J+1.
template <typename T, int S, bool EDGE, int J>
struct YStages {
    static __device__ __forceinline__ void run(const YcolParams<T>& p, int y, Row2<T> (&W)[S][2][2],
                                               const int u, Row2<T>& x0, Row2<T>& x1) {
        Row2<T>& a0 = W[J][u][0];
        Row2<T>& a1 = W[J][u][1];
        Row2<T>& g = W[J][u ^ 1][0];
        Row2<T>& h = W[J][u ^ 1][1];
        a0 = x0; a1 = x1;
        ypair2(a0, a1, p.te[J]);
        const int yj = y - 2 * J;
        // closed lattice: the odd pair (yj-1, yj) does not exist at yj = 0 and yj = ny; the ghost
        // row is zero and stays zero, the real row takes 1/cos of the omitted sweep
        const bool yedge = EDGE && (yj == 0 || yj == p.ny);
        const T t_yo = yedge ? T(0) : p.to[J];
        ypair2(h, a0, t_yo);
        if (EDGE) { const T sy = yedge ? p.sec_o[J] : T(1); scale2(h, sy); scale2(a0, sy); }
        if (J == S - 1) ypair2(g, h, p.te[S]);
        x0 = g; x1 = h;
        if constexpr (J + 1 < S) YStages<T, S, EDGE, J + 1>::run(p, y, W, u, x0, x1);
    }
};

// resident blocks per SM the register budget of the pipeline allows: S+1 row pairs + the incoming
// pair, 4 (fp32) / 8 (fp64) registers per row, ~56 for addresses, counters and temporaries
template <typename T, int S>
constexpr int ycol_min_blocks() {
    constexpr int est = ((S + 1) * 8 + 8) * (int)(sizeof(T) / 4) + 56;
    return est <= 128 ? 4 : est <= 168 ? 3 : 2;
}

template <typename T, int S, bool PERY>
__global__ void __launch_bounds__(kYWarps * 32, ycol_min_blocks<T, S>())
ycol_kernel(const YcolParams<T> p) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr uint32_t ROWB = kYCols * sizeof(T);
    constexpr uint32_t SLOTB = 4 * ROWB;          // re0 im0 re1 im1

    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int strip = blockIdx.x * kYWarps + warp;
    if (strip >= p.n_strips) return;
    const int NST = p.nst;
    const int DIST = NST - 1;
    const int x0c = strip * kYCols;
    const int cols = min(kYCols, p.nx - x0c);
    const uint32_t bytes = cols * sizeof(T);
    const bool lane_ok = 2 * lane < cols;
    const uint32_t ring = smem_u32(smem_raw) + warp * NST * SLOTB;
    const uint32_t bars = smem_u32(smem_raw) + kYWarps * NST * SLOTB + warp * NST * 8;
    const uint32_t lane_off = lane * 2 * sizeof(T);

    const int y_out0 = blockIdx.y * p.seg_rows;
    const int y_out1 = min(y_out0 + p.seg_rows, p.ny);
    const int y_in0 = y_out0 - 2 * S;
    const int n_iter = ((y_out1 - y_out0) / 2 + 2 * S + 1) & ~1;

    const bool leader = elect_one();
    if (leader) {
        for (int s = 0; s < NST; ++s) mbar_init(bars + 8 * s, 1);
        mbar_fence_init();
    }
    __syncwarp();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;");

    // running fetch position (warp-uniform): rows (fy, fy+1) of the strip's columns
    int fy = PERY ? rows::wrap_index(y_in0, p.ny) : y_in0;
    const int64_t pitchB = (int64_t)p.nx * sizeof(T);
    const int64_t planeB = pitchB * p.ny;
    const char* f_re = reinterpret_cast<const char*>(p.src_re + x0c) + (int64_t)fy * pitchB;
    const char* f_im = reinterpret_cast<const char*>(p.src_im + x0c) + (int64_t)fy * pitchB;
    uint32_t f_dst = ring, f_bar = bars;
    int f_slot = 0;
    auto issue = [&]() {
        const bool rowok = PERY || (fy >= 0 && fy < p.ny);
        if (leader) {
            if (rowok) {
                mbar_arrive_expect_tx(f_bar, 4 * bytes);
                bulk_g2s(f_dst, f_re, bytes, f_bar);
                bulk_g2s(f_dst + ROWB, f_im, bytes, f_bar);
                bulk_g2s(f_dst + 2 * ROWB, f_re + pitchB, bytes, f_bar);
                bulk_g2s(f_dst + 3 * ROWB, f_im + pitchB, bytes, f_bar);
            } else {
                mbar_arrive(f_bar);
            }
        }
        fy += 2; f_re += 2 * pitchB; f_im += 2 * pitchB;
        if (PERY && fy >= p.ny) { fy -= p.ny; f_re -= planeB; f_im -= planeB; }
        f_dst += SLOTB; f_bar += 8;
        if (++f_slot == NST) { f_slot = 0; f_dst = ring; f_bar = bars; }
    };
    for (int k = 0; k < DIST; ++k)
        if (k < n_iter) issue();

    auto run = [&](auto edge_tag) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        Row2<T> W[S][2][2];
#pragma unroll
        for (int s = 0; s < S; ++s) { zero2(W[s][0][0]); zero2(W[s][0][1]); zero2(W[s][1][0]); zero2(W[s][1][1]); }
        uint32_t c_src = ring + lane_off, c_bar = bars, cph = 0;
        int c_slot = 0;
        int y = y_in0;
        T* o_re = p.dst_re + (int64_t)(y_in0 - 2 * S) * p.nx + x0c + 2 * lane;
        T* o_im = p.dst_im + (int64_t)(y_in0 - 2 * S) * p.nx + x0c + 2 * lane;
#pragma unroll 1
        for (int it0 = 0; it0 < n_iter; it0 += 2) {
            auto half = [&](auto utag) {
                constexpr int U = decltype(utag)::value;
                const int it = it0 + U;
                __syncwarp();      // every lane is done with the slot about to be refilled
                if (it + DIST < n_iter) issue();
                mbar_wait(c_bar, cph);
                Row2<T> x0, x1;
                const bool rowok = !EDGE || (y >= 0 && y < p.ny);
                if (rowok) {
                    lds2(c_src, x0.re);
                    lds2(c_src + ROWB, x0.im);
                    lds2(c_src + 2 * ROWB, x1.re);
                    lds2(c_src + 3 * ROWB, x1.im);
                } else {
                    zero2(x0); zero2(x1);
                }
                YStages<T, S, EDGE, 0>::run(p, y, W, U, x0, x1);
                if (it >= 2 * S && lane_ok && y - 2 * S < y_out1) {
                    st2(o_re, x0.re, p.out_scale);
                    st2(o_im, x0.im, p.out_scale);
                    st2(o_re + p.nx, x1.re, p.out_scale);
                    st2(o_im + p.nx, x1.im, p.out_scale);
                }
                y += 2; o_re += 2 * (int64_t)p.nx; o_im += 2 * (int64_t)p.nx;
                c_src += SLOTB; c_bar += 8;
                if (++c_slot == NST) { c_slot = 0; c_src = ring + lane_off; c_bar = bars; cph ^= 1; }
            };
            half(std::integral_constant<int, 0>{});
            half(std::integral_constant<int, 1>{});
        }
    };
    const bool edge = !PERY && (y_in0 < 0 || y_in0 + 2 * n_iter >= p.ny);
    if (edge) run(std::true_type{});
    else run(std::false_type{});
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
struct Angle {          // cos, sin
    double c, s;
};
Angle add(const Angle& a, const Angle& b) { return {a.c * b.c - a.s * b.s, a.s * b.c + a.c * b.s}; }

// half / odd angle of sub-step c along the axis: rows compose the odd sweep from the two half
// sweeps the regrouping brings together, columns use the caller's full-angle coefficients (the
// "full middle sweep", include/ts.h) -- as in ts_stream.cu
Angle half_of(const StepCoef& c) { return {c.a_h, c.b_h}; }
Angle odd_of(const StepCoef& c, bool col) {
    if (col) return {c.a_f, c.b_f};
    return add(half_of(c), half_of(c));
}

// resident lines: the smallest NS (sites per lane) with n = NS * lanes, lanes <= 32
int line_sites_per_lane(int64_t n, int dtype, bool col) {
    const int cand32[] = {2, 4, 8, 16, 32};
    const int cand64[] = {2, 4, 8, 16};
    const int* cand = dtype == TS_F32 ? cand32 : cand64;
    const int nc = dtype == TS_F32 ? 5 : 4;
    for (int i = 0; i < nc; ++i) {
        const int ns = cand[i];
        // rows are read with 16-byte accesses (8-byte for NS = 2 in fp32)
        if (n % ns == 0 && n / ns <= 32 && n / ns >= 1) return ns;
        (void)col;
    }
    return 0;
}

template <typename T, int NS, bool EDGE, bool COL>
int launch_line(const LineParams<T>& p, cudaStream_t st) {
    const int wpb = COL ? 8 : 4;
    int64_t warps;
    if (COL) warps = p.n_lines;
    else warps = (int64_t)p.n_win * ((p.n_lines + p.lines_per_warp - 1) / p.lines_per_warp);
    const int64_t blocks = (warps + wpb - 1) / wpb;
    line_kernel<T, NS, EDGE, COL><<<(unsigned)blocks, wpb * 32, 0, st>>>(p);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}

template <typename T, int NS>
int launch_line_ns(const LineParams<T>& p, bool edge, bool col, cudaStream_t st) {
    if (col) return edge ? launch_line<T, NS, true, true>(p, st) : launch_line<T, NS, false, true>(p, st);
    return edge ? launch_line<T, NS, true, false>(p, st) : launch_line<T, NS, false, false>(p, st);
}

template <typename T>
int launch_line_t(const LineParams<T>& p, int ns, bool edge, bool col, cudaStream_t st) {
    switch (ns) {
        case 2: return launch_line_ns<T, 2>(p, edge, col, st);
        case 4: return launch_line_ns<T, 4>(p, edge, col, st);
        case 8: return launch_line_ns<T, 8>(p, edge, col, st);
        case 16: return launch_line_ns<T, 16>(p, edge, col, st);
        case 32:
            if constexpr (sizeof(T) == 4) return launch_line_ns<T, 32>(p, edge, col, st);
    }
    set_error("axis: no line kernel for this extent");
    return TS_EUNSUPPORTED;
}

// One launch of the line kernel: sub-steps [first, first + n_sub) of the periodic pattern along
// rows (col = false) or columns.  windowed: rows longer than one window, n_sub <= kMaxChain.
template <typename T>
int line_pass(const LatticeDesc& L, const T* src_re, const T* src_im, T* dst_re, T* dst_im,
              const StepCoef* pat, int period, int64_t first, int64_t n_sub, bool col,
              bool windowed, cudaStream_t st) {
    LineParams<T> p;
    p.src_re = src_re; p.src_im = src_im; p.dst_re = dst_re; p.dst_im = dst_im;
    const int64_t n = col ? L.ny : L.nx;
    const bool periodic = col ? L.periodic_y : L.periodic_x;
    p.n_lines = (int)(col ? L.nx : L.ny);
    p.n_sites = (int)n;
    p.line_stride = col ? 1 : L.nx;
    p.site_stride = col ? L.nx : 1;
    p.periodic = periodic;
    int ns;
    if (windowed) {
        ns = L.dtype == TS_F32 ? 32 : 16;
        p.n_lanes = 32;
        // the halo: 2 sites per sub-step; lane-aligned on a closed line so that its ends fall
        // between two lanes
        int halo = (int)((2 * n_sub + 3) / 4 * 4);
        if (!periodic) halo = (halo + ns - 1) / ns * ns;
        p.halo = halo;
        p.wi = 32 * ns - 2 * halo;
        p.n_win = (int)((n + p.wi - 1) / p.wi);
        // about two waves of warps (148 SMs x 12), at least 8 rows per warp
        int64_t lpw = ((int64_t)p.n_lines * p.n_win + 2 * 148 * 12 - 1) / (2 * 148 * 12);
        if (lpw < 8) lpw = 8;
        p.lines_per_warp = (int)lpw;
    } else {
        ns = line_sites_per_lane(n, L.dtype, col);
        if (!ns) { set_error("axis: line does not fit a warp"); return TS_EUNSUPPORTED; }
        p.n_lanes = (int)(n / ns);
        p.halo = 0; p.wi = (int)n; p.n_win = 1;
        int64_t lpw = ((int64_t)p.n_lines + 148 * 12 - 1) / (148 * 12);
        p.lines_per_warp = (int)(lpw < 1 ? 1 : lpw);
    }
    p.n_sub = n_sub;
    p.period = period;
    p.phase0 = (int)(first % period);
    // tangents, deferred cosines (all in double, rounded once)
    const StepCoef& c_first = pat[first % period];
    const StepCoef& c_last = pat[(first + n_sub - 1) % period];
    p.te_first = (T)(c_first.b_h / c_first.a_h);
    p.te_last = (T)(c_last.b_h / c_last.a_h);
    double log_period = 0.0;       // log of the deferred cosines of one pattern period (odd + merged even)
    for (int k = 0; k < kMaxPeriod; ++k) {
        if (k < period) {
            const Angle m = add(half_of(pat[k]), half_of(pat[(k + 1) % period]));
            const Angle o = odd_of(pat[k], col);
            p.te_mid[k] = (T)(m.s / m.c);
            p.to[k] = (T)(o.s / o.c);
            p.sec_o[k] = (T)(1.0 / o.c);
            log_period += log(m.c) + log(o.c);
        } else {
            p.te_mid[k] = T(0); p.to[k] = T(0); p.sec_o[k] = T(1);
        }
    }
    // total: cos(opening half) * prod over sub-steps of cos(odd) * cos(following even sweep); the
    // last even sweep is the closing half sweep, not a merged one.  Pattern entry k occurs
    // cnt[k] times among the n_sub sub-steps (n_sub may be millions: no loop over them).
    double log_total = log(c_first.a_h) + log(c_last.a_h);
    const int k_last = (int)((first + n_sub - 1) % period);
    for (int k = 0; k < period; ++k) {
        const int64_t r = ((k - first) % period + period) % period;     // first s with entry k
        const int64_t cnt = r < n_sub ? (n_sub - r + period - 1) / period : 0;
        const Angle m = add(half_of(pat[k]), half_of(pat[(k + 1) % period]));
        const Angle o = odd_of(pat[k], col);
        log_total += (double)cnt * log(o.c) + (double)(cnt - (k == k_last ? 1 : 0)) * log(m.c);
    }
    // every resc_every sub-steps (a multiple of the period: the factor is then the same each
    // time) the kernel multiplies by resc; what is left goes into final_scale, together with the
    // accumulated rounding error of resc
    int every = period * ((8 + period - 1) / period);
    p.resc_every = every;
    p.resc = (T)exp(log_period * (every / period));
    const int64_t n_resc = n_sub / every;
    p.final_scale = (T)exp(log_total - (double)n_resc * log((double)p.resc));
    const bool edge = !periodic || p.n_lanes < 32;
    return launch_line_t<T>(p, ns, edge, col, st);
}

template <typename T, int S, bool PERY>
int launch_ycol(const YcolParams<T>& p, cudaStream_t st) {
    constexpr uint32_t SLOTB = 4 * kYCols * sizeof(T);
    const size_t smem = (size_t)kYWarps * p.nst * (SLOTB + 8);
    auto kern = ycol_kernel<T, S, PERY>;
    static std::atomic<size_t> configured[64];
    int dev = 0;
    TS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64 || smem > configured[dev].load(std::memory_order_relaxed)) {
        TS_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (dev >= 0 && dev < 64) configured[dev].store(smem, std::memory_order_relaxed);
    }
    const int n_seg = (p.ny + p.seg_rows - 1) / p.seg_rows;
    dim3 grid((p.n_strips + kYWarps - 1) / kYWarps, n_seg);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(kYWarps * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    // as in ts_stream.cu: dependent launch only for grids of at most one wave
    cfg.numAttrs = ((int64_t)grid.x * grid.y <= 148 * 3) ? 1 : 0;
    TS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, p));
    return TS_OK;
}

template <typename T, int S>
int launch_ycol_s(const YcolParams<T>& p, cudaStream_t st) {
    return p.periodic_y ? launch_ycol<T, S, true>(p, st) : launch_ycol<T, S, false>(p, st);
}

// One pipelined pass along the columns: sub-steps subs[0 .. n) chained, padded with identity
// sub-steps (zero angle) up to the instantiated depth S.
template <typename T>
int ycol_pass(const LatticeDesc& L, const T* src_re, const T* src_im, T* dst_re, T* dst_im,
              const StepCoef* subs, int n, int S, int seg_rows, int nst, cudaStream_t st) {
    YcolParams<T> p;
    p.src_re = src_re; p.src_im = src_im; p.dst_re = dst_re; p.dst_im = dst_im;
    p.nx = (int)L.nx; p.ny = (int)L.ny;
    p.n_strips = (int)((L.nx + kYCols - 1) / kYCols);
    p.seg_rows = seg_rows;
    p.nst = nst;
    p.periodic_y = L.periodic_y;
    double log_scale = 0.0;
    Angle prev{1.0, 0.0};
    for (int j = 0; j <= kMaxChain; ++j) p.te[j] = T(0);
    for (int j = 0; j < kMaxChain; ++j) { p.to[j] = T(0); p.sec_o[j] = T(1); }
    for (int j = 0; j < S; ++j) {
        const Angle h = j < n ? half_of(subs[j]) : Angle{1.0, 0.0};
        const Angle o = j < n ? odd_of(subs[j], true) : Angle{1.0, 0.0};
        const Angle m = add(prev, h);            // closing half of j-1 merged with opening half of j
        p.te[j] = (T)(m.s / m.c);
        p.to[j] = (T)(o.s / o.c);
        p.sec_o[j] = (T)(1.0 / o.c);
        log_scale += log(m.c) + log(o.c);
        prev = h;
    }
    p.te[S] = (T)(prev.s / prev.c);
    log_scale += log(prev.c);
    p.out_scale = (T)exp(log_scale);
    switch (S) {
        case 4: return launch_ycol_s<T, 4>(p, st);
        case 8: return launch_ycol_s<T, 8>(p, st);
        case 12:
            if constexpr (sizeof(T) == 4) return launch_ycol_s<T, 12>(p, st);
            break;
        case 16:
            if constexpr (sizeof(T) == 4) return launch_ycol_s<T, 16>(p, st);
            break;
    }
    set_error("axis: pipeline depth not instantiated");
    return TS_EINVAL;
}

}  // namespace

// ---- entry points (ts_internal.h) -----------------------------------------------------------------

bool axis_supported(const LatticeDesc& L, const StepCoef* pat, int period) {
    if (period < 1 || period > kMaxPeriod) return false;
    if (L.nx % 4 || L.ny % 2 || L.nx >= (int64_t(1) << 30) || L.ny >= (int64_t(1) << 30)) return false;
    for (int k = 0; k < period; ++k) {
        const StepCoef& c = pat[k];
        const Angle m = add(half_of(c), half_of(pat[(k + 1) % period]));
        const Angle o = odd_of(c, false);
        if (!(c.a_h > 0.25 && c.a_f > 0.25 && m.c > 0.25 && o.c > 0.25)) return false;
    }
    // rows: resident, or windows of 1024 (fp32) / 512 (fp64) sites; a closed row needs its ends
    // on lane boundaries
    const int wns = L.dtype == TS_F32 ? 32 : 16;
    const bool x_res = line_sites_per_lane(L.nx, L.dtype, false) != 0 &&
                       (L.nx % 4 == 0 || L.dtype == TS_F32);
    const bool x_win = L.nx > 32 * wns && (L.periodic_x || L.nx % wns == 0);
    // columns: resident, or the pipeline (whole segments of at least the warm-up depth)
    const bool y_res = line_sites_per_lane(L.ny, L.dtype, true) != 0;
    const bool y_pipe = L.ny >= 64;
    return (x_res || x_win) && (y_res || y_pipe);
}

int axis_default_chain(const LatticeDesc& L) {
    return L.dtype == TS_F32 ? 12 : 8;
}

template <typename T>
static int axis_evolve_t(const LatticeDesc& L, T* psi_re, T* psi_im, T* scr_re, T* scr_im,
                         const StepCoef* pat, int period, int64_t n_sub, int chain, int seg_rows,
                         int nst, cudaStream_t st, AxisInfo* info) {
    T* cur_re = psi_re; T* cur_im = psi_im;
    T* nxt_re = scr_re; T* nxt_im = scr_im;
    auto flip = [&]() {
        T* t;
        t = cur_re; cur_re = nxt_re; nxt_re = t;
        t = cur_im; cur_im = nxt_im; nxt_im = t;
    };
    info->passes = 0; info->launches = 0; info->chain_x = info->chain_y = 0; info->seg_rows = 0;
    const bool x_res = line_sites_per_lane(L.nx, L.dtype, false) != 0;
    const bool y_res = line_sites_per_lane(L.ny, L.dtype, true) != 0;
    int rc;
    // ---- rows
    if (x_res) {
        rc = line_pass<T>(L, cur_re, cur_im, cur_re, cur_im, pat, period, 0, n_sub, false, false, st);
        if (rc != TS_OK) return rc;
        ++info->passes; ++info->launches;
        info->chain_x = n_sub;
    } else {
        const int sx = chain < kMaxChain ? chain : kMaxChain;
        for (int64_t i = 0; i < n_sub; i += sx) {
            const int64_t s = n_sub - i < sx ? n_sub - i : sx;
            rc = line_pass<T>(L, cur_re, cur_im, nxt_re, nxt_im, pat, period, i, s, false, true, st);
            if (rc != TS_OK) return rc;
            flip();
            ++info->passes; ++info->launches;
        }
        info->chain_x = sx;
    }
    // ---- columns
    if (y_res) {
        rc = line_pass<T>(L, cur_re, cur_im, cur_re, cur_im, pat, period, 0, n_sub, true, false, st);
        if (rc != TS_OK) return rc;
        ++info->passes; ++info->launches;
        info->chain_y = n_sub;
    } else {
        // pipeline depth: the smallest instantiated one that holds the chain length asked for
        const int smax = sizeof(T) == 4 ? kMaxChain : 8;
        int want = (int)(n_sub < chain ? n_sub : chain);
        if (want > smax) want = smax;
        const int S = want <= 4 ? 4 : want <= 8 ? 8 : want <= 12 ? 12 : 16;
        const int per_pass = want;
        int seg = seg_rows;
        if (seg <= 0) {
            // whole waves of warps (148 SMs x 12 resident warps), segments of at most 1024 rows
            // (the 4S warm-up rows per segment against the fill of the last wave)
            const int64_t strips = (L.nx + kYCols - 1) / kYCols;
            const int64_t blocks_x = (strips + kYWarps - 1) / kYWarps;
            const int64_t slots = 148 * 3;
            const int64_t cap = 1024;
            const int64_t min_segs = (L.ny + cap - 1) / cap;
            int64_t waves = (min_segs * blocks_x + slots - 1) / slots;
            if (waves < 1) waves = 1;
            int64_t segs = waves * slots / blocks_x;
            if (segs < 1) segs = 1;
            int64_t r = (L.ny + segs - 1) / segs;
            r += r % 2;
            if (r > cap) r = cap;
            if (r < 16) r = 16;
            if (r > L.ny) r = L.ny;
            seg = (int)r;
        }
        const int slots = nst > 1 ? nst : 8;
        StepCoef subs[kMaxChain];
        for (int64_t i = 0; i < n_sub; i += per_pass) {
            const int s = (int)(n_sub - i < per_pass ? n_sub - i : per_pass);
            for (int j = 0; j < s; ++j) subs[j] = pat[(i + j) % period];
            rc = ycol_pass<T>(L, cur_re, cur_im, nxt_re, nxt_im, subs, s, S, seg, slots, st);
            if (rc != TS_OK) return rc;
            flip();
            ++info->passes; ++info->launches;
        }
        info->chain_y = per_pass;
        info->seg_rows = seg;
    }
    if (cur_re != psi_re) {
        const size_t plane_bytes = (size_t)L.nx * (size_t)L.ny * sizeof(T);
        TS_CUDA_TRY(cudaMemcpyAsync(psi_re, cur_re, plane_bytes, cudaMemcpyDeviceToDevice, st));
        TS_CUDA_TRY(cudaMemcpyAsync(psi_im, cur_im, plane_bytes, cudaMemcpyDeviceToDevice, st));
        info->launches += 2;
    }
    return TS_OK;
}

bool axis_needs_scratch(const LatticeDesc& L) {
    return line_sites_per_lane(L.nx, L.dtype, false) == 0 ||
           line_sites_per_lane(L.ny, L.dtype, true) == 0;
}

int axis_evolve(const LatticeDesc& L, void* psi_re, void* psi_im, void* scr_re, void* scr_im,
                const StepCoef* pat, int period, int64_t n_sub, int chain, int seg_rows, int nst,
                cudaStream_t st, AxisInfo* info) {
    if (chain <= 0) chain = axis_default_chain(L);
    if (L.dtype == TS_F32)
        return axis_evolve_t<float>(L, (float*)psi_re, (float*)psi_im, (float*)scr_re,
                                    (float*)scr_im, pat, period, n_sub, chain, seg_rows, nst, st,
                                    info);
    return axis_evolve_t<double>(L, (double*)psi_re, (double*)psi_im, (double*)scr_re,
                                 (double*)scr_im, pat, period, n_sub, chain, seg_rows, nst, st,
                                 info);
}

}  // namespace ts
