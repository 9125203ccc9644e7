// ts_axis.cu -- axis-split evolution for steps WITHOUT a potential (a flat potential
// drops the diagonal factor; the step is then the four kinetic parts only).
//
// A horizontal sweep acts inside rows, a vertical sweep along columns, both with scalar
// coefficients, so every X sweep commutes with every Y sweep (tensor-product structure; SURVEY
// 8(c)-5; pinned on the oracle by test_xy_regrouping / test_axis_split_identity and on dense
// matrices by test_stage_order...).  A chain of n second-order sub-steps therefore factorises
// EXACTLY,
//
//     U2(c_{n-1}) ... U2(c_0)  =  [X-chain along every row]  (x)  [Y-chain along every column],
//     axis chain = E(h_0) O(f_0) E(h_0 + h_1) O(f_1) ... O(f_{n-1}) E(h_{n-1}),
//
// E / O = even / odd pair sweep along the axis, h = half angle, f = full angle (adjacent half
// sweeps of chained sub-steps merged).  Only the rounding differs from the literal stage order.
// The two chains are independent 1-D problems -- no 2-D halo, no x-y coupling inside a kernel --
// and each gets the decomposition that suits it:
//
//   line_kernel   a WHOLE line (row or column) lives in registers for the complete chain -- all n
//                 sub-steps in ONE launch, the state read once and written once: NS consecutive
//                 sites per lane, 32 lanes per warp, up to 16 warps per line (16384 sites in fp32,
//                 8192 in fp64).  In-thread pairs are plain FMAs, one pair per lane and odd sweep
//                 crosses lanes by shuffle, one pair per warp crosses warps through 16 bytes of
//                 shared memory and an mbarrier per line (arrive after the even sweep, wait after
//                 the in-thread odd pairs).  No halo, no passes, no redundant work.
//   xwin_kernel   rows too long for a thread block: windows of 32 * NS sites with a halo of 2
//                 sites per sub-step and side that is recomputed and discarded,
//                 n <= 24 sub-steps per pass.
//   ycol_kernel   long COLUMNS: a streaming register pipeline -- a warp walks down a strip of 32
//                 columns, one per lane, S <= 24 chained sub-steps in flight, rows brought in by
//                 bulk async copies (TMA) into a per-warp shared-memory ring.  No x halo at all;
//                 4S warm-up rows per segment.
//
// A site is held as the register pair (re, im), so that EVERY pair rotation, even or odd, is two
// packed FMAs:  (p.re, p.im) += (-t, t) * (q.im, q.re)  and the same with p and q exchanged
// (sm_100 fma.rn.f32x2; ptxas folds the swapped source pair into an operand modifier).
#include <math.h>
#include <stdlib.h>

#include <atomic>
#include <type_traits>

#include "ts_internal.h"
#include "ts_rows.cuh"
#include "ts_tma.cuh"

namespace ts {
namespace {

using namespace tma;

constexpr int kMaxPeriod = 8;     // longest pattern of distinct sub-steps (ts_evolve 1, ts_evolve_u4 5)
constexpr int kMaxChain = 24;     // sub-steps per windowed / pipelined pass
constexpr int kMaxLineWarps = 16; // warps that share one resident line

// ---------------------------------------------------------------------------------------------
// one site = (re, im); scaled pair rotation (ts_rows.cuh):
// (p, q) <- (p + i t q, q + i t p) from the old values of both; the factor cos is deferred
// ---------------------------------------------------------------------------------------------
template <typename T>
struct Cx {
    T re, im;
};
template <typename T>
struct Coef {   // (-t, +t): the multiplier pair of one packed FMA
    T n, p;
};
template <typename T>
__device__ __forceinline__ Coef<T> coef(T t) { return Coef<T>{-t, t}; }

template <typename T>
__device__ __forceinline__ void rotc(Cx<T>& p, Cx<T>& q, const Coef<T> c) {
    const T npr = fma(c.n, q.im, p.re), npi = fma(c.p, q.re, p.im);
    const T nqr = fma(c.n, p.im, q.re), nqi = fma(c.p, p.re, q.im);
    p.re = npr; p.im = npi; q.re = nqr; q.im = nqi;
}
// one side only: p <- p + i t q (the partner belongs to another lane, which does its own side)
template <typename T>
__device__ __forceinline__ void rot1(Cx<T>& p, const Cx<T>& q, const Coef<T> c) {
    const T npr = fma(c.n, q.im, p.re), npi = fma(c.p, q.re, p.im);
    p.re = npr; p.im = npi;
}
template <typename T>
__device__ __forceinline__ void mulc(Cx<T>& p, T s) { p.re *= s; p.im *= s; }
#ifndef TS_SCALAR_F32
__device__ __forceinline__ void rotc(Cx<float>& p, Cx<float>& q, const Coef<float> c) {
    float npr, npi, nqr, nqi;
    rows::fma2v(npr, npi, c.n, c.p, q.im, q.re, p.re, p.im);
    rows::fma2v(nqr, nqi, c.n, c.p, p.im, p.re, q.re, q.im);
    p.re = npr; p.im = npi; q.re = nqr; q.im = nqi;
}
__device__ __forceinline__ void rot1(Cx<float>& p, const Cx<float>& q, const Coef<float> c) {
    float npr, npi;
    rows::fma2v(npr, npi, c.n, c.p, q.im, q.re, p.re, p.im);
    p.re = npr; p.im = npi;
}
__device__ __forceinline__ void mulc(Cx<float>& p, float s) {
    rows::mul2v(p.re, p.im, p.re, p.im, s, s);
}
#endif

// ---------------------------------------------------------------------------------------------
// resident lines
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
    int n_lanes;            // one warp per line: lanes that hold sites (lines shorter than 32 * NS)
    int n_warps;            // warps per line (W); W > 1: every lane of every warp holds NS sites
    int lines_per_block;
    int periodic;
    // windows (xwin_kernel only)
    int n_win, wi, halo, lines_per_warp;
    int64_t n_sub;          // sub-steps of this launch
    int period, phase0;     // pattern of distinct sub-steps; index of this launch's first sub-step
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
    Cx<T> s[NS];
};

template <typename T, int NS>
__device__ __forceinline__ void line_even(Line<T, NS>& L, T t) {
    const Coef<T> c = coef(t);
#pragma unroll
    for (int k = 0; k < NS; k += 2) rotc(L.s[k], L.s[k + 1], c);
}
template <typename T, int NS>
__device__ __forceinline__ void line_scale(Line<T, NS>& L, T s) {
#pragma unroll
    for (int k = 0; k < NS; ++k) mulc(L.s[k], s);
}
// the in-thread pairs (1,2), (3,4), ... of the odd sweep
template <typename T, int NS>
__device__ __forceinline__ void line_odd_inner(Line<T, NS>& L, T t) {
    const Coef<T> c = coef(t);
#pragma unroll
    for (int k = 1; k + 1 < NS; k += 2) rotc(L.s[k], L.s[k + 1], c);
}
// the two sites whose partners (up: last site of the previous lane, dn: first site of the next)
// live elsewhere.  EDGE: a pair may be cut (closed end, ghost lanes): its coupling is 0 and the
// unpaired real site takes 1/cos of the omitted sweep instead (ts_rows.cuh).
template <typename T, int NS, bool EDGE>
__device__ __forceinline__ void line_odd_outer(Line<T, NS>& L, const Cx<T>& up, const Cx<T>& dn,
                                               T t, T sec, bool cut_up, bool cut_dn) {
    T t_up = t, t_dn = t;
    if (EDGE) {
        t_up = cut_up ? T(0) : t;
        t_dn = cut_dn ? T(0) : t;
        mulc(L.s[0], cut_up ? sec : T(1));
        mulc(L.s[NS - 1], cut_dn ? sec : T(1));
    }
    rot1(L.s[0], up, coef(t_up));
    rot1(L.s[NS - 1], dn, coef(t_dn));
}

template <typename T>
struct Piece {   // sites per 16-byte access
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

// the chain E(h_0) O(f_0) E(h_0 + h_1) ... O(f_{n-1}) E(h_{n-1}) on the sites a lane holds;
// pattern entry k = (phase0 + s) mod period.  `outer` supplies the cross-lane partners of one odd
// sweep and applies them.  Uniform steps (period 1, ts_evolve) keep their three tangents in
// uniform registers: a coefficient that is indexed by the running pattern position ends up in a
// vector register instead, and a packed FMA with three vector-register sources issues at two
// thirds of the rate.
template <typename T, int NS, typename Outer>
__device__ __forceinline__ void run_chain(const LineParams<T>& p, Line<T, NS>& L, Outer&& outer) {
    line_even(L, p.te_first);
    int since = 0;
    if (p.period == 1) {
        const T to = p.to[0], sec = p.sec_o[0], tm = p.te_mid[0];
#pragma unroll 1
        for (int64_t s = 1; s < p.n_sub; ++s) {
            outer(L, to, sec);
            line_even(L, tm);
            if (++since == p.resc_every) { since = 0; line_scale(L, p.resc); }
        }
        outer(L, to, sec);
    } else {
        int k = p.phase0;
#pragma unroll 1
        for (int64_t s = 1; s < p.n_sub; ++s) {
            outer(L, p.to[k], p.sec_o[k]);
            line_even(L, p.te_mid[k]);
            if (++k == p.period) k = 0;
            if (++since == p.resc_every) { since = 0; line_scale(L, p.resc); }
        }
        outer(L, p.to[k], p.sec_o[k]);
    }
    line_even(L, p.te_last);
}

// COL = false: rows (site stride 1, 16-byte accesses); COL = true: columns (site stride = pitch,
// scalar accesses; the warps of a block take adjacent columns at the same time, so that the
// 32-byte sectors they share are fetched once).  MW = false: one warp per line, nothing but
// registers and shuffles; MW = true: n_warps warps per line, the pair that straddles two warps
// exchanged through shared memory.  In place: a line is read completely before it is written.
template <typename T, int NS, bool EDGE, bool COL, bool MW>
__global__ void __launch_bounds__(MW ? 512 : 128, MW ? 1 : (sizeof(T) * NS >= 128 ? 3 : 4))
line_kernel(const __grid_constant__ LineParams<T> p) {
    constexpr int PW = (Piece<T>::n < NS) ? Piece<T>::n : NS;     // sites per vector access
    // per line: an mbarrier and two (parity) sets of per-warp boundary sites {first, last}
    __shared__ __align__(16) Cx<T> xbuf[MW ? kMaxLineWarps : 1][2][MW ? kMaxLineWarps : 1][2];
    __shared__ __align__(8) uint64_t xbar[MW ? kMaxLineWarps : 1];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int W = MW ? p.n_warps : 1;
    const int wl = MW ? warp % W : 0;           // this warp's place in its line
    const int grp = MW ? warp / W : warp;       // the line of the block this warp belongs to
    if (MW) {
        if (threadIdx.x < p.lines_per_block) mbar_init(smem_u32(&xbar[threadIdx.x]), W);
        mbar_fence_init();
        __syncthreads();
    }
    const uint32_t bar = smem_u32(&xbar[MW ? grp : 0]);
    uint32_t ph = 0, par = 0;

    const int xl = (wl * 32 + lane) * NS;       // first site of the lane
    const bool active = MW || lane < p.n_lanes;
    // one warp per line: the ring of lanes that hold sites closes on itself (periodic line)
    const int up_src = MW ? lane - 1 : (lane == 0 ? p.n_lanes - 1 : lane - 1);
    const int dn_src = MW ? lane + 1 : (lane == p.n_lanes - 1 ? 0 : lane + 1);
    bool cut_up = false, cut_dn = false;
    if (EDGE) {
        // lanes beyond the line (ghosts: zeros that must stay zero) and the two ends of a closed line
        cut_up = !active || (!p.periodic && xl == 0);
        cut_dn = !active || (!p.periodic && xl + NS == p.n_sites);
    }

    for (int line = blockIdx.x * p.lines_per_block + grp; line < p.n_lines;
         line += gridDim.x * p.lines_per_block) {
        const int64_t base = (int64_t)line * p.line_stride;
        Line<T, NS> L;
        if (COL) {
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                const int64_t off = base + (int64_t)(xl + k) * p.site_stride;
                L.s[k].re = active ? __ldg(p.src_re + off) : T(0);
                L.s[k].im = active ? __ldg(p.src_im + off) : T(0);
            }
        } else {
#pragma unroll
            for (int k = 0; k < NS; k += PW) {
                T r[PW], i[PW];
                if (active) {
                    ld_piece(p.src_re + base + xl + k, r, PW);
                    ld_piece(p.src_im + base + xl + k, i, PW);
                }
#pragma unroll
                for (int j = 0; j < PW; ++j) {
                    L.s[k + j].re = active ? r[j] : T(0);
                    L.s[k + j].im = active ? i[j] : T(0);
                }
            }
        }

        run_chain<T, NS>(p, L, [&](Line<T, NS>& M, T t, T sec) {
            if (MW) {
                // publish the boundary sites (state after the even sweep), then the in-warp work,
                // then pick up the neighbours' -- the wait overlaps the in-thread pairs
                if (lane == 0) xbuf[grp][par][wl][0] = M.s[0];
                if (lane == 31) xbuf[grp][par][wl][1] = M.s[NS - 1];
                __syncwarp();
                if (lane == 0) mbar_arrive(bar);
            }
            Cx<T> up, dn;
            up.re = __shfl_sync(0xffffffffu, M.s[NS - 1].re, up_src);
            up.im = __shfl_sync(0xffffffffu, M.s[NS - 1].im, up_src);
            dn.re = __shfl_sync(0xffffffffu, M.s[0].re, dn_src);
            dn.im = __shfl_sync(0xffffffffu, M.s[0].im, dn_src);
            line_odd_inner(M, t);
            if (MW) {
                mbar_wait(bar, ph);
                ph ^= 1;
                const int wu = wl == 0 ? W - 1 : wl - 1, wd = wl == W - 1 ? 0 : wl + 1;
                if (lane == 0) up = xbuf[grp][par][wu][1];
                if (lane == 31) dn = xbuf[grp][par][wd][0];
                par ^= 1;
            }
            line_odd_outer<T, NS, EDGE>(M, up, dn, t, sec, cut_up, cut_dn);
        });

        line_scale(L, p.final_scale);
        if (!active) continue;
        if (COL) {
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                const int64_t off = base + (int64_t)(xl + k) * p.site_stride;
                p.dst_re[off] = L.s[k].re;
                p.dst_im[off] = L.s[k].im;
            }
        } else {
#pragma unroll
            for (int k = 0; k < NS; k += PW) {
                T r[PW], i[PW];
#pragma unroll
                for (int j = 0; j < PW; ++j) { r[j] = L.s[k + j].re; i[j] = L.s[k + j].im; }
                st_piece(p.dst_re + base + xl + k, r, PW);
                st_piece(p.dst_im + base + xl + k, i, PW);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// windowed rows (rows longer than a thread block holds)
// ---------------------------------------------------------------------------------------------
// A warp takes a window of 32 * NS sites of a block of consecutive rows, out of place; the next
// row is loaded into a second register set while the current one is computed.
template <typename T, int NS, bool EDGE>
__global__ void __launch_bounds__(128, 2)
xwin_kernel(const __grid_constant__ LineParams<T> p) {
    constexpr int PW = Piece<T>::n;
    const int lane = threadIdx.x & 31;
    const int wg = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int win = wg % p.n_win;
    const int line0 = (wg / p.n_win) * p.lines_per_warp;
    const int line1 = min(line0 + p.lines_per_warp, p.n_lines);
    if (line0 >= p.n_lines) return;

    const int xs = win * p.wi - p.halo;          // first site of the window (may be < 0)
    const int xl = xs + NS * lane;               // first site of the lane
    // the wrap-around partners of lanes 0 / 31 only reach the halo, which is discarded
    const int up_src = (lane + 31) & 31, dn_src = (lane + 1) & 31;
    bool cut_up = false, cut_dn = false;
    if (EDGE) {   // closed row: its ends fall between two lanes (the halo is a multiple of NS)
        cut_up = xl == 0 || xl == p.n_sites;
        cut_dn = xl + NS == p.n_sites || xl + NS == 0;
    }
    const int st_lo = win * p.wi;                // interior of the window: what this warp stores
    const int st_hi = min(st_lo + p.wi, p.n_sites);

    auto load = [&](int line, Line<T, NS>& L) {
        const int64_t base = (int64_t)line * p.line_stride;
#pragma unroll
        for (int k = 0; k < NS; k += PW) {
            int x = xl + k;
            bool ok = true;
            if (p.periodic) x = rows::wrap_index(x, p.n_sites);
            else ok = x >= 0 && x < p.n_sites;
            T r[PW], i[PW];
            if (ok) {
                ld_piece(p.src_re + base + x, r, PW);
                ld_piece(p.src_im + base + x, i, PW);
            }
#pragma unroll
            for (int j = 0; j < PW; ++j) {
                L.s[k + j].re = ok ? r[j] : T(0);
                L.s[k + j].im = ok ? i[j] : T(0);
            }
        }
    };
    auto store = [&](int line, Line<T, NS>& L) {
        const int64_t base = (int64_t)line * p.line_stride;
        line_scale(L, p.final_scale);
#pragma unroll
        for (int k = 0; k < NS; k += PW) {
            const int x = xl + k;
            if (x >= st_lo && x < st_hi) {
                T r[PW], i[PW];
#pragma unroll
                for (int j = 0; j < PW; ++j) { r[j] = L.s[k + j].re; i[j] = L.s[k + j].im; }
                st_piece(p.dst_re + base + x, r, PW);
                st_piece(p.dst_im + base + x, i, PW);
            }
        }
    };
    auto chain = [&](Line<T, NS>& L) {
        run_chain<T, NS>(p, L, [&](Line<T, NS>& M, T t, T sec) {
            Cx<T> up, dn;
            up.re = __shfl_sync(0xffffffffu, M.s[NS - 1].re, up_src);
            up.im = __shfl_sync(0xffffffffu, M.s[NS - 1].im, up_src);
            dn.re = __shfl_sync(0xffffffffu, M.s[0].re, dn_src);
            dn.im = __shfl_sync(0xffffffffu, M.s[0].im, dn_src);
            line_odd_inner(M, t);
            line_odd_outer<T, NS, EDGE>(M, up, dn, t, sec, cut_up, cut_dn);
        });
    };

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

// ---------------------------------------------------------------------------------------------
// column pipeline kernel
// ---------------------------------------------------------------------------------------------
constexpr int kYWarps = 4;
constexpr int kYCols = 32;        // columns per warp: one per lane

template <typename T>
struct YcolParams {
    const T* src_re;
    const T* src_im;
    T* dst_re;
    T* dst_im;
    int nx, ny;
    int n_strips, seg_rows, nst;
    int periodic_y;
    Coef<T> te[kMaxChain + 1];   // even sweeps: opening half, S-1 merged, closing half
    Coef<T> to[kMaxChain];       // odd sweep of sub-step j (the caller's full-angle coefficients)
    T sec_o[kMaxChain];
    T out_scale;
};

// stages 0..S-1 of one iteration.  Stage J holds the row pair that still waits for its odd
// partner below; the incoming pair (x0, x1) = rows (y - 2J, y - 2J + 1) gets the even sweep that
// opens sub-step J (merged with the one that closed sub-step J-1), then the odd sweep couples
// the waiting pair's lower row with x0, and the waiting pair moves on to stage J+1.  Stage J owns
// two register sets (ts_stream.cu: ping-pong form): the incoming pair is written to set u while
// the pair that waited in set u^1 leaves.
template <typename T, int S, bool EDGE, int J>
struct YStages {
    static __device__ __forceinline__ void run(const YcolParams<T>& p, int y, Cx<T> (&W)[S][2][2],
                                               const int u, Cx<T>& x0, Cx<T>& x1) {
        Cx<T>& a0 = W[J][u][0];
        Cx<T>& a1 = W[J][u][1];
        Cx<T>& g = W[J][u ^ 1][0];
        Cx<T>& h = W[J][u ^ 1][1];
        a0 = x0; a1 = x1;
        rotc(a0, a1, p.te[J]);
        if (EDGE) {
            // closed lattice: the odd pair (yj-1, yj) does not exist at yj = 0 and yj = ny; the
            // ghost row is zero and stays zero, the real row takes 1/cos of the omitted sweep
            const int yj = y - 2 * J;
            const bool yedge = yj == 0 || yj == p.ny;
            Coef<T> c = p.to[J];
            if (yedge) { c.n = T(0); c.p = T(0); }
            rotc(h, a0, c);
            const T sy = yedge ? p.sec_o[J] : T(1);
            mulc(h, sy); mulc(a0, sy);
        } else {
            rotc(h, a0, p.to[J]);
        }
        if (J == S - 1) rotc(g, h, p.te[S]);
        x0 = g; x1 = h;
        if constexpr (J + 1 < S) YStages<T, S, EDGE, J + 1>::run(p, y, W, u, x0, x1);
    }
};

__device__ __forceinline__ float lds1(uint32_t addr, float) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ double lds1(uint32_t addr, double) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}

// resident blocks per SM the register budget of the pipeline allows: S waiting row pairs, the
// incoming and the prefetched pair at 2 (fp32) / 4 (fp64) registers per site, ~64 for addresses,
// counters and temporaries (ptxas -v)
constexpr int ycol_blocks_for(int S, int words) {
    const int est = (S + 3) * 4 * words + 64;
    return est <= 128 ? 4 : est <= 168 ? 3 : 2;
}
template <typename T, int S>
constexpr int ycol_min_blocks() {
    return ycol_blocks_for(S, (int)(sizeof(T) / 4));
}

template <typename T, int S, bool PERY>
__global__ void __launch_bounds__(kYWarps * 32, ycol_min_blocks<T, S>())
ycol_kernel(const __grid_constant__ YcolParams<T> p) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr uint32_t ROWB = kYCols * sizeof(T);
    constexpr uint32_t SLOTB = 4 * ROWB;          // re0 im0 re1 im1

    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int strip = blockIdx.x * kYWarps + warp;
    if (strip >= p.n_strips) return;
    const int NST = p.nst;
    const int x0c = strip * kYCols;
    const int cols = min(kYCols, p.nx - x0c);
    const uint32_t bytes = cols * sizeof(T);
    const bool lane_ok = lane < cols;
    const uint32_t ring = smem_u32(smem_raw) + warp * NST * SLOTB;
    const uint32_t bars = smem_u32(smem_raw) + kYWarps * NST * SLOTB + warp * NST * 8;
    const uint32_t lane_off = lane * sizeof(T);

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
    // the ring is filled completely; iteration i lives in slot i mod NST and is refilled, for
    // iteration i + NST, at the top of iteration i + 1 (when its values have been consumed)
    for (int k = 0; k < NST; ++k)
        if (k < n_iter) issue();

    auto run = [&](auto edge_tag) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        Cx<T> W[S][2][2];
#pragma unroll
        for (int s = 0; s < S; ++s)
#pragma unroll
            for (int a = 0; a < 4; ++a) { W[s][a >> 1][a & 1].re = T(0); W[s][a >> 1][a & 1].im = T(0); }
        // software pipeline over the ring: while iteration i is computed, the row pair of
        // iteration i+1 is read from its slot (known complete) and the barrier of iteration i+2 is
        // tested; the blocking wait on it comes after the arithmetic has been issued
        uint32_t l_src = ring + lane_off, l_bar = bars, l_ph = 0;      // slot of iteration i + 1
        int l_slot = 0;
        auto advance = [&]() {
            l_src += SLOTB; l_bar += 8;
            if (++l_slot == NST) { l_slot = 0; l_src = ring + lane_off; l_bar = bars; l_ph ^= 1; }
        };
        auto fetch_regs = [&](int y, Cx<T>& a, Cx<T>& b) {
            const bool rowok = !EDGE || (y >= 0 && y < p.ny);
            if (rowok) {
                a.re = lds1(l_src, T()); a.im = lds1(l_src + ROWB, T());
                b.re = lds1(l_src + 2 * ROWB, T()); b.im = lds1(l_src + 3 * ROWB, T());
            } else {
                a.re = a.im = b.re = b.im = T(0);
            }
        };
        Cx<T> xa[2], xb[2];
        mbar_wait(l_bar, l_ph);
        fetch_regs(y_in0, xa[0], xa[1]);
        advance();
        if (1 < n_iter) mbar_wait(l_bar, l_ph);     // n_iter is even and >= 2
        int y = y_in0;
        T* o_re = p.dst_re + (int64_t)(y_in0 - 2 * S) * p.nx + x0c + lane;
        T* o_im = p.dst_im + (int64_t)(y_in0 - 2 * S) * p.nx + x0c + lane;
#pragma unroll 1
        for (int it0 = 0; it0 < n_iter; it0 += 2) {
            auto half = [&](auto utag, Cx<T> (&cur)[2], Cx<T> (&nxt)[2]) {
                constexpr int U = decltype(utag)::value;
                const int it = it0 + U;
                __syncwarp();      // every lane has consumed the slot of iteration it - 1
                if (it >= 1 && it - 1 + NST < n_iter) issue();
                // slot of iteration it + 1: complete (waited for below, one iteration ago)
                if (it + 1 < n_iter) fetch_regs(y + 2, nxt[0], nxt[1]);
                advance();
                bool ready = true;
                if (it + 2 < n_iter) ready = mbar_test(l_bar, l_ph);
                Cx<T> x0 = cur[0], x1 = cur[1];
                YStages<T, S, EDGE, 0>::run(p, y, W, U, x0, x1);
                if (it >= 2 * S && lane_ok && y - 2 * S < y_out1) {
                    mulc(x0, p.out_scale); mulc(x1, p.out_scale);
                    o_re[0] = x0.re; o_im[0] = x0.im;
                    o_re[p.nx] = x1.re; o_im[p.nx] = x1.im;
                }
                y += 2; o_re += 2 * (int64_t)p.nx; o_im += 2 * (int64_t)p.nx;
                if (!ready) mbar_wait(l_bar, l_ph);
            };
            half(std::integral_constant<int, 0>{}, xa, xb);
            half(std::integral_constant<int, 1>{}, xb, xa);
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

// How a line of n sites is held: NS sites per lane, W warps.  One warp: any n = NS * lanes with
// lanes <= 32; several warps: n = W * 32 * NS, W <= 16.  The smallest NS that fits (more lanes
// and warps share the work of a line).
struct LineShape {
    int ns, warps, lanes;
    bool ok() const { return ns != 0; }
};
LineShape line_shape(int64_t n, int dtype) {
    const int ns_max = dtype == TS_F32 ? 32 : 16;
    for (int ns = 2; ns <= ns_max; ns *= 2)
        if (n % ns == 0 && n / ns <= 32) return {ns, 1, (int)(n / ns)};
    for (int ns = 2; ns <= ns_max; ns *= 2)
        if (n % (32 * ns) == 0 && n / (32 * ns) <= kMaxLineWarps) return {ns, (int)(n / (32 * ns)), 32};
    return {0, 0, 0};
}

// resident columns are read with scalar accesses at stride nx: fine while the state stays in L2
bool column_resident(const LatticeDesc& L) {
    const int64_t bytes = L.nx * L.ny * (L.dtype == TS_F32 ? 8 : 16);
    static const int64_t mb = [] { const char* e = getenv("TS_PROBE_COLRES_MB"); return e ? atoll(e) : 48; }();
    return line_shape(L.ny, L.dtype).ok() && bytes <= (mb << 20);
}

int sm_count() {
    static int n = [] {
        int dev = 0, v = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v < 1)
            v = 148;
        return v;
    }();
    return n;
}

// tangents and deferred cosines of a chain of n_sub sub-steps starting at pattern position first
template <typename T>
void fill_chain(LineParams<T>& p, const StepCoef* pat, int period, int64_t first, int64_t n_sub,
                bool col) {
    p.n_sub = n_sub;
    p.period = period;
    p.phase0 = (int)(first % period);
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
    const int every = period * ((8 + period - 1) / period);
    p.resc_every = every;
    p.resc = (T)exp(log_period * (every / period));
    const int64_t n_resc = (n_sub - 1) / every;      // the last sub-step is outside the loop
    p.final_scale = (T)exp(log_total - (double)n_resc * log((double)p.resc));
}

template <typename T, int NS, bool EDGE, bool COL, bool MW>
int launch_line(const LineParams<T>& p, cudaStream_t st) {
    const int threads = p.lines_per_block * p.n_warps * 32;
    const int64_t groups = ((int64_t)p.n_lines + p.lines_per_block - 1) / p.lines_per_block;
    // several warps per line: the grid strides over the lines (barrier state lives in the block)
    int64_t blocks = groups;
    if (MW) {
        const int64_t resident = (int64_t)sm_count() * (512 / threads);
        if (blocks > resident) blocks = resident;
    }
    line_kernel<T, NS, EDGE, COL, MW><<<(unsigned)blocks, threads, 0, st>>>(p);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}
template <typename T, int NS, bool EDGE, bool COL>
int launch_line_mw(const LineParams<T>& p, cudaStream_t st) {
    return p.n_warps > 1 ? launch_line<T, NS, EDGE, COL, true>(p, st)
                         : launch_line<T, NS, EDGE, COL, false>(p, st);
}
template <typename T, int NS>
int launch_line_ns(const LineParams<T>& p, bool edge, bool col, cudaStream_t st) {
    if (col) return edge ? launch_line_mw<T, NS, true, true>(p, st) : launch_line_mw<T, NS, false, true>(p, st);
    return edge ? launch_line_mw<T, NS, true, false>(p, st) : launch_line_mw<T, NS, false, false>(p, st);
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

// One launch of the line kernel: ALL n_sub sub-steps of the pattern along the rows (col = false)
// or the columns, in place.
template <typename T>
int line_pass(const LatticeDesc& L, T* re, T* im, const StepCoef* pat, int period, int64_t n_sub,
              bool col, cudaStream_t st) {
    LineParams<T> p = {};
    p.src_re = re; p.src_im = im; p.dst_re = re; p.dst_im = im;
    const int64_t n = col ? L.ny : L.nx;
    const bool periodic = col ? L.periodic_y : L.periodic_x;
    p.n_lines = (int)(col ? L.nx : L.ny);
    p.n_sites = (int)n;
    p.line_stride = col ? 1 : L.nx;
    p.site_stride = col ? L.nx : 1;
    p.periodic = periodic;
    const LineShape sh = line_shape(n, L.dtype);
    if (!sh.ok()) { set_error("axis: line does not fit a thread block"); return TS_EUNSUPPORTED; }
    p.n_lanes = sh.lanes;
    p.n_warps = sh.warps;
    if (sh.warps == 1) {
        // 4 lines per block; columns: 8, so that a block covers whole 32-byte sectors in fp32
        p.lines_per_block = 4;
        const int64_t want = ((int64_t)p.n_lines + sm_count() * 4 - 1) / (sm_count() * 4);
        if (want < 4) p.lines_per_block = want < 1 ? 1 : (int)want;
    } else {
        p.lines_per_block = 1;
        if (sh.warps <= 8) p.lines_per_block = 4 / sh.warps > 1 ? 4 / sh.warps : 1;
    }
    fill_chain(p, pat, period, 0, n_sub, col);
    const bool edge = !periodic || sh.lanes < 32;
    return launch_line_t<T>(p, sh.ns, edge, col, st);
}

// One windowed pass along the rows: sub-steps [first, first + n_sub), n_sub <= kMaxChain, out of
// place.
template <typename T>
int xwin_pass(const LatticeDesc& L, const T* src_re, const T* src_im, T* dst_re, T* dst_im,
              const StepCoef* pat, int period, int64_t first, int64_t n_sub, cudaStream_t st) {
    LineParams<T> p = {};
    p.src_re = src_re; p.src_im = src_im; p.dst_re = dst_re; p.dst_im = dst_im;
    p.n_lines = (int)L.ny;
    p.n_sites = (int)L.nx;
    p.line_stride = L.nx;
    p.site_stride = 1;
    p.periodic = L.periodic_x;
    constexpr int ns = sizeof(T) == 4 ? 32 : 16;
    // the halo: 2 sites per sub-step; lane-aligned on a closed row so that its ends fall between
    // two lanes
    int halo = (int)((2 * n_sub + 3) / 4 * 4);
    if (!L.periodic_x) halo = (halo + ns - 1) / ns * ns;
    p.halo = halo;
    p.wi = 32 * ns - 2 * halo;
    p.n_win = (int)((L.nx + p.wi - 1) / p.wi);
    // about two waves of warps (8 per SM), at least 8 rows per warp
    int64_t lpw = ((int64_t)p.n_lines * p.n_win + 2 * sm_count() * 8 - 1) / (2 * sm_count() * 8);
    if (lpw < 8) lpw = 8;
    p.lines_per_warp = (int)lpw;
    fill_chain(p, pat, period, first, n_sub, false);
    const int64_t warps = (int64_t)p.n_win * ((p.n_lines + p.lines_per_warp - 1) / p.lines_per_warp);
    const unsigned blocks = (unsigned)((warps + 3) / 4);
    if (L.periodic_x) xwin_kernel<T, ns, false><<<blocks, 128, 0, st>>>(p);
    else xwin_kernel<T, ns, true><<<blocks, 128, 0, st>>>(p);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
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
    cfg.numAttrs = ((int64_t)grid.x * grid.y <= (int64_t)sm_count() * ycol_min_blocks<T, S>()) ? 1 : 0;
    TS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, p));
    return TS_OK;
}

template <typename T, int S>
int launch_ycol_s(const YcolParams<T>& p, cudaStream_t st) {
    return p.periodic_y ? launch_ycol<T, S, true>(p, st) : launch_ycol<T, S, false>(p, st);
}

// pipeline depths that are instantiated: the smallest one that holds n sub-steps
int ycol_depth(int n, int dtype) {
    const int d32[] = {4, 8, 12, 16, 20, 24};
    const int d64[] = {4, 8, 12};
    const int* d = dtype == TS_F32 ? d32 : d64;
    const int nd = dtype == TS_F32 ? 6 : 3;
    for (int i = 0; i < nd; ++i)
        if (n <= d[i]) return d[i];
    return d[nd - 1];
}
int ycol_blocks_per_sm(int S, int dtype) { return ycol_blocks_for(S, dtype == TS_F32 ? 1 : 2); }

// One pipelined pass along the columns: sub-steps subs[0 .. n) chained, padded with identity
// sub-steps (zero angle) up to the instantiated depth S.
template <typename T>
int ycol_pass(const LatticeDesc& L, const T* src_re, const T* src_im, T* dst_re, T* dst_im,
              const StepCoef* subs, int n, int S, int seg_rows, int nst, cudaStream_t st) {
    YcolParams<T> p = {};
    p.src_re = src_re; p.src_im = src_im; p.dst_re = dst_re; p.dst_im = dst_im;
    p.nx = (int)L.nx; p.ny = (int)L.ny;
    p.n_strips = (int)((L.nx + kYCols - 1) / kYCols);
    p.seg_rows = seg_rows;
    p.nst = nst;
    p.periodic_y = L.periodic_y;
    double log_scale = 0.0;
    Angle prev{1.0, 0.0};
    for (int j = 0; j <= kMaxChain; ++j) p.te[j] = Coef<T>{T(0), T(0)};
    for (int j = 0; j < kMaxChain; ++j) { p.to[j] = Coef<T>{T(0), T(0)}; p.sec_o[j] = T(1); }
    for (int j = 0; j < S; ++j) {
        const Angle h = j < n ? half_of(subs[j]) : Angle{1.0, 0.0};
        const Angle o = j < n ? odd_of(subs[j], true) : Angle{1.0, 0.0};
        const Angle m = add(prev, h);            // closing half of j-1 merged with opening half of j
        const T te = (T)(m.s / m.c), to = (T)(o.s / o.c);
        p.te[j] = Coef<T>{-te, te};
        p.to[j] = Coef<T>{-to, to};
        p.sec_o[j] = (T)(1.0 / o.c);
        log_scale += log(m.c) + log(o.c);
        prev = h;
    }
    const T tl = (T)(prev.s / prev.c);
    p.te[S] = Coef<T>{-tl, tl};
    log_scale += log(prev.c);
    p.out_scale = (T)exp(log_scale);
    switch (S) {
        case 4: return launch_ycol_s<T, 4>(p, st);
        case 8: return launch_ycol_s<T, 8>(p, st);
        case 12: return launch_ycol_s<T, 12>(p, st);
        case 16: if constexpr (sizeof(T) == 4) return launch_ycol_s<T, 16>(p, st); break;
        case 20: if constexpr (sizeof(T) == 4) return launch_ycol_s<T, 20>(p, st); break;
        case 24: if constexpr (sizeof(T) == 4) return launch_ycol_s<T, 24>(p, st); break;
    }
    set_error("axis: pipeline depth not instantiated");
    return TS_EINVAL;
}

// rows per segment of the column pipeline: a segment costs seg + 4S rows of work, so long
// segments win until the grid no longer fills the machine evenly.  Among the segment counts that
// give at most `cap` rows, take the one with the smallest makespan (waves of resident blocks x
// rows per block).
int ycol_default_seg(const LatticeDesc& L, int S) {
    const int64_t strips = (L.nx + kYCols - 1) / kYCols;
    const int64_t blocks_x = (strips + kYWarps - 1) / kYWarps;
    const int64_t slots = (int64_t)sm_count() * ycol_blocks_per_sm(S, L.dtype);
    const int64_t cap = 4096;
    int64_t best_seg = L.ny, best_cost = -1;
    for (int64_t segs = 1; segs <= L.ny / 2; ++segs) {
        int64_t r = (L.ny + segs - 1) / segs;
        r += r % 2;
        if (r < 16 && segs > 1) break;
        if (r > cap) continue;
        const int64_t n_seg = (L.ny + r - 1) / r;
        const int64_t waves = (n_seg * blocks_x + slots - 1) / slots;
        const int64_t cost = waves * (r + 4 * S);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_seg = r; }
        if (n_seg * blocks_x > 64 * slots) break;
    }
    return (int)best_seg;
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
    const bool x_res = line_shape(L.nx, L.dtype).ok();
    const bool x_win = L.nx > 32 * wns && (L.periodic_x || L.nx % wns == 0);
    // columns: resident, or the pipeline (whole segments of at least the warm-up depth)
    const bool y_res = column_resident(L);
    const bool y_pipe = L.ny >= 64;
    return (x_res || x_win) && (y_res || y_pipe);
}

int axis_default_chain(const LatticeDesc& L) {
    return L.dtype == TS_F32 ? 24 : 12;
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
    const bool x_res = line_shape(L.nx, L.dtype).ok();
    const bool y_res = column_resident(L);
    int rc;
    // ---- rows
    if (x_res) {
        rc = line_pass<T>(L, cur_re, cur_im, pat, period, n_sub, false, st);
        if (rc != TS_OK) return rc;
        ++info->passes; ++info->launches;
        info->chain_x = n_sub;
    } else {
        const int sx = chain < kMaxChain ? chain : kMaxChain;
        for (int64_t i = 0; i < n_sub; i += sx) {
            const int64_t s = n_sub - i < sx ? n_sub - i : sx;
            rc = xwin_pass<T>(L, cur_re, cur_im, nxt_re, nxt_im, pat, period, i, s, st);
            if (rc != TS_OK) return rc;
            flip();
            ++info->passes; ++info->launches;
        }
        info->chain_x = sx;
    }
    // ---- columns
    if (y_res) {
        rc = line_pass<T>(L, cur_re, cur_im, pat, period, n_sub, true, st);
        if (rc != TS_OK) return rc;
        ++info->passes; ++info->launches;
        info->chain_y = n_sub;
    } else {
        const int smax = ycol_depth(kMaxChain, L.dtype);
        int want = (int)(n_sub < chain ? n_sub : chain);
        if (want > smax) want = smax;
        // equal passes: 200 sub-steps at depth 24 are 9 passes of 22 or 23, not 8 of 24 and one of 8
        const int64_t n_pass = (n_sub + want - 1) / want;
        const int per_pass = (int)((n_sub + n_pass - 1) / n_pass);
        const int S = ycol_depth(per_pass, L.dtype);
        const int seg = seg_rows > 0 ? seg_rows : ycol_default_seg(L, S);
        // ring slots per warp: at least 3 (iteration i+2 is waited for while slot i-1 is the one
        // being refilled), at most what 200 KB of shared memory per block hold
        int slots = nst >= 3 ? nst : (nst > 0 ? 3 : 8);
        const int slot_max = (int)((200 << 10) / (kYWarps * (4 * kYCols * sizeof(T) + 8)));
        if (slots > slot_max) slots = slot_max;
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
    return !line_shape(L.nx, L.dtype).ok() || !column_resident(L);
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
