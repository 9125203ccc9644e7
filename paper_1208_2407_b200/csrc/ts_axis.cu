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
//                 sites per lane (2..32; 64 for some fp32 rows), 32 lanes per warp, up to 16 warps
//                 per line (16384 sites in fp32, 8192 in fp64).  In-thread pairs are plain FMAs, one pair per lane and odd sweep
//                 crosses lanes by shuffle, one pair per warp crosses warps through 16 bytes of
//                 shared memory and an mbarrier per line (arrive after the even sweep, wait after
//                 the in-thread odd pairs).  No halo, no passes, no redundant work.
//   xwin_kernel   rows too long for a thread block: windows of 32 * NS sites with a halo of 2
//                 sites per sub-step and side that is recomputed and discarded,
//                 n <= 24 sub-steps per pass.
//   ycol_kernel   long COLUMNS: a streaming register pipeline -- a warp walks down a strip of 32
//                 columns, one per lane, S <= 24 chained sub-steps in flight, rows brought in by
//                 2-D tensor-map copies (TMA, cp.async.bulk.tensor.2d) into a per-warp shared-memory
//                 ring whose slots hold the row pairs of two iterations under one mbarrier.  No x
//                 halo at all; 4S warm-up rows per segment.
//   tline_kernel  strided lines of a state that does not stay in L2 (y and z of a 3-D lattice):
//                 one LANE per line, 32 adjacent lines per warp (coalesced rows), the line cut
//                 over the warps of the block.
//
// The resident kernels use the IN-PLACE form of the rotation (first += i k1 second, then
// second += i k2 first') with one scale per index parity followed on the host -- see SubCoef --
// and can run, instead of a chain, a short sweep PROGRAM followed by the potential phase (the
// per-axis regrouping of 3-D steps with a potential, axis3_evolve).
//
// A site is held as the register pair (re, im), so that EVERY pair rotation, even or odd, is two
// packed FMAs:  (p.re, p.im) += (-t, t) * (q.im, q.re)  and the same with p and q exchanged
// (sm_100 fma.rn.f32x2; ptxas folds the swapped source pair into an operand modifier).
#include <cuda.h>       // CUtensorMap and its enums only: the encoder is fetched from the runtime
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <vector>
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
// In-place form of the pair rotation.  The from-old form above needs both old values for both
// results, so a sweep over a lane's NS sites writes a second register set (ptxas ping-pongs two
// full sets: 4 * NS registers in fp32, and the resident kernels spill).  Here the two sites of a
// pair are updated one after the other, each in place:
//
//     first  += i k1 * second            second += i k2 * first(new)
//
// With the sites stored as actual = scale * stored, scale xi on the first and eta on the second
// site, this is the rotation cos * [[1, i t],[i t, 1]] exactly when k1 = t eta / xi,
// k2 = t cos^2 xi / eta, and the scales become cos * xi and eta / cos.  Even sweeps update the
// even-index site first, odd sweeps the odd-index site, so over a sub-step (odd sweep + even sweep
// of the same angle) the two scales return to where they were: nothing is deferred, nothing grows,
// and the constants of uniform steps are the same in every sub-step.  All sites of one index
// parity share one scale; the host follows the two scales in double (fill_chain) and the kernel
// multiplies by what is left at the store.  Still two FMAs per site and sweep.
constexpr int kMaxTab = 16;       // sub-steps per table cycle of a non-uniform pattern
constexpr int kMaxProg = 4;       // sweeps of a sweep program

template <typename T>
struct SubCoef {   // one sub-step of a line chain: its odd sweep and the even sweep that follows it
    T o1, o2;      // odd sweep: odd-index site += i o1 * partner, then even-index site += i o2 * partner'
    // the even-index site of a cross-lane pair is computed from OLD values, second' = cos^2 second
    // + i o2 first_old, and the unpaired sites of a closed line only follow their scale (site 0
    // * cos, site n-1 / cos).  All three factors are 1 + (something tiny) and are applied as
    // s += d * s: a factor rounded to T next to 1 is off by up to 3e-8, the same in every sweep,
    // and the norm drifts (measured: -3e-5 over 100 steps on 64 x 64); d rounded to T is exact
    // to 1e-7 * |d|.
    T od2;         // -sin^2 = cos^2 - 1
    T odc, ods;    // cos - 1, 1 / cos - 1
    T e1, e2;      // the even sweep that follows: even-index site += i e1 * partner, then odd += i e2 * partner'
};

template <typename T>
struct LineParams {
    const T* src_re;
    const T* src_im;
    T* dst_re;
    T* dst_im;
    int64_t line_stride;    // elements between consecutive lines of one group
    int64_t site_stride;    // elements between consecutive sites of a line (1: rows)
    int64_t group_stride;   // elements between groups of lines_inner lines (3-D: planes)
    int n_lines, n_sites;
    int lines_inner;        // lines per group (2-D: all of them)
    int n_lanes;            // one warp per line: lanes that hold sites (lines shorter than 32 * NS)
    int n_warps;            // warps per line (W); W > 1: every lane of every warp holds NS sites
    int lines_per_block;
    int periodic;
    // windows (xwin_kernel only)
    int n_win, wi, halo, lines_per_warp;
    int64_t n_sub;          // sub-steps of this launch
    int n_tab;              // sub-steps per table cycle; 1: uniform steps (constants in uniform registers)
    int has_fix;            // after every cycle: s += fix * s per index parity (scales back to the cycle start)
    T fix_e, fix_o;
    T open1, open2;         // opening even half sweep
    T close1, close2;       // closing even half sweep (replaces the even sweep of the last sub-step)
    T fin_e, fin_o;         // what is left of the scales of even- / odd-index sites, applied at the store
    SubCoef<T> tab[kMaxTab];
    // sweep program (n_prog > 0, instead of a chain): up to kMaxProg sweeps with their own parity,
    // then optionally the potential phase of the lane's sites (3-D steps with a potential)
    int n_prog;
    int prog_parity[kMaxProg];
    SubCoef<T> prog[kMaxProg];      // odd sweep: o1, o2, od2, odc, ods; even sweep: e1, e2
    const T* ph_re;
    const T* ph_im;
};

template <typename T, int NS>
struct Line {
    Cx<T> s[NS];
};

// first += i k1 second, then second += i k2 first (in place)
template <typename T>
__device__ __forceinline__ void rot_seq(Cx<T>& first, Cx<T>& second, T k1, T k2) {
    rot1(first, second, coef(k1));
    rot1(second, first, coef(k2));
}
// p += d * p
template <typename T>
__device__ __forceinline__ void fixc(Cx<T>& p, T d) {
    p.re = fma(d, p.re, p.re); p.im = fma(d, p.im, p.im);
}
template <typename T, int NS>
__device__ __forceinline__ void line_even_all(Line<T, NS>& L, T e1, T e2) {
#pragma unroll
    for (int k = 0; k < NS; k += 2) rot_seq(L.s[k], L.s[k + 1], e1, e2);
}
// the even pairs that do not contain the lane's first or last site
template <typename T, int NS>
__device__ __forceinline__ void line_even_mid(Line<T, NS>& L, T e1, T e2) {
#pragma unroll
    for (int k = 2; k + 2 < NS; k += 2) rot_seq(L.s[k], L.s[k + 1], e1, e2);
}
template <typename T, int NS>
__device__ __forceinline__ void line_even_ends(Line<T, NS>& L, T e1, T e2) {
    rot_seq(L.s[0], L.s[1], e1, e2);
    if (NS > 2) rot_seq(L.s[NS - 2], L.s[NS - 1], e1, e2);
}
// the in-thread pairs (1,2), (3,4), ... of the odd sweep: the odd-index site goes first
template <typename T, int NS>
__device__ __forceinline__ void line_odd_inner(Line<T, NS>& L, T o1, T o2) {
#pragma unroll
    for (int k = 1; k + 1 < NS; k += 2) rot_seq(L.s[k], L.s[k + 1], o1, o2);
}
// the two sites whose partners (up: last site of the previous lane, dn: first site of the next)
// live elsewhere, both taken BEFORE this sweep.  The last site (odd index) goes first in its pair
// and uses the plain form; the first site (even index) goes second in its pair, whose other half
// is updated by the neighbour, so it is computed from the old values:
// second' = cos^2 second + i k2 first_old.  EDGE: a pair may be cut (closed end, ghost lanes): its
// coupling is 0 and the unpaired site only follows its scale (site 0: * cos, last site: / cos).
template <typename T, int NS, bool EDGE>
__device__ __forceinline__ void line_odd_outer(Line<T, NS>& L, const Cx<T>& up, const Cx<T>& dn,
                                               const SubCoef<T>& c, bool cut_up, bool cut_dn) {
    T k1 = c.o1, k2 = c.o2, d0 = c.od2;
    if (EDGE) {
        k1 = cut_dn ? T(0) : k1;
        k2 = cut_up ? T(0) : k2;
        d0 = cut_up ? c.odc : d0;
        fixc(L.s[NS - 1], cut_dn ? c.ods : T(0));
    }
    rot1(L.s[NS - 1], dn, coef(k1));
    fixc(L.s[0], d0);
    rot1(L.s[0], up, coef(k2));
}
template <typename T, int NS>
__device__ __forceinline__ void line_scale2(Line<T, NS>& L, T fe, T fo) {
#pragma unroll
    for (int k = 0; k < NS; k += 2) { mulc(L.s[k], fe); mulc(L.s[k + 1], fo); }
}
template <typename T, int NS>
__device__ __forceinline__ void line_fix(Line<T, NS>& L, T de, T dd) {
#pragma unroll
    for (int k = 0; k < NS; k += 2) { fixc(L.s[k], de); fixc(L.s[k + 1], dd); }
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

// The chain E(h_0) O(f_0) E(h_0 + h_1) ... O(f_{n-1}) E(h_{n-1}) on the sites a lane holds.  One
// sub-step = an odd sweep and the even sweep after it, in the order that hides the exchange of the
// two boundary sites: begin(L, up, dn) starts it (shuffles; several warps per line: publish +
// arrive), the in-thread odd pairs and the even pairs that do not need the boundary sites follow,
// end(up, dn) completes it (several warps: wait + pick up the neighbouring warps' sites), then the
// two outer odd pairs and the two outer even pairs.  Uniform steps keep their constants in uniform
// registers: a coefficient indexed by the running table position ends up in a vector register,
// and a packed FMA with three vector-register sources issues at two thirds of the rate.
template <typename T, int NS, bool EDGE, typename Begin, typename End>
__device__ __forceinline__ void run_chain(const LineParams<T>& p, Line<T, NS>& L, bool cut_up,
                                          bool cut_dn, Begin&& begin, End&& end) {
    auto substep = [&](const SubCoef<T>& c, T e1, T e2) {
        Cx<T> up, dn;
        begin(L, up, dn);
        line_odd_inner(L, c.o1, c.o2);
        // (the wait placed BEFORE these even pairs, so that they cover the shared-memory latency
        // of the exchange, measured the same: C4 rows 8.87 ms against 8.80 ms)
        line_even_mid(L, e1, e2);
        end(up, dn);
        line_odd_outer<T, NS, EDGE>(L, up, dn, c, cut_up, cut_dn);
        line_even_ends(L, e1, e2);
    };
    line_even_all(L, p.open1, p.open2);
    if (p.n_tab == 1) {
        const SubCoef<T> c = p.tab[0];
        // counted down in 32 bits: no loop bound to re-read, no 64-bit compare in the inner loop
        int64_t left = p.n_sub - 1;
#pragma unroll 1
        while (left > 0) {
            const int n = left > (1 << 30) ? (1 << 30) : (int)left;
            left -= n;
#pragma unroll 1
            for (int s = n; s > 0; --s) substep(c, c.e1, c.e2);
        }
        substep(c, p.close1, p.close2);
    } else {
        int j = 0;
#pragma unroll 1
        for (int64_t s = 1; s < p.n_sub; ++s) {
            const SubCoef<T> c = p.tab[j];
            substep(c, c.e1, c.e2);
            if (++j == p.n_tab) {
                j = 0;
                if (p.has_fix) line_fix(L, p.fix_e, p.fix_o);
            }
        }
        substep(p.tab[j], p.close1, p.close2);
    }
    line_scale2(L, p.fin_e, p.fin_o);
}

// A sweep program: a few sweeps with their own parities and angles (3-D steps with a potential:
// O(h) E(f) O(h) between two applications of the phase).  The final scales are applied by the
// caller after the phase.
template <typename T, int NS, bool EDGE, typename Begin, typename End>
__device__ __forceinline__ void run_prog(const LineParams<T>& p, Line<T, NS>& L, bool cut_up,
                                         bool cut_dn, Begin&& begin, End&& end) {
#pragma unroll 1
    for (int i = 0; i < p.n_prog; ++i) {
        const SubCoef<T> c = p.prog[i];
        if (p.prog_parity[i] == 0) {
            line_even_all(L, c.e1, c.e2);
        } else {
            Cx<T> up, dn;
            begin(L, up, dn);
            line_odd_inner(L, c.o1, c.o2);
            end(up, dn);
            line_odd_outer<T, NS, EDGE>(L, up, dn, c, cut_up, cut_dn);
        }
    }
}
// psi <- psi * (pr + i pi)
template <typename T>
__device__ __forceinline__ void phase_mul(Cx<T>& s, T pr, T pi) {
    const T r = s.re, m = s.im;
    s.re = fma(-m, pi, r * pr);
    s.im = fma(m, pr, r * pi);
}

// Shared-memory accesses of the exchange between the lanes of a line, as inline PTX under a
// predicate (the line kernel passes `true` and ptxas drops it; with a per-lane predicate they are
// the branch-free form of `if (lane == 0) ...`, which as an `if` cost two divergent branches and a
// reconvergence per sub-step -- ncu, r2d: branch_resolving was the top stall of the 16-warp kernel).
__device__ __forceinline__ void st_if(bool pred, uint32_t addr, const Cx<float>& v) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.u32 p, %0, 0;\n\t"
        "@p st.shared.v2.f32 [%1], {%2, %3};\n\t"
        "}" ::"r"((uint32_t)pred), "r"(addr), "f"(v.re), "f"(v.im) : "memory");
}
__device__ __forceinline__ void st_if(bool pred, uint32_t addr, const Cx<double>& v) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.u32 p, %0, 0;\n\t"
        "@p st.shared.v2.f64 [%1], {%2, %3};\n\t"
        "}" ::"r"((uint32_t)pred), "r"(addr), "d"(v.re), "d"(v.im) : "memory");
}
// wait with a bound: a protocol error traps instead of hanging the device
__device__ __forceinline__ void mbar_wait_bounded(uint32_t bar, uint32_t parity) {
    uint32_t done = 0, spins = 0;
    while (true) {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (done) break;
        if (++spins > (1u << 24)) __trap();
    }
}
__device__ __forceinline__ void ld_if(bool pred, uint32_t addr, Cx<float>& v) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.u32 p, %2, 0;\n\t"
        "@p ld.shared.v2.f32 {%0, %1}, [%3];\n\t"
        "}" : "+f"(v.re), "+f"(v.im) : "r"((uint32_t)pred), "r"(addr) : "memory");
}
__device__ __forceinline__ void ld_if(bool pred, uint32_t addr, Cx<double>& v) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.u32 p, %2, 0;\n\t"
        "@p ld.shared.v2.f64 {%0, %1}, [%3];\n\t"
        "}" : "+d"(v.re), "+d"(v.im) : "r"((uint32_t)pred), "r"(addr) : "memory");
}

// COL = false: rows (site stride 1, 16-byte accesses); COL = true: columns (site stride = pitch,
// scalar accesses; the warps of a block take adjacent columns at the same time, so that the
// 32-byte sectors they share are fetched once).  MW = false: one warp per line, nothing but
// registers and shuffles; MW = true: n_warps warps per line, the pair that straddles two warps
// exchanged through shared memory.  In place: a line is read completely before it is written.
template <typename T, int NS, bool EDGE, bool COL, bool MW>
__global__ void __launch_bounds__(MW ? (sizeof(T) * NS >= 256 ? 256 : 512) : 128,
                                  MW ? 1 : (sizeof(T) * NS >= 128 ? 3 : 4))
line_kernel(const __grid_constant__ LineParams<T> p) {
    constexpr int PW = (Piece<T>::n < NS) ? Piece<T>::n : NS;     // sites per vector access
    // Exchange between the lanes of a line that several warps share: every thread publishes its
    // first and its last site in shared memory (two parity sets, used by alternate sub-steps) and
    // reads its two neighbours' from there -- no shuffles, nothing predicated on the lane -- and
    // the line has ONE mbarrier that every THREAD arrives on after publishing (its own stores are
    // ordered before its own arrival: no __syncwarp, no elected lane; C4 rows 8.27 -> 8.17 ms).  (Before, r2: shuffles
    // inside a warp and only the pair that straddles two warps through shared memory, by
    // predicated accesses of lanes 0 / 31: 110 instructions per sub-step against 101, C4 rows
    // 8.55 ms against 8.26.  Measured alternative, r2g: neighbour-to-neighbour barriers -- two
    // arrivals and two waits per warp and sub-step, warps free to drift apart by a sub-step -- C4
    // rows 10.97 ms against 9.22 ms with the line-wide barrier.)
    __shared__ __align__(16) Cx<T> xs[2][2][MW ? 512 : 1];      // [parity set][first | last][thread]
    __shared__ __align__(8) uint64_t xbar[MW ? kMaxLineWarps : 1];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int W = MW ? p.n_warps : 1;
    const int wl = MW ? warp % W : 0;           // this warp's place in its line
    const int grp = MW ? warp / W : warp;       // the line of the block this warp belongs to
    if (MW) {
        if (threadIdx.x < p.lines_per_block) mbar_init(smem_u32(&xbar[threadIdx.x]), W * 32);
        mbar_fence_init();
        __syncthreads();
    }
    const uint32_t bar = smem_u32(&xbar[MW ? grp : 0]);
    uint32_t ph = 0;
    // the threads of a line are consecutive in the block; its ends close on each other (a closed
    // line ignores what it reads there)
    const int t_line0 = MW ? grp * W * 32 : 0;
    const int t_me = MW ? (int)threadIdx.x : 0;
    const int t_up = MW ? (t_me == t_line0 ? t_line0 + W * 32 - 1 : t_me - 1) : 0;
    const int t_dn = MW ? (t_me == t_line0 + W * 32 - 1 ? t_line0 : t_me + 1) : 0;
    // one running address (own `first` slot of the current parity set); everything else is a
    // constant distance from it: own `last` slot (immediate), the upper neighbour's `last`, the
    // lower neighbour's `first` (two per-thread constants: the ends of a line differ)
    constexpr uint32_t kWhichX = (MW ? 512 : 1) * sizeof(Cx<T>);
    constexpr uint32_t kParX = 2 * kWhichX;
    uint32_t sx = smem_u32(&xs[0][0][t_me]);
    const uint32_t d_up = kWhichX + (uint32_t)((t_up - t_me) * (int)sizeof(Cx<T>));
    const uint32_t d_dn = (uint32_t)((t_dn - t_me) * (int)sizeof(Cx<T>));

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
        const int grp_i = line / p.lines_inner;
        const int64_t base = (int64_t)grp_i * p.group_stride +
                             (int64_t)(line - grp_i * p.lines_inner) * p.line_stride;
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

        auto xbegin = [&](Line<T, NS>& M, Cx<T>& up, Cx<T>& dn) {
            if (MW) {
                // publish the two outer sites (state after the even sweep); the wait for the
                // neighbours' comes after the in-thread work
                st_if(true, sx, M.s[0]);
                st_if(true, sx + kWhichX, M.s[NS - 1]);
                mbar_arrive(bar);      // every thread: its own stores are ordered before its arrival
                return;
            }
            // one warp per line: the ring of lanes by shuffles
            up.re = __shfl_sync(0xffffffffu, M.s[NS - 1].re, up_src);
            up.im = __shfl_sync(0xffffffffu, M.s[NS - 1].im, up_src);
            dn.re = __shfl_sync(0xffffffffu, M.s[0].re, dn_src);
            dn.im = __shfl_sync(0xffffffffu, M.s[0].im, dn_src);
        };
        auto xend = [&](Cx<T>& up, Cx<T>& dn) {
            if (MW) {
                mbar_wait_bounded(bar, ph);
                ph ^= 1;
                ld_if(true, sx + d_up, up);
                ld_if(true, sx + d_dn, dn);
                sx ^= kParX;
            }
        };
        if (p.n_prog == 0) {
            run_chain<T, NS, EDGE>(p, L, cut_up, cut_dn, xbegin, xend);
        } else {
            run_prog<T, NS, EDGE>(p, L, cut_up, cut_dn, xbegin, xend);
            if (p.ph_re != nullptr && active) {
                if (COL) {
#pragma unroll
                    for (int k = 0; k < NS; ++k) {
                        const int64_t off = base + (int64_t)(xl + k) * p.site_stride;
                        phase_mul(L.s[k], __ldg(p.ph_re + off), __ldg(p.ph_im + off));
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < NS; k += PW) {
                        T r[PW], i[PW];
                        ld_piece(p.ph_re + base + xl + k, r, PW);
                        ld_piece(p.ph_im + base + xl + k, i, PW);
#pragma unroll
                        for (int j = 0; j < PW; ++j) phase_mul(L.s[k + j], r[j], i[j]);
                    }
                }
            }
            line_scale2(L, p.fin_e, p.fin_o);
        }

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
// strided lines, transposed: one LANE per line
// ---------------------------------------------------------------------------------------------
// Lines whose sites are far apart in memory (y and z of a 3-D lattice: stride nx, nx * ny) but
// whose NEIGHBOURING lines are adjacent: a warp takes 32 adjacent lines, one per lane, so every
// access is a coalesced 128-byte (fp32) row of 32 lines.  The line itself is cut over the W warps
// of the block: thread (warp w, lane l) holds sites [w NS, (w+1) NS) of line l -- all pairs are
// in-thread except the one that straddles two warps, which all 32 lanes exchange through shared
// memory (one mbarrier per block as in line_kernel, no shuffles at all).  The resident
// kernel above with strided scalar accesses (COL) touches a different DRAM page with every lane:
// 512^3 fp32, z lines: 7.5 ms per 100-step chain there, and 13.9 ms per 3-sweep launch with a
// potential (0.04 of the HBM roofline).
constexpr int kTWarps = 16;
template <typename T, int NS, bool EDGE>
__global__ void __launch_bounds__(kTWarps * 32, 1)
tline_kernel(const __grid_constant__ LineParams<T> p) {
    __shared__ __align__(16) Cx<T> xbuf[2][kTWarps][2][32];
    __shared__ __align__(8) uint64_t xbar;
    const int lane = threadIdx.x & 31;
    const int w = threadIdx.x >> 5;
    const int W = p.n_warps;
    if (threadIdx.x == 0) mbar_init(smem_u32(&xbar), W * 32);
    mbar_fence_init();
    __syncthreads();
    const uint32_t bar = smem_u32(&xbar);
    uint32_t ph = 0;
    int par = 0;
    const int wu = w == 0 ? W - 1 : w - 1, wd = w == W - 1 ? 0 : w + 1;
    const bool cut_up = EDGE && !p.periodic && w == 0;
    const bool cut_dn = EDGE && !p.periodic && w == W - 1;

    for (int64_t l0 = (int64_t)blockIdx.x * 32; l0 < p.n_lines; l0 += (int64_t)gridDim.x * 32) {
        const int64_t line = l0 + lane;
        const bool active = line < p.n_lines;
        const int64_t li = active ? line : p.n_lines - 1;
        const int64_t g = li / p.lines_inner;
        const int64_t base = g * p.group_stride + (li - g * p.lines_inner) * p.line_stride +
                             (int64_t)(w * NS) * p.site_stride;
        Line<T, NS> L;
        {   // running pointers: NS precomputed 64-bit offsets would cost 2 NS registers
            const T* q_re = p.src_re + base;
            const T* q_im = p.src_im + base;
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                L.s[k].re = active ? __ldg(q_re) : T(0);
                L.s[k].im = active ? __ldg(q_im) : T(0);
                q_re += p.site_stride; q_im += p.site_stride;
            }
        }
        auto xbegin = [&](Line<T, NS>& M, Cx<T>& up, Cx<T>& dn) {
            if (W == 1) { up = M.s[NS - 1]; dn = M.s[0]; return; }     // the line closes on itself
            xbuf[par][w][0][lane] = M.s[0];
            xbuf[par][w][1][lane] = M.s[NS - 1];
            mbar_arrive(bar);      // every thread, as in line_kernel: own stores before own arrival
        };
        auto xend = [&](Cx<T>& up, Cx<T>& dn) {
            if (W == 1) return;
            mbar_wait_bounded(bar, ph);
            ph ^= 1;
            up = xbuf[par][wu][1][lane];
            dn = xbuf[par][wd][0][lane];
            par ^= 1;
        };
        if (p.n_prog == 0) {
            run_chain<T, NS, EDGE>(p, L, cut_up, cut_dn, xbegin, xend);
        } else {
            run_prog<T, NS, EDGE>(p, L, cut_up, cut_dn, xbegin, xend);
            if (p.ph_re != nullptr && active) {
                const T* q_re = p.ph_re + base;
                const T* q_im = p.ph_im + base;
#pragma unroll
                for (int k = 0; k < NS; ++k) {
                    phase_mul(L.s[k], __ldg(q_re), __ldg(q_im));
                    q_re += p.site_stride; q_im += p.site_stride;
                }
            }
            line_scale2(L, p.fin_e, p.fin_o);
        }
        if (!active) continue;
        T* o_re = p.dst_re + base;
        T* o_im = p.dst_im + base;
#pragma unroll
        for (int k = 0; k < NS; ++k) {
            *o_re = L.s[k].re;
            *o_im = L.s[k].im;
            o_re += p.site_stride; o_im += p.site_stride;
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
        run_chain<T, NS, EDGE>(
            p, L, cut_up, cut_dn,
            [&](Line<T, NS>& M, Cx<T>& up, Cx<T>& dn) {
                up.re = __shfl_sync(0xffffffffu, M.s[NS - 1].re, up_src);
                up.im = __shfl_sync(0xffffffffu, M.s[NS - 1].im, up_src);
                dn.re = __shfl_sync(0xffffffffu, M.s[0].re, dn_src);
                dn.im = __shfl_sync(0xffffffffu, M.s[0].im, dn_src);
            },
            [&](Cx<T>&, Cx<T>&) {});
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
    int edge_rows;               // closed in y: rows of the short first and last segment (0: none)
    int periodic_y;
    Coef<T> te[kMaxChain + 1];   // even sweeps: opening half, S-1 merged, closing half
    Coef<T> to[kMaxChain];       // odd sweep of sub-step j (the caller's full-angle coefficients)
    T sec_o[kMaxChain];
    T out_scale;
    // uniform passes (UNI: S equal sub-steps, nothing padded): four coefficient pairs that stay in
    // uniform registers instead of 2S + 1 pairs in vector registers
    Coef<T> u_open, u_mid, u_odd, u_close;
    T u_sec;
};

// coefficient of stage J: per-stage table, or the uniform pass's four pairs
template <typename T, int S, bool UNI>
struct YCoef {
    static __device__ __forceinline__ Coef<T> even(const YcolParams<T>& p, int J) {
        if (UNI) return J == 0 ? p.u_open : (J == S ? p.u_close : p.u_mid);
        return p.te[J];
    }
    static __device__ __forceinline__ Coef<T> odd(const YcolParams<T>& p, int J) {
        return UNI ? p.u_odd : p.to[J];
    }
    static __device__ __forceinline__ T sec(const YcolParams<T>& p, int J) {
        return UNI ? p.u_sec : p.sec_o[J];
    }
};

// stages 0..S-1 of one iteration.  Stage J holds the row pair that still waits for its odd
// partner below; the incoming pair (x0, x1) = rows (y - 2J, y - 2J + 1) gets the even sweep that
// opens sub-step J (merged with the one that closed sub-step J-1), then the odd sweep couples
// the waiting pair's lower row with x0, and the waiting pair moves on to stage J+1.  Stage J owns
// two register sets (ts_stream.cu: ping-pong form): the incoming pair is written to set u while
// the pair that waited in set u^1 leaves.
template <typename T, int S, bool EDGE, bool UNI, int J>
struct YStages {
    static __device__ __forceinline__ void run(const YcolParams<T>& p, int y, Cx<T> (&W)[S][2][2],
                                               const int u, Cx<T>& x0, Cx<T>& x1) {
        using C = YCoef<T, S, UNI>;
        Cx<T>& a0 = W[J][u][0];
        Cx<T>& a1 = W[J][u][1];
        Cx<T>& g = W[J][u ^ 1][0];
        Cx<T>& h = W[J][u ^ 1][1];
        a0 = x0; a1 = x1;
        rotc(a0, a1, C::even(p, J));
        if (EDGE) {
            // closed lattice: the odd pair (yj-1, yj) does not exist at yj = 0 and yj = ny; the
            // ghost row is zero and stays zero, the real row takes 1/cos of the omitted sweep
            const int yj = y - 2 * J;
            const bool yedge = yj == 0 || yj == p.ny;
            Coef<T> c = C::odd(p, J);
            if (yedge) { c.n = T(0); c.p = T(0); }
            rotc(h, a0, c);
            const T sy = yedge ? C::sec(p, J) : T(1);
            mulc(h, sy); mulc(a0, sy);
        } else {
            rotc(h, a0, C::odd(p, J));
        }
        if (J == S - 1) rotc(g, h, C::even(p, S));
        x0 = g; x1 = h;
        if constexpr (J + 1 < S) YStages<T, S, EDGE, UNI, J + 1>::run(p, y, W, u, x0, x1);
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
constexpr int ycol_blocks_for(int S, int words, bool uni) {
    // uniform fp32 passes (ptxas -v: no spills at these caps); the others by estimate
    if (uni && words == 1) return S <= 12 ? 4 : S <= 20 ? 3 : 2;
    const int est = (S + 3) * 4 * words + 64;
    return est <= 128 ? 4 : est <= 168 ? 3 : 2;
}
template <typename T, int S, bool UNI>
constexpr int ycol_min_blocks() {
    return ycol_blocks_for(S, (int)(sizeof(T) / 4), UNI);
}

template <typename T, int S, bool PERY, bool UNI>
__global__ void __launch_bounds__(kYWarps * 32, ycol_min_blocks<T, S, UNI>())
ycol_kernel(const __grid_constant__ YcolParams<T> p, const __grid_constant__ CUtensorMap tm_re,
            const __grid_constant__ CUtensorMap tm_im) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr uint32_t ROWB = kYCols * sizeof(T);
    constexpr uint32_t SLOTB = 8 * ROWB;          // two row pairs: re0 re1 im0 im1, twice

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

    // Closed lattices: the segments that touch row 0 / ny run the edge variant of the loop, which
    // costs about 1.5x per row; as whole segments they ended every pass late (a closed 16384^2
    // lattice was 21 % slower than a periodic one).  They are cut SHORT instead (edge_rows), so
    // that the edge arithmetic covers a few per cent of the rows and those blocks finish early.
    int y_out0, y_out1;
    if (p.edge_rows > 0) {
        const int last = (int)gridDim.y - 1;
        if ((int)blockIdx.y == 0) { y_out0 = 0; y_out1 = p.edge_rows; }
        else if ((int)blockIdx.y == last) { y_out0 = p.ny - p.edge_rows; y_out1 = p.ny; }
        else {
            y_out0 = p.edge_rows + ((int)blockIdx.y - 1) * p.seg_rows;
            y_out1 = min(y_out0 + p.seg_rows, p.ny - p.edge_rows);
        }
    } else {
        y_out0 = blockIdx.y * p.seg_rows;
        y_out1 = min(y_out0 + p.seg_rows, p.ny);
    }
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

    // running fetch position (warp-uniform): rows (fy, fy+1) and (fy+2, fy+3) of the strip's columns
    int fy = PERY ? rows::wrap_index(y_in0, p.ny) : y_in0;
    uint32_t f_dst = ring, f_bar = bars;
    int f_slot = 0;
    // A ring slot holds the row pairs of TWO iterations (the loop body below is two iterations long)
    // and has ONE mbarrier: the slot counters, the barrier arithmetic and the refill test are paid
    // once per body, not once per iteration (they were ~23 of the 168 instructions of an
    // iteration).  Per pair and plane one tensor-map copy: the box is 32 columns x 2 rows at
    // element coordinates (x0c, y) -- no 64-bit address arithmetic in the loop, columns beyond the
    // lattice arrive as zeros, and the second pair wraps on its own on a periodic lattice.
    // Slot layout: pair A = re row 0, re row 1, im row 0, im row 1; pair B the same, 4 rows on.
    (void)bytes;
    auto issue = [&](auto edge_tag) {
        // (only the warps of the edge variant ever fetch rows beyond a closed lattice)
        constexpr bool EDGE = decltype(edge_tag)::value;
        int fy2 = fy + 2;
        if (PERY && fy2 >= p.ny) fy2 -= p.ny;
        const bool ok1 = !EDGE || (fy >= 0 && fy < p.ny);
        const bool ok2 = !EDGE || (fy2 >= 0 && fy2 < p.ny);
        if (leader) {
            if (ok1 || ok2) {
                mbar_arrive_expect_tx(f_bar, ((ok1 ? 4u : 0u) + (ok2 ? 4u : 0u)) * ROWB);
                if (ok1) {
                    tensor2d_g2s(f_dst, &tm_re, x0c, fy, f_bar);
                    tensor2d_g2s(f_dst + 2 * ROWB, &tm_im, x0c, fy, f_bar);
                }
                if (ok2) {
                    tensor2d_g2s(f_dst + 4 * ROWB, &tm_re, x0c, fy2, f_bar);
                    tensor2d_g2s(f_dst + 6 * ROWB, &tm_im, x0c, fy2, f_bar);
                }
            } else {
                mbar_arrive(f_bar);
            }
        }
        fy = fy2 + 2;
        if (PERY && fy >= p.ny) fy -= p.ny;
        f_dst += SLOTB; f_bar += 8;
        if (++f_slot == NST) { f_slot = 0; f_dst = ring; f_bar = bars; }
    };
    constexpr uint32_t kOffAim = 2 * ROWB, kOffBre = ROWB;      // a = row 0, b = row 1 of the pair
    // the ring is filled completely; body b (iterations 2b, 2b+1) lives in slot b mod NST, which is
    // refilled for body b + NST in the middle of body b (when both its pairs are in registers)
    auto run = [&](auto edge_tag) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        for (int k = 0; k < NST; ++k)
            if (2 * k < n_iter) issue(edge_tag);
        Cx<T> W[S][2][2];
#pragma unroll
        for (int s = 0; s < S; ++s)
#pragma unroll
            for (int a = 0; a < 4; ++a) { W[s][a >> 1][a & 1].re = T(0); W[s][a >> 1][a & 1].im = T(0); }
        // software pipeline over the ring: in the first half of body b pair A (read during the
        // previous body) is computed while pair B is read from the same slot and the barrier of
        // slot b+1 is tested (the blocking wait comes after the arithmetic has been issued); in
        // the second half the slot is handed back for refilling, pair A of body b+1 is read from
        // the next slot and pair B is computed
        uint32_t c_src = ring + lane_off;                       // slot of body b
        uint32_t n_src = c_src + SLOTB, n_bar = bars + 8, n_ph = 0;      // slot of body b + 1
        int n_slot = 1;
        if (NST == 1) { n_src = c_src; n_bar = bars; n_ph = 1; n_slot = 0; }
        auto fetch_regs = [&](uint32_t src, int y, Cx<T>& a, Cx<T>& b) {
            const bool rowok = !EDGE || (y >= 0 && y < p.ny);
            if (rowok) {
                a.re = lds1(src, T()); a.im = lds1(src + kOffAim, T());
                b.re = lds1(src + kOffBre, T()); b.im = lds1(src + 3 * ROWB, T());
            } else {
                a.re = a.im = b.re = b.im = T(0);
            }
        };
        Cx<T> xa[2], xb[2];
        mbar_wait(bars, 0);
        fetch_regs(c_src, y_in0, xa[0], xa[1]);
        int y = y_in0;
        T* o_re = p.dst_re + (int64_t)(y_in0 - 2 * S) * p.nx + x0c + lane;
        T* o_im = p.dst_im + (int64_t)(y_in0 - 2 * S) * p.nx + x0c + lane;
        auto stages = [&](auto utag, int it, Cx<T> (&cur)[2]) {
            constexpr int U = decltype(utag)::value;
            Cx<T> x0 = cur[0], x1 = cur[1];
            YStages<T, S, EDGE, UNI, 0>::run(p, y, W, U, x0, x1);
            if (it >= 2 * S && lane_ok && y - 2 * S < y_out1) {
                mulc(x0, p.out_scale); mulc(x1, p.out_scale);
                o_re[0] = x0.re; o_im[0] = x0.im;
                o_re[p.nx] = x1.re; o_im[p.nx] = x1.im;
            }
            y += 2; o_re += 2 * (int64_t)p.nx; o_im += 2 * (int64_t)p.nx;
        };
#pragma unroll 1
        for (int it0 = 0; it0 < n_iter; it0 += 2) {
            // ---- first half: pair A
            fetch_regs(c_src + 4 * ROWB, y + 2, xb[0], xb[1]);       // n_iter is even
            bool ready = true;
            if (it0 + 2 < n_iter) ready = mbar_test(n_bar, n_ph);
            stages(std::integral_constant<int, 0>{}, it0, xa);
            if (!ready) mbar_wait(n_bar, n_ph);
            // ---- second half: pair B
            __syncwarp();      // every lane has both pairs of this slot in registers
            if (it0 + 2 * NST < n_iter) issue(edge_tag);
            if (it0 + 2 < n_iter) fetch_regs(n_src, y + 2, xa[0], xa[1]);
            c_src = n_src;
            n_src += SLOTB; n_bar += 8;
            if (++n_slot == NST) { n_slot = 0; n_src = ring + lane_off; n_bar = bars; n_ph ^= 1; }
            stages(std::integral_constant<int, 1>{}, it0 + 1, xb);
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
// lanes <= 32 -- the smallest NS that fits (more lanes share the work of a line).  Several warps:
// n = W * 32 * NS, W <= 16 -- the LARGEST NS that fits: the warps of a line meet at a barrier every
// sub-step, so fewer warps with more in-lane work each is the cheaper cut (2048 sites: 2 warps of
// 32 sites per lane, not 16 warps of 4).
struct LineShape {
    int ns, warps, lanes;
    bool ok() const { return ns != 0; }
};
LineShape line_shape(int64_t n, int dtype) {
    const int ns_max = dtype == TS_F32 ? 32 : 16;
    for (int ns = 2; ns <= ns_max; ns *= 2)
        if (n % ns == 0 && n / ns <= 32) return {ns, 1, (int)(n / ns)};
    static const bool small_ns = getenv("TS_PROBE_MW_SMALL") != nullptr;     // tuning probe only
    if (small_ns) {
        for (int ns = 2; ns <= ns_max; ns *= 2)
            if (n % (32 * ns) == 0 && n / (32 * ns) <= kMaxLineWarps) return {ns, (int)(n / (32 * ns)), 32};
        return {0, 0, 0};
    }
    for (int ns = ns_max; ns >= 2; ns /= 2)
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

// Constants of a chain of n_sub sub-steps starting at pattern position `first`, for the in-place
// form of the rotations (see SubCoef).  The host follows the scales of the even-index and the
// odd-index sites (actual = scale * stored) in double through every sweep:
//   even sweep, angle (c, t = tan):  k1 = t be / al,  k2 = t c^2 al / be,  al *= c,  be /= c
//   odd sweep:                       k1 = t al / be,  k2 = t c^2 be / al,  be *= c,  al /= c
// (al: even-index sites, be: odd-index sites).  Uniform steps: the scales return after every
// sub-step (to rounding, which goes into the final scale) and one table entry serves all of them.
// Other patterns: a table cycle of n_tab sub-steps, after which the stored values are corrected
// by s += fix * s so that the scales are back at the start of the cycle (fix is tiny: the FMA form
// keeps its rounding error ~1e-7 * |fix|).
template <typename T>
void fill_chain(LineParams<T>& p, const StepCoef* pat, int period, int64_t first, int64_t n_sub,
                bool col) {
    p.n_sub = n_sub;
    double al = 1.0, be = 1.0;
    auto even_sweep = [&](const Angle& a, T& k1, T& k2) {
        const double t = a.s / a.c, rho = be / al;
        k1 = (T)(t * rho);
        k2 = (T)(t * a.c * a.c / rho);
        al *= a.c; be /= a.c;
    };
    auto odd_sweep = [&](const Angle& a, SubCoef<T>& sc) {
        const double t = a.s / a.c, rho = al / be;
        sc.o1 = (T)(t * rho);
        sc.o2 = (T)(t * a.c * a.c / rho);
        // cos - 1 without cancellation: -sin^2 / (1 + cos)
        const double cm1 = -(a.s * a.s) / (1.0 + a.c);
        sc.od2 = (T)(-(a.s * a.s));
        sc.odc = (T)cm1;
        sc.ods = (T)(-cm1 / a.c);
        be *= a.c; al /= a.c;
    };
    auto entry = [&](int64_t s) -> const StepCoef& { return pat[(first + s) % period]; };
    auto merged = [&](int64_t s) { return add(half_of(entry(s)), half_of(entry(s + 1))); };

    even_sweep(half_of(entry(0)), p.open1, p.open2);
    const double al0 = al, be0 = be;
    // uniform: one pattern entry whose merged even angle is the odd angle (the scales then return
    // after each sub-step up to the rounding of the caller's coefficients)
    bool uniform = period == 1;
    if (uniform) {
        const Angle m = merged(0), o = odd_of(entry(0), col);
        uniform = fabs(m.c / o.c - 1.0) < 1e-12;
    }
    p.n_tab = uniform ? 1 : period * (kMaxTab / period);
    for (int j = 0; j < kMaxTab; ++j) p.tab[j] = SubCoef<T>{T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    for (int j = 0; j < p.n_tab; ++j) {
        odd_sweep(odd_of(entry(j), col), p.tab[j]);
        even_sweep(merged(j), p.tab[j].e1, p.tab[j].e2);
    }
    // one cycle multiplies the scales by (ce, co); the fix takes that out of the stored values
    const double ce = al / al0, co = be / be0;
    p.has_fix = uniform ? 0 : 1;
    p.fix_e = uniform ? T(0) : (T)(ce - 1.0);
    p.fix_o = uniform ? T(0) : (T)(co - 1.0);
    // what a cycle really leaves behind (the fix is rounded to T; uniform: no fix at all)
    const double ge = ce / (1.0 + (double)p.fix_e), go = co / (1.0 + (double)p.fix_o);
    const int64_t n_cycles = (n_sub - 1) / p.n_tab;       // complete cycles before the last sub-step
    const int64_t rest = (n_sub - 1) - n_cycles * p.n_tab;
    // the last, partial cycle with the table's own (nominal) scales: `rest` whole sub-steps, then
    // the odd sweep of the last sub-step and the closing half sweep
    al = al0; be = be0;
    SubCoef<T> scratch;
    T k1, k2;
    for (int64_t j = 0; j < rest; ++j) {
        odd_sweep(odd_of(entry(j), col), scratch);
        even_sweep(merged(j), k1, k2);
    }
    odd_sweep(odd_of(entry(rest), col), scratch);
    even_sweep(half_of(entry(n_sub - 1)), p.close1, p.close2);
    p.fin_e = (T)(al * exp((double)n_cycles * log(ge)));
    p.fin_o = (T)(be * exp((double)n_cycles * log(go)));
}

template <typename T, int NS, bool EDGE, bool COL, bool MW>
int launch_line(const LineParams<T>& p, cudaStream_t st) {
    const int threads = p.lines_per_block * p.n_warps * 32;
    const int64_t groups = ((int64_t)p.n_lines + p.lines_per_block - 1) / p.lines_per_block;
    // several warps per line: the grid strides over the lines (barrier state lives in the block)
    int64_t blocks = groups;
    if (MW) {
        const int64_t resident = (int64_t)sm_count() * ((sizeof(T) * NS >= 256 ? 256 : 512) / threads);
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
            break;
        case 64:      // rows of fp32, several warps per line only (launch_lines)
            if constexpr (sizeof(T) == 4) {
                if (!col && p.n_warps > 1)
                    return edge ? launch_line<T, 64, true, false, true>(p, st)
                                : launch_line<T, 64, false, false, true>(p, st);
            }
    }
    set_error("axis: no line kernel for this extent");
    return TS_EUNSUPPORTED;
}

// transposed strided lines: n = W * NS, W <= 16 warps; the largest NS (fewest warps at the barrier,
// as for line_shape)
struct TShape {
    int ns, warps;
    bool ok() const { return ns != 0; }
};
TShape tline_shape(int64_t n, int dtype) {
    const int ns_max = dtype == TS_F32 ? 32 : 16;
    for (int ns = ns_max; ns >= 2; ns /= 2)
        if (n % ns == 0 && n / ns <= kTWarps) return {ns, (int)(n / ns)};
    return {0, 0};
}
template <typename T, int NS>
int launch_tline_ns(const LineParams<T>& p, bool edge, cudaStream_t st) {
    const int64_t groups = ((int64_t)p.n_lines + 31) / 32;
    const int64_t resident = (int64_t)sm_count() * ((kTWarps * 32) / (p.n_warps * 32));
    const unsigned blocks = (unsigned)(groups < resident ? groups : resident);
    if (edge) tline_kernel<T, NS, true><<<blocks, p.n_warps * 32, 0, st>>>(p);
    else tline_kernel<T, NS, false><<<blocks, p.n_warps * 32, 0, st>>>(p);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}
template <typename T>
int launch_tline(const LineParams<T>& p, int ns, bool edge, cudaStream_t st) {
    switch (ns) {
        case 2: return launch_tline_ns<T, 2>(p, edge, st);
        case 4: return launch_tline_ns<T, 4>(p, edge, st);
        case 8: return launch_tline_ns<T, 8>(p, edge, st);
        case 16: return launch_tline_ns<T, 16>(p, edge, st);
        case 32:
            if constexpr (sizeof(T) == 4) return launch_tline_ns<T, 32>(p, edge, st);
    }
    set_error("axis: no transposed line kernel for this extent");
    return TS_EUNSUPPORTED;
}

// Where the lines of one launch lie: line l = group g = l / lines_inner, member m = l % lines_inner
// starts at g * group_stride + m * line_stride; consecutive sites are site_stride apart.
struct LineGeom {
    int64_t n_sites;
    int periodic;
    int64_t n_lines, line_stride, site_stride, lines_inner, group_stride;
    bool col;              // site_stride != 1: scalar accesses, adjacent lines in one block
    bool transposed;       // strided lines of a state that does not stay in L2: one lane per line
};
LineGeom rows_of(const LatticeDesc& L) {
    return LineGeom{L.nx, L.periodic_x, L.ny, L.nx, 1, L.ny, 0, false, false};
}
LineGeom cols_of(const LatticeDesc& L) {
    return LineGeom{L.ny, L.periodic_y, L.nx, 1, L.nx, L.nx, 0, true, false};
}

// launch the line kernel on lines held completely in registers; p carries a chain (fill_chain) or
// a sweep program (fill_prog)
template <typename T>
int launch_lines(const LineGeom& g, int dtype, LineParams<T>& p, T* re, T* im, cudaStream_t st,
                 T* out_re = nullptr, T* out_im = nullptr) {
    p.src_re = re; p.src_im = im;
    p.dst_re = out_re ? out_re : re; p.dst_im = out_im ? out_im : im;
    p.n_lines = (int)g.n_lines;
    p.n_sites = (int)g.n_sites;
    p.line_stride = g.line_stride;
    p.site_stride = g.site_stride;
    p.lines_inner = (int)g.lines_inner;
    p.group_stride = g.group_stride;
    p.periodic = g.periodic;
    if (g.transposed) {
        const TShape ts_ = tline_shape(g.n_sites, dtype);
        if (ts_.ok()) {
            p.n_warps = ts_.warps; p.n_lanes = 32; p.lines_per_block = 32;
            return launch_tline<T>(p, ts_.ns, !g.periodic, st);
        }
    }
    LineShape sh = line_shape(g.n_sites, dtype);
    if (!sh.ok()) { set_error("axis: line does not fit a thread block"); return TS_EUNSUPPORTED; }
    // fp32 rows of 4096 / 8192 sites: 64 sites per lane and half the warps -- the per-sub-step
    // cost of the exchange (~32 instructions per warp) is spread over twice the sites, at 255
    // registers, i.e. 8 warps per SM in whole lines of 2 or 4 warps.  Measured with the final
    // exchange (200 sub-steps, rows only, ms, 32 -> 64 sites per lane): 4096^2 0.549 -> 0.537 /
    // closed 0.582 -> 0.541, 8192^2 2.20 -> 2.13 / closed 2.31 -> 2.13; NOT for rows of 16384 (one
    // line of 8 warps per SM cannot hide its own barrier: closed 8.57 -> 8.75; periodic, with the
    // earlier exchange, 8.53 -> 8.86) nor
    // where the warps do not fill the SM (12288: 1.76 -> 2.12).
    static const bool ns64 = getenv("TS_PROBE_NO_NS64") == nullptr;
    if (ns64 && !g.col && dtype == TS_F32 && sh.ns == 32 && (sh.warps == 4 || sh.warps == 8)) {
        sh.ns = 64;
        sh.warps /= 2;
    }
    p.n_lanes = sh.lanes;
    p.n_warps = sh.warps;
    if (sh.warps == 1) {
        // 4 lines per block (adjacent columns share their 32-byte sectors)
        p.lines_per_block = 4;
        const int64_t want = ((int64_t)p.n_lines + sm_count() * 4 - 1) / (sm_count() * 4);
        if (want < 4) p.lines_per_block = want < 1 ? 1 : (int)want;
    } else {
        p.lines_per_block = 1;
        if (sh.warps <= 8) p.lines_per_block = 4 / sh.warps > 1 ? 4 / sh.warps : 1;
    }
    const bool edge = !g.periodic || sh.lanes < 32;
    return launch_line_t<T>(p, sh.ns, edge, g.col, st);
}

// One launch of the line kernel: ALL n_sub sub-steps of the pattern along the rows (col = false)
// or the columns, in place.
template <typename T>
int line_pass(const LatticeDesc& L, T* re, T* im, const StepCoef* pat, int period, int64_t n_sub,
              bool col, cudaStream_t st, T* out_re = nullptr, T* out_im = nullptr) {
    LineParams<T> p = {};
    fill_chain(p, pat, period, 0, n_sub, col);
    return launch_lines<T>(col ? cols_of(L) : rows_of(L), L.dtype, p, re, im, st, out_re, out_im);
}

// Constants of a sweep program: sweeps (parity, angle) applied in order, scales followed as in
// fill_chain; phase planes (or null) multiplied in after the last sweep.
struct ProgStep {
    int parity;
    Angle a;
};
template <typename T>
void fill_prog(LineParams<T>& p, const ProgStep* steps, int n, const T* ph_re, const T* ph_im) {
    double al = 1.0, be = 1.0;
    p.n_prog = n;
    p.n_sub = 0; p.n_tab = 1;
    for (int i = 0; i < n; ++i) {
        const Angle& a = steps[i].a;
        const double t = a.s / a.c;
        SubCoef<T> sc = {};
        p.prog_parity[i] = steps[i].parity;
        if (steps[i].parity == 0) {
            const double rho = be / al;
            sc.e1 = (T)(t * rho);
            sc.e2 = (T)(t * a.c * a.c / rho);
            al *= a.c; be /= a.c;
        } else {
            const double rho = al / be;
            const double cm1 = -(a.s * a.s) / (1.0 + a.c);
            sc.o1 = (T)(t * rho);
            sc.o2 = (T)(t * a.c * a.c / rho);
            sc.od2 = (T)(-(a.s * a.s));
            sc.odc = (T)cm1;
            sc.ods = (T)(-cm1 / a.c);
            be *= a.c; al /= a.c;
        }
        p.prog[i] = sc;
    }
    p.fin_e = (T)al; p.fin_o = (T)be;
    p.ph_re = ph_re; p.ph_im = ph_im;
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
    p.lines_inner = p.n_lines;
    p.group_stride = 0;
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

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled() {
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess) {
            (void)cudaGetLastError();
            f = nullptr;
        }
        return (EncodeTiledFn)f;
    }();
    return fn;
}
// a plane [ny][nx] of T as a 2-D tensor, box = 32 columns x 2 rows
template <typename T>
int plane_map(CUtensorMap* m, const T* plane, int nx, int ny) {
    EncodeTiledFn enc = encode_tiled();
    if (!enc) { set_error("cuTensorMapEncodeTiled is not available from this driver"); return TS_ECUDA; }
    const cuuint64_t dims[2] = {(cuuint64_t)nx, (cuuint64_t)ny};
    const cuuint64_t strides[1] = {(cuuint64_t)nx * sizeof(T)};
    const cuuint32_t box[2] = {(cuuint32_t)kYCols, 2};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(m, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64,
                           2, const_cast<T*>(plane), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed"); return TS_ECUDA; }
    return TS_OK;
}

template <typename T, int S, bool PERY, bool UNI>
int launch_ycol(const YcolParams<T>& p, cudaStream_t st) {
    constexpr uint32_t SLOTB = 8 * kYCols * sizeof(T);
    const size_t smem = (size_t)kYWarps * p.nst * (SLOTB + 8);
    auto kern = ycol_kernel<T, S, PERY, UNI>;
    static std::atomic<size_t> configured[64];
    int dev = 0;
    TS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64 || smem > configured[dev].load(std::memory_order_relaxed)) {
        TS_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (dev >= 0 && dev < 64) configured[dev].store(smem, std::memory_order_relaxed);
    }
    const int n_seg = p.edge_rows > 0
                          ? 2 + (p.ny - 2 * p.edge_rows + p.seg_rows - 1) / p.seg_rows
                          : (p.ny + p.seg_rows - 1) / p.seg_rows;
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
    cfg.numAttrs = ((int64_t)grid.x * grid.y <= (int64_t)sm_count() * ycol_min_blocks<T, S, UNI>()) ? 1 : 0;
    alignas(64) CUtensorMap tm_re, tm_im;
    int rc = plane_map<T>(&tm_re, p.src_re, p.nx, p.ny);
    if (rc == TS_OK) rc = plane_map<T>(&tm_im, p.src_im, p.nx, p.ny);
    if (rc != TS_OK) return rc;
    TS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, p, tm_re, tm_im));
    return TS_OK;
}

template <typename T, int S>
int launch_ycol_s(const YcolParams<T>& p, bool uni, cudaStream_t st) {
    if (uni)
        return p.periodic_y ? launch_ycol<T, S, true, true>(p, st) : launch_ycol<T, S, false, true>(p, st);
    return p.periodic_y ? launch_ycol<T, S, true, false>(p, st) : launch_ycol<T, S, false, false>(p, st);
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
int ycol_blocks_per_sm(int S, int dtype, bool uni) { return ycol_blocks_for(S, dtype == TS_F32 ? 1 : 2, uni); }

// rows of the short first / last segment of a lattice that is closed in y (0: uniform segments):
// where the interior is worth several segments
constexpr int kEdgeRows = 128;
int ycol_edge_rows(const LatticeDesc& L, int seg_rows) {
    return (!L.periodic_y && L.ny >= 2 * kEdgeRows + 4 * (int64_t)seg_rows && seg_rows > kEdgeRows)
               ? kEdgeRows : 0;
}

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
    p.edge_rows = ycol_edge_rows(L, seg_rows);
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
    // S equal sub-steps and nothing padded: the coefficients are four pairs
    bool uni = n == S && S > 1;
    for (int j = 1; j < n && uni; ++j) uni = memcmp(&subs[j], &subs[0], sizeof(StepCoef)) == 0;
    if (uni) {
        p.u_open = p.te[0]; p.u_mid = p.te[1]; p.u_odd = p.to[0]; p.u_close = p.te[S];
        p.u_sec = p.sec_o[0];
    }
    switch (S) {
        case 4: return launch_ycol_s<T, 4>(p, uni, st);
        case 8: return launch_ycol_s<T, 8>(p, uni, st);
        case 12: return launch_ycol_s<T, 12>(p, uni, st);
        case 16: if constexpr (sizeof(T) == 4) return launch_ycol_s<T, 16>(p, uni, st); break;
        case 20: if constexpr (sizeof(T) == 4) return launch_ycol_s<T, 20>(p, uni, st); break;
        case 24: if constexpr (sizeof(T) == 4) return launch_ycol_s<T, 24>(p, uni, st); break;
    }
    set_error("axis: pipeline depth not instantiated");
    return TS_EINVAL;
}

// rows per segment of the column pipeline: a segment costs seg + 4S rows of work, so long
// segments win until the grid no longer fills the machine evenly.  Among the segment counts that
// give at most `cap` rows, take the one with the smallest makespan (waves of resident blocks x
// rows per block).
int ycol_default_seg(const LatticeDesc& L, int S, bool uni) {
    const int64_t strips = (L.nx + kYCols - 1) / kYCols;
    const int64_t blocks_x = (strips + kYWarps - 1) / kYWarps;
    const int64_t slots = (int64_t)sm_count() * ycol_blocks_per_sm(S, L.dtype, uni);
    const int64_t cap = 4096;
    int64_t best_seg = L.ny, best_cost = -1;
    for (int64_t segs = 1; segs <= L.ny / 2; ++segs) {
        int64_t r = (L.ny + segs - 1) / segs;
        r += r % 2;
        if (r < 16 && segs > 1) break;
        if (r > cap) continue;
        // closed lattices: two short edge segments besides the interior ones; a block of theirs is
        // the fraction 1.5 (e + 4S) / (r + 4S) of an interior block (the edge variant of the loop
        // costs about half as much again per row).  Without them the first and last segment run
        // the edge variant as a whole.
        const int64_t e = ycol_edge_rows(L, (int)r);
        const int64_t n_seg = e ? 2 + (L.ny - 2 * e + r - 1) / r : (L.ny + r - 1) / r;
        double eff = (double)n_seg * blocks_x;
        if (e) eff += 2.0 * blocks_x * (1.5 * (e + 4 * S) / (double)(r + 4 * S) - 1.0);
        const int64_t waves = (int64_t)ceil(eff / (double)slots - 1e-9);
        const int64_t cost = waves * (r + 4 * S) * ((!L.periodic_y && e == 0) ? 3 : 2);
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
                         int nst, cudaStream_t st, AxisInfo* info, LaunchTimer* tm,
                         const RowFeed* feed) {
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
    // ---- the windowed / pipelined passes of this call (out of place, ping-pong)
    struct Pass { int s, S; };
    std::vector<Pass> ypasses;
    int x_chain = 0;
    int64_t n_xpass = 0;
    if (!x_res) {
        x_chain = chain < kMaxChain ? chain : kMaxChain;
        n_xpass = (n_sub + x_chain - 1) / x_chain;
    }
    if (!y_res) {
        const int smax = ycol_depth(kMaxChain, L.dtype);
        int want = (int)(n_sub < chain ? n_sub : chain);
        if (want > smax) want = smax;
        for (int64_t i = 0; i < n_sub;) {
            Pass ps;
            if (period == 1) {
                // uniform steps: passes of exactly an instantiated depth run on the kernel whose
                // coefficients stay in uniform registers (200 = 8 x 24 + 8); what is left below
                // the smallest depth is one padded pass
                const int64_t left = n_sub - i;
                const int cap = (int)(left < want ? left : want);
                ps.S = ycol_depth(cap, L.dtype);
                if (ps.S > cap && cap >= 4) ps.S = cap / 4 * 4;       // depths are the multiples of 4
                ps.s = ps.S < cap ? ps.S : cap;
            } else {
                // equal passes: 200 sub-steps at depth 24 are 9 passes of 22 or 23
                const int64_t n_pass = (n_sub + want - 1) / want;
                const int per_pass = (int)((n_sub + n_pass - 1) / n_pass);
                ps.S = ycol_depth(per_pass, L.dtype);
                ps.s = (int)(n_sub - i < per_pass ? n_sub - i : per_pass);
            }
            ypasses.push_back(ps);
            i += ps.s;
        }
    }
    // a resident-line launch works in place or, for free, into the other buffer: it takes the odd
    // flip when the out-of-place passes are odd in number, so that the result lands in the caller's
    // planes without a final copy
    const bool odd_flips = ((n_xpass + (int64_t)ypasses.size()) & 1) != 0;
    // ---- rows
    if (x_res) {
        const bool flip_here = odd_flips;
        if (feed && feed->n > 1) {
            // rows are independent lines: one launch per piece of the feed, each after its copy
            int64_t y0 = 0;
            for (int k = 0; k < feed->n; ++k) {
                const int64_t y1 = feed->y_end[k];
                TS_CUDA_TRY(cudaStreamWaitEvent(st, feed->ready[k], 0));
                if (y1 > y0) {
                    LatticeDesc Lk = L;
                    Lk.ny = y1 - y0;
                    const int64_t off = y0 * L.nx;
                    timer_begin(tm, kKindLineRows, st);
                    rc = line_pass<T>(Lk, cur_re + off, cur_im + off, pat, period, n_sub, false, st,
                                      flip_here ? nxt_re + off : nullptr,
                                      flip_here ? nxt_im + off : nullptr);
                    timer_end(tm, st);
                    if (rc != TS_OK) return rc;
                    ++info->launches;
                }
                y0 = y1;
            }
        } else {
            if (feed && feed->n == 1) TS_CUDA_TRY(cudaStreamWaitEvent(st, feed->ready[0], 0));
            timer_begin(tm, kKindLineRows, st);
            rc = line_pass<T>(L, cur_re, cur_im, pat, period, n_sub, false, st,
                              flip_here ? nxt_re : nullptr, flip_here ? nxt_im : nullptr);
            timer_end(tm, st);
            if (rc != TS_OK) return rc;
            ++info->launches;
        }
        if (flip_here) flip();
        ++info->passes;
        info->chain_x = n_sub;
    } else {
        for (int64_t i = 0; i < n_sub; i += x_chain) {
            const int64_t s = n_sub - i < x_chain ? n_sub - i : x_chain;
            timer_begin(tm, kKindXwin, st);
            rc = xwin_pass<T>(L, cur_re, cur_im, nxt_re, nxt_im, pat, period, i, s, st);
            timer_end(tm, st);
            if (rc != TS_OK) return rc;
            flip();
            ++info->passes; ++info->launches;
        }
        info->chain_x = x_chain;
    }
    // ---- columns
    if (y_res) {
        const bool flip_here = odd_flips && !x_res;
        timer_begin(tm, kKindLineCols, st);
        rc = line_pass<T>(L, cur_re, cur_im, pat, period, n_sub, true, st,
                          flip_here ? nxt_re : nullptr, flip_here ? nxt_im : nullptr);
        timer_end(tm, st);
        if (rc != TS_OK) return rc;
        if (flip_here) flip();
        ++info->passes; ++info->launches;
        info->chain_y = n_sub;
    } else {
        // ring slots per warp: at least 3 (iteration i+2 is waited for while slot i-1 is the one
        // being refilled), at most what 200 KB of shared memory per block hold
        // (nst counts row pairs, as for the tile kernel; a ring slot holds two)
        int slots = nst >= 3 ? (nst + 1) / 2 : (nst > 0 ? 2 : 4);
        const int slot_max = (int)((200 << 10) / (kYWarps * (8 * kYCols * sizeof(T) + 8)));
        if (slots > slot_max) slots = slot_max;
        StepCoef subs[kMaxChain];
        int64_t i = 0;
        for (size_t k = 0; k < ypasses.size(); ++k) {
            const int s = ypasses[k].s, S = ypasses[k].S;
            for (int j = 0; j < s; ++j) subs[j] = pat[(i + j) % period];
            const bool uni = period == 1 && s == S && S > 1;
            const int seg = seg_rows > 0 ? seg_rows : ycol_default_seg(L, S, uni);
            timer_begin(tm, kKindYcol, st);
            rc = ycol_pass<T>(L, cur_re, cur_im, nxt_re, nxt_im, subs, s, S, seg, slots, st);
            timer_end(tm, st);
            if (rc != TS_OK) return rc;
            flip();
            ++info->passes; ++info->launches;
            if (k == 0) { info->chain_y = s; info->seg_rows = seg; }
            i += s;
        }
    }
    if (cur_re != psi_re) {
        const size_t plane_bytes = (size_t)L.nx * (size_t)L.ny * sizeof(T);
        timer_begin(tm, kKindCopy, st);
        TS_CUDA_TRY(cudaMemcpyAsync(psi_re, cur_re, plane_bytes, cudaMemcpyDeviceToDevice, st));
        TS_CUDA_TRY(cudaMemcpyAsync(psi_im, cur_im, plane_bytes, cudaMemcpyDeviceToDevice, st));
        timer_end(tm, st);
        info->launches += 2;
    }
    return TS_OK;
}

bool axis_needs_scratch(const LatticeDesc& L) {
    return !line_shape(L.nx, L.dtype).ok() || !column_resident(L);
}

int axis_evolve(const LatticeDesc& L, void* psi_re, void* psi_im, void* scr_re, void* scr_im,
                const StepCoef* pat, int period, int64_t n_sub, int chain, int seg_rows, int nst,
                cudaStream_t st, AxisInfo* info, LaunchTimer* tm, const RowFeed* feed) {
    if (chain <= 0) chain = axis_default_chain(L);
    if (feed && !axis_takes_feed(L)) {       // windowed rows: whole lattice first
        if (feed->n > 0) TS_CUDA_TRY(cudaStreamWaitEvent(st, feed->ready[feed->n - 1], 0));
        feed = nullptr;
    }
    if (L.dtype == TS_F32)
        return axis_evolve_t<float>(L, (float*)psi_re, (float*)psi_im, (float*)scr_re,
                                    (float*)scr_im, pat, period, n_sub, chain, seg_rows, nst, st,
                                    info, tm, feed);
    return axis_evolve_t<double>(L, (double*)psi_re, (double*)psi_im, (double*)scr_re,
                                 (double*)scr_im, pat, period, n_sub, chain, seg_rows, nst, st,
                                 info, tm, feed);
}

bool axis_takes_feed(const LatticeDesc& L) { return line_shape(L.nx, L.dtype).ok(); }


// ---- three-dimensional lattices (ts_internal.h) -------------------------------------------------------
// psi[nz][ny][nx]: the step Xe Xo Ye Yo Ze [Zo | Zo P Zo] Ze Yo Ye Xo Xe.  Sweeps
// along different axes commute, so without a potential n steps are three chains (one launch per
// axis with every line resident in registers), and with one the sweeps between two applications of
// the phase regroup per axis into O(h) E(2h) O(h):
//   [X: E O] [Y: E O] [Z: E O, P]  { [X: O E O] [Y: O E O] [Z: O E O, P] }^(n-1)  [Z: O E] [Y: O E] [X: O E]
// -- three launches per step, 16 B per site each (+ 8 B phase on the z launch, fp32) instead of
// thirteen sweeps.
namespace {
LineGeom geom3(const Lattice3& L, int axis) {
    const int64_t plane = L.nx * L.ny;
    if (axis == 0) return LineGeom{L.nx, L.per[0], L.ny * L.nz, L.nx, 1, L.ny * L.nz, 0, false, false};
    if (axis == 1) return LineGeom{L.ny, L.per[1], L.nx * L.nz, 1, L.nx, L.nx, plane, true, true};
    return LineGeom{L.nz, L.per[2], plane, 1, plane, plane, 0, true, true};
}
const int kKindOfAxis[3] = {kKindLineRows, kKindLineCols, kKindLineZ};

template <typename T>
int axis3_evolve_t(const Lattice3& L, T* re, T* im, const StepCoef& c, const T* pot,
                   int64_t n_steps, cudaStream_t st, AxisInfo* info, LaunchTimer* tm) {
    info->passes = info->launches = 0;
    info->chain_x = info->chain_y = n_steps; info->seg_rows = 0;
    int rc;
    if (pot == nullptr) {
        for (int axis = 0; axis < 3; ++axis) {
            LineParams<T> p = {};
            fill_chain(p, &c, 1, 0, n_steps, /*innermost axis: the caller's full angle*/ axis == 2);
            timer_begin(tm, kKindOfAxis[axis], st);
            rc = launch_lines<T>(geom3(L, axis), L.dtype, p, re, im, st);
            timer_end(tm, st);
            if (rc != TS_OK) return rc;
            ++info->passes; ++info->launches;
        }
        return TS_OK;
    }
    const Angle h = half_of(c), f = add(h, h);
    const int64_t sites = L.nx * L.ny * L.nz;
    auto run = [&](int axis, const ProgStep* steps, int n, bool phase) -> int {
        LineParams<T> p = {};
        fill_prog<T>(p, steps, n, phase ? pot : nullptr, phase ? pot + sites : nullptr);
        timer_begin(tm, kKindOfAxis[axis], st);
        const int r = launch_lines<T>(geom3(L, axis), L.dtype, p, re, im, st);
        timer_end(tm, st);
        ++info->passes; ++info->launches;
        return r;
    };
    const ProgStep open[2] = {{0, h}, {1, h}};
    const ProgStep mid[3] = {{1, h}, {0, f}, {1, h}};
    const ProgStep close[2] = {{1, h}, {0, h}};
    for (int axis = 0; axis < 3; ++axis)
        if ((rc = run(axis, open, 2, axis == 2)) != TS_OK) return rc;
    for (int64_t s = 1; s < n_steps; ++s)
        for (int axis = 0; axis < 3; ++axis)
            if ((rc = run(axis, mid, 3, axis == 2)) != TS_OK) return rc;
    for (int axis = 2; axis >= 0; --axis)
        if ((rc = run(axis, close, 2, false)) != TS_OK) return rc;
    return TS_OK;
}
}  // namespace

bool axis3_supported(const Lattice3& L, const StepCoef& c) {
    const Angle h = half_of(c), f = add(h, h);
    if (!(c.a_h > 0.25 && c.a_f > 0.25 && f.c > 0.25)) return false;
    const int64_t n[3] = {L.nx, L.ny, L.nz};
    for (int a = 0; a < 3; ++a)
        if (n[a] < 2 || n[a] >= (int64_t(1) << 30) || !line_shape(n[a], L.dtype).ok()) return false;
    return L.nx * L.ny < (int64_t(1) << 31) && L.ny * L.nz < (int64_t(1) << 31) &&
           L.nx * L.nz < (int64_t(1) << 31);
}

int axis3_evolve(const Lattice3& L, void* re, void* im, const StepCoef& c, const void* pot,
                 int64_t n_steps, cudaStream_t st, AxisInfo* info, LaunchTimer* tm) {
    if (L.dtype == TS_F32)
        return axis3_evolve_t<float>(L, (float*)re, (float*)im, c, (const float*)pot, n_steps, st, info, tm);
    return axis3_evolve_t<double>(L, (double*)re, (double*)im, c, (const double*)pot, n_steps, st, info, tm);
}

}  // namespace ts
