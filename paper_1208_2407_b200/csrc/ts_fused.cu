// ts_fused.cu -- fused, temporally blocked second-order step: S full steps per pass over HBM.
//
// Design: the lattice is cut into column strips of 128 sites, one
// WARP per strip and y-segment.  A lane owns 4 consecutive sites of a row (one 128-bit load for
// fp32), so X-even pairs (0,1),(2,3) and the X-odd pair (1,2) are in-thread and the X-odd pair
// (3,0') is one warp shuffle with the neighbouring lane.  The warp STREAMS down its strip two
// rows at a time; the vertical sweeps of S chained steps run as an S-stage register pipeline
// (each stage holds two rows), so a row is read from HBM once and written once per S steps and
// there is no halo recomputation in y apart from 2S warm-up rows per segment.  The strip carries
// a halo of 2S sites (rounded to 4) per side in x, recomputed redundantly and discarded -- the
// block + halo idea of PAPER.md:115 -- and results go to the other buffer.
//
// Arithmetic form: every rotation [[a, i b],[i b, a]] is applied as
// a * [[1, i t],[i t, 1]] with t = b/a; the common factors a are collected into one
// multiplication at the store.  This halves the FMA count (2 per site per sweep) and keeps
// a^2 (1 + t^2) = 1 to rounding.  At closed edges an unpaired site is instead multiplied by 1/a
// of that sweep so that the deferred factor stays uniform.
#include <math.h>

#include "ts_internal.h"
#include "ts_rows.cuh"

namespace ts {
namespace {

using namespace rows;

constexpr int kWarpsPerBlock = 4;

template <typename T>
struct FusedParams {
    const T* src_re;
    const T* src_im;
    T* dst_re;
    T* dst_im;
    const T* pot_re;
    const T* pot_im;
    int nx, ny;
    int n_strips;   // strips across x
    int wi;         // interior sites per strip = 128 - 2*halo
    int halo;       // 4 (S <= 2) or 8
    int seg_rows;   // output rows per segment (even)
    T t_h, t_f;     // tan(theta/2), tan(theta)
    T sec_h, sec_f; // 1/cos of the same
    T out_scale;    // product of all deferred cos factors of one pass
};


// Per-thread constants of one (strip, segment) work unit.
template <typename T>
struct LaneCtx {
    int xl;         // column of the lane's first site used for loads (wrapped when periodic)
    bool xvalid;    // the lane's four sites exist (always true when periodic)
    bool xedge;     // warp-uniform: this strip touches a closed edge in x
    XEdge<T> e;
};

// Load rows y and y+1 (y even) of the source into r0, r1; rows/columns outside a closed lattice
// read as zero (ghost sites), periodic ones wrap.
template <typename T, bool PER>
__device__ __forceinline__ void load_pair(const FusedParams<T>& p, const LaneCtx<T>& c, int y,
                                          Row4<T>& r0, Row4<T>& r1) {
    int yl = y;
    bool ok = c.xvalid;
    if (PER) yl = wrap_index(y, p.ny);
    else ok = ok && (y >= 0) && (y < p.ny);
    if (ok) {
        const int64_t off = (int64_t)yl * p.nx + c.xl;
        ld4(p.src_re + off, r0.re);
        ld4(p.src_im + off, r0.im);
        ld4(p.src_re + off + p.nx, r1.re);
        ld4(p.src_im + off + p.nx, r1.im);
    } else {
        zero_row(r0);
        zero_row(r1);
    }
}

// potential phase on row y (skipped on ghost rows, which hold zeros)
template <typename T, bool PER>
__device__ __forceinline__ void apply_pot(const FusedParams<T>& p, const LaneCtx<T>& c, int y,
                                          Row4<T>& r) {
    int yl = y;
    bool ok = c.xvalid;
    if (PER) yl = wrap_index(y, p.ny);
    else ok = ok && (y >= 0) && (y < p.ny);
    if (ok) {
        T pr[4], pi[4];
        const int64_t off = (int64_t)yl * p.nx + c.xl;
        ld4(p.pot_re + off, pr);
        ld4(p.pot_im + off, pi);
        phase_row(r, pr, pi);
    }
}

template <typename T>
__device__ __forceinline__ void xo_any(Row4<T>& r, T t, const LaneCtx<T>& c) {
    if (c.xedge) xo<T, true>(r, t, c.e);
    else xo<T, false>(r, t, c.e);
}

// One full second-order step on the streaming pipeline.
//   in : (r0, r1) = rows (yj, yj+1) before the step; g = row yj-2 and h = row yj-1 in mid-step
//        state (g: vertical-odd done, h: vertical-even done, waiting for its odd partner yj).
//   out: (r0, r1) = rows (yj-2, yj-1) after the step; g, h = rows (yj, yj+1) in mid-step state.
// Stage list per row pair follows include/ts.h: Xe Xo Ye [Yo | Yo P Yo] Ye Xo Xe.
template <typename T, bool POT, bool PER>
__device__ __forceinline__ void step_stage(const FusedParams<T>& p, const LaneCtx<T>& c, int yj,
                                           Row4<T>& r0, Row4<T>& r1, Row4<T>& g, Row4<T>& h) {
    xe(r0, p.t_h); xe(r1, p.t_h);
    xo_any(r0, p.t_h, c); xo_any(r1, p.t_h, c);
    ypair(r0, r1, p.t_h);                                  // Ye on (yj, yj+1)
    // Yo on (yj-1, yj) = (h, r0)
    const bool yedge = !PER && (yj == 0 || yj == p.ny);    // the pair straddles a closed edge
    if (!POT) {
        if (yedge) {
            // unpaired real row: 1/a_f; the ghost row stays zero
            if (yj == 0) scale_row(r0, p.sec_f); else scale_row(h, p.sec_f);
        } else {
            ypair(h, r0, p.t_f);
        }
    } else {
        if (yedge) {
            if (yj == 0) scale_row(r0, p.sec_h * p.sec_h); else scale_row(h, p.sec_h * p.sec_h);
        } else {
            ypair(h, r0, p.t_h);
        }
        apply_pot<T, PER>(p, c, yj - 1, h);
        apply_pot<T, PER>(p, c, yj, r0);
        if (!yedge) ypair(h, r0, p.t_h);
    }
    ypair(g, h, p.t_h);                                    // Ye on (yj-2, yj-1)
    xo_any(g, p.t_h, c); xo_any(h, p.t_h, c);
    xe(g, p.t_h); xe(h, p.t_h);
    // rotate roles: finished rows leave through (r0, r1); (yj, yj+1) become the held rows
    const Row4<T> og = g, oh = h;
    g = r0; h = r1;
    r0 = og; r1 = oh;
}

template <typename T, int S, bool POT, bool PER, int D>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
fused_kernel(const FusedParams<T> p) {
    const int lane = threadIdx.x & 31;
    const int strip = blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
    if (strip >= p.n_strips) return;

    const int x0 = strip * p.wi;              // first interior column of the strip
    const int xb = x0 - p.halo + 4 * lane;    // lane's first site, may be outside the lattice
    LaneCtx<T> c;
    c.xl = PER ? wrap_index(xb, p.nx) : xb;
    c.xvalid = PER ? true : (xb >= 0 && xb < p.nx);
    c.xedge = !PER && (x0 - p.halo < 0 || x0 - p.halo + kStripSites > p.nx);
    c.e.t_up = (xb == 0 || xb == p.nx) ? T(0) : p.t_h;
    c.e.t_dn = (xb + 4 == p.nx || xb + 4 == 0) ? T(0) : p.t_h;
    c.e.c0 = (xb == 0) ? p.sec_h : T(1);
    c.e.c3 = (xb + 4 == p.nx) ? p.sec_h : T(1);
    const bool store_ok = (4 * lane >= p.halo) && (4 * lane < kStripSites - p.halo) && (xb < p.nx);

    const int y_out0 = blockIdx.y * p.seg_rows;
    const int y_out1 = min(y_out0 + p.seg_rows, p.ny);
    const int y_in0 = y_out0 - 2 * S;
    const int n_iter = (y_out1 - y_out0) / 2 + 2 * S;

    Row4<T> g[S], h[S];
#pragma unroll
    for (int j = 0; j < S; ++j) { zero_row(g[j]); zero_row(h[j]); }

    Row4<T> n0[D], n1[D];
#pragma unroll
    for (int d = 0; d < D; ++d) {
        if (d < n_iter) load_pair<T, PER>(p, c, y_in0 + 2 * d, n0[d], n1[d]);
        else { zero_row(n0[d]); zero_row(n1[d]); }
    }

    for (int it0 = 0; it0 < n_iter; it0 += D) {
#pragma unroll
        for (int d = 0; d < D; ++d) {
            const int it = it0 + d;
            if (it < n_iter) {
                const int y = y_in0 + 2 * it;
                Row4<T> r0 = n0[d], r1 = n1[d];
                if (it + D < n_iter) load_pair<T, PER>(p, c, y + 2 * D, n0[d], n1[d]);
#pragma unroll
                for (int j = 0; j < S; ++j)
                    step_stage<T, POT, PER>(p, c, y - 2 * j, r0, r1, g[j], h[j]);
                if (it >= 2 * S && store_ok) {
                    const int64_t off = (int64_t)(y - 2 * S) * p.nx + xb;
                    st4(p.dst_re + off, r0.re, p.out_scale);
                    st4(p.dst_im + off, r0.im, p.out_scale);
                    st4(p.dst_re + off + p.nx, r1.re, p.out_scale);
                    st4(p.dst_im + off + p.nx, r1.im, p.out_scale);
                }
            }
        }
    }
}

constexpr int kPrefetchDepth = 2;   // row pairs in flight per lane beyond the one being computed

template <typename T, int S, bool POT, bool PER>
int launch(const FusedParams<T>& p, cudaStream_t st) {
    const int n_seg = (p.ny + p.seg_rows - 1) / p.seg_rows;
    dim3 grid((p.n_strips + kWarpsPerBlock - 1) / kWarpsPerBlock, n_seg);
    fused_kernel<T, S, POT, PER, kPrefetchDepth><<<grid, kWarpsPerBlock * 32, 0, st>>>(p);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}

template <typename T, int S>
int launch_s(const FusedParams<T>& p, bool pot, bool per, cudaStream_t st) {
    if (pot) return per ? launch<T, S, true, true>(p, st) : launch<T, S, true, false>(p, st);
    return per ? launch<T, S, false, true>(p, st) : launch<T, S, false, false>(p, st);
}

template <typename T>
int pass_t(const LatticeDesc& L, const T* src_re, const T* src_im, T* dst_re, T* dst_im,
           const StepCoef& c, const T* pot, int S, int seg_rows, cudaStream_t st) {
    FusedParams<T> p;
    p.src_re = src_re; p.src_im = src_im; p.dst_re = dst_re; p.dst_im = dst_im;
    p.pot_re = pot;
    p.pot_im = pot ? pot + L.nx * L.ny : nullptr;
    p.nx = (int)L.nx; p.ny = (int)L.ny;
    p.halo = (2 * S + 3) / 4 * 4;
    p.wi = kStripSites - 2 * p.halo;
    p.n_strips = (int)((L.nx + p.wi - 1) / p.wi);
    p.seg_rows = seg_rows;
    p.t_h = (T)(c.b_h / c.a_h);
    p.t_f = (T)(c.b_f / c.a_f);
    p.sec_h = (T)(1.0 / c.a_h);
    p.sec_f = (T)(1.0 / c.a_f);
    // deferred cos factors of one step: 6 half sweeps + the full one, or 8 half sweeps
    const double per_step = pot ? pow(c.a_h, 8) : pow(c.a_h, 6) * c.a_f;
    p.out_scale = (T)pow(per_step, S);
    const bool per = L.periodic_x != 0;
    switch (S) {
        case 1: return launch_s<T, 1>(p, pot != nullptr, per, st);
        case 2: return launch_s<T, 2>(p, pot != nullptr, per, st);
        case 3: return launch_s<T, 3>(p, pot != nullptr, per, st);
        case 4: return launch_s<T, 4>(p, pot != nullptr, per, st);
    }
    set_error("fused_pass: steps per pass out of range");
    return TS_EINVAL;
}

}  // namespace

bool fused_shape_ok(const LatticeDesc& L, const StepCoef& c) {
    // 128-bit row accesses need nx % 4 == 0; the row-pair pipeline needs even ny; the tangent
    // form needs cos well away from zero; 32-bit row/column indices inside the kernel.
    return L.nx % 4 == 0 && L.ny % 2 == 0 && L.nx >= 4 && L.ny >= 2 &&
           L.nx < (1 << 30) && L.ny < (1 << 30) && c.a_h > 0.25 && c.a_f > 0.25 &&
           c.a_h * c.a_h - c.b_h * c.b_h > 0.25;   // two half sweeps merged into one
}

bool fused_supported(const LatticeDesc& L, const StepCoef& c) {
    return fused_shape_ok(L, c) && L.periodic_x == L.periodic_y;
}

int fused_default_seg_rows(const LatticeDesc& L, int S, int blocks_per_sm) {
    // One warp per (strip, segment), 4 strips per block; a segment recomputes 2S warm-up row pairs,
    // so its cost is seg/2 + 2S iterations: longer segments win until the grid no longer fills the
    // machine.  Pick the number of waves the cap on the segment height allows (256 rows, 512 for
    // S >= 5: round-1 probes), then the segment count that fills those waves and no more -- a grid of
    // 1.1 waves costs two (4096^2: 490 blocks on 444 slots ran at 60 % of the 16384^2 rate).
    const int halo = (2 * S + 3) / 4 * 4;
    const int64_t strips = (L.nx + (kStripSites - 2 * halo) - 1) / (kStripSites - 2 * halo);
    const int64_t blocks_x = (strips + 3) / 4;
    const int64_t slots = 148 * (int64_t)(blocks_per_sm > 0 ? blocks_per_sm : 3);
    const int64_t cap = S >= 5 ? 512 : 256;
    const int64_t min_segs = (L.ny + cap - 1) / cap;
    int64_t waves = (min_segs * blocks_x + slots - 1) / slots;
    if (waves < 1) waves = 1;
    int64_t segs = waves * slots / blocks_x;
    if (segs < 1) segs = 1;
    int64_t r = (L.ny + segs - 1) / segs;
    r += r % 2;
    if (r > cap) r = cap;
    if (r < 8) r = 8;     // small lattices: parallelism over warm-up redundancy
    if (r > L.ny) r = L.ny;
    return (int)r;
}

int fused_default_steps(const LatticeDesc& L, bool pot) {
    // steps fused per pass, measured on B200 (round-1 probes): fp32 without potential 6
    // (regrouped sweeps, packed FMAs; ts_evolve clamps to what the chosen kernel has) -- 4 on
    // small lattices (below 8 M sites), where segments are short and the 2S warm-up iterations dominate; fp32 with
    // potential 3; fp64 3 with, 4 without.
    if (L.dtype == TS_F32) {
        if (pot) return 3;
        return L.nx * L.ny < (int64_t(1) << 23) ? 4 : 6;
    }
    return pot ? 3 : 4;
}

int fused_pass(const LatticeDesc& L, const void* src_re, const void* src_im, void* dst_re,
               void* dst_im, const StepCoef& c, const void* pot, int S, int seg_rows,
               cudaStream_t st) {
    if (seg_rows <= 0 || seg_rows % 2) {
        set_error("fused_pass: seg_rows must be positive and even");
        return TS_EINVAL;
    }
    if (L.dtype == TS_F32)
        return pass_t<float>(L, (const float*)src_re, (const float*)src_im, (float*)dst_re,
                             (float*)dst_im, c, (const float*)pot, S, seg_rows, st);
    return pass_t<double>(L, (const double*)src_re, (const double*)src_im, (double*)dst_re,
                          (double*)dst_im, c, (const double*)pot, S, seg_rows, st);
}

}  // namespace ts
