// ts_stream.cu -- fused streaming kernel v2: TMA bulk copies into a per-warp shared-memory ring.
//
// Same decomposition and arithmetic as ts_fused.cu (one warp per 128-site column strip and
// y-segment, 4 sites per lane, S chained steps as a register pipeline over row pairs), but the
// rows are brought on chip by cp.async.bulk (TMA, completion on an mbarrier) into a ring of NST
// row-pair slots owned by the warp, several iterations ahead of their use.  Global-load latency
// is therefore hidden by shared memory, not by registers, which removes the long-scoreboard
// stalls that bound v1 (round 1): registers only hold the S+1 row pairs of the pipeline.
// The register pipeline is unrolled over its rotation period S+1 so that rows never move between
// registers.  Potential-phase rows travel with the row pair (same copies batch, same mbarrier)
// but land in a ring of their own, where they are kept S+1 iterations longer, because stage j of
// the pipeline applies the phase to rows that arrived j iterations earlier.
//
// Results are written straight from registers with 128-bit stores into the other buffer
// (double buffering); halo columns of a strip are recomputed and discarded
// (PAPER.md:115).
#include <math.h>
#include <stdlib.h>

#include <atomic>
#include <type_traits>

#include "ts_internal.h"
#include "ts_rows.cuh"
#include "ts_tma.cuh"

namespace ts {
namespace {

using namespace rows;
using namespace tma;

constexpr int kWarps = 4;
constexpr int kMaxDevices = 64;


template <typename T>
struct StreamParams {
    const T* src_re;
    const T* src_im;
    T* dst_re;
    T* dst_im;
    const T* pot_re;      // phase planes [ny][nx] (phase mode 1)
    const T* pot_im;
    const T* px_re;       // separable phase (mode 2): P(x, y) = px(x) * py(y), px [nx], py [ny]
    const T* px_im;
    const T* py_re;
    const T* py_im;
    // row slab with peer halos (ts_slab_pass): rows above row 0 / below row ny-1 are read from
    // the neighbours' source planes (their last up_rows / first dn_rows rows; possibly another
    // GPU's memory over NVLink).  NULL = no neighbour: a real closed edge (or plain lattice).
    const T* up_re;
    const T* up_im;
    const T* dn_re;
    const T* dn_im;
    int up_rows, dn_rows;
    int edge_top, edge_bot;   // closed in y: row 0 / row ny-1 is a lattice edge (not a cut)
    int py_off, py_n, py_wrap;   // separable phase: global row of local row 0, global height, wrap
    int nx, ny;
    int n_strips, wi, halo, seg_rows, n_seg;
    // warps that run the closed-edge variant of the loop get shorter segments (seg_edge <=
    // seg_rows): the n_xe x-edge strips (first / last strip of a lattice closed in x; 0, 1 or 2)
    // are cut into n_seg_x segments of seg_edge rows; with y_short the first and the last segment
    // of every other strip are seg_edge rows high and the n_seg - 2 between them seg_rows
    int seg_edge, n_seg_x, n_xe, y_short;
    int nst;        // ring slots per warp (state row pairs)
    int nph;        // with phase planes: slots of the separate phase ring (>= prefetch + S + 1)
    // tangents of the sweeps of the S chained sub-steps of this pass (angles may differ from
    // sub-step to sub-step: Eq. 4 chains U2 with three different time fractions)
    T te[TS_MAX_FUSE + 1];   // even sweeps: te[0] opening half sweep, te[j] the merged sweep between
                             // sub-steps j-1 and j (half + half angle), te[S] the closing half sweep
    T to[TS_MAX_FUSE];       // Y-odd sweep of sub-step j: the caller's full-angle coefficients
                             // without potential; with one, every odd sweep at the half angle
    T sec_o[TS_MAX_FUSE];    // 1 / cos of that sweep (unpaired sites at closed edges)
    T tox[TS_MAX_FUSE];      // X-odd sweep without potential: the two half sweeps Xo(h) Xo(h) that
    T sec_ox[TS_MAX_FUSE];   // regrouping brings together, composed from the HALF coefficients
    T out_scale;             // product of all deferred cosines of the pass
};

template <typename T>
struct StreamCtx {
    bool xvalid;         // lane's sites exist (always when periodic)
    bool xedge;          // warp-uniform: strip touches a closed edge in x
    XCut e;              // where the lane's cross-lane X-odd pairs meet a closed edge
    T pxr[4], pxi[4];    // separable potential: phase factor of the lane's four columns
    uint32_t ring;       // shared address of the warp's slot ring
    uint32_t pot_ring;   // ... of its phase ring (phase planes only)
    uint32_t lane_off;   // byte offset of the lane's 4 sites inside a row chunk
};

// One second-order sub-step (stage J of S) of the register pipeline, WITH a potential.
//   in : (a0, a1) = rows (yj, yj+1) before the step; (g, h) = rows (yj-2, yj-1) in mid-step state
//   out: (g, h) = rows (yj-2, yj-1) after the step; (a0, a1) = rows (yj, yj+1) in mid-step state
// Between two chained sub-steps the closing Y-even, X-odd, X-even half sweeps of one and the
// opening X-even, X-odd, Y-even half sweeps of the next act on the same rows; X sweeps commute
// with Y sweeps, so the two X-even and the two Y-even half sweeps are each applied as ONE sweep
// by the sum of the two half angles (te[J]) in the later sub-step: 6 sweeps + P per sub-step
// instead of 8 + P.  The deferred cosines are accounted for in out_scale.
// pot_yj / pot_yjm1: shared addresses of the potential rows yj (row 0 of its slot) and yj-1
// (row 1 of the previous slot).
template <typename T, int PM, int BND, bool XEDGE, int S, int J>
__device__ __forceinline__ void stream_stage(const StreamParams<T>& p, const StreamCtx<T>& c,
                                             int yj, Row4<T>& a0, Row4<T>& a1, Row4<T>& g,
                                             Row4<T>& h, uint32_t pot_yj, uint32_t pot_yjm1) {
    constexpr uint32_t ROWB = kStripSites * sizeof(T);
    constexpr bool LAST = J == S - 1;
    const T th = p.to[J];
    xe(a0, p.te[J]); xe(a1, p.te[J]);
    xo<T, XEDGE>(a0, th, p.sec_o[J], c.e); xo<T, XEDGE>(a1, th, p.sec_o[J], c.e);
    // opening Y-even sweep, merged with the closing one of the previous sub-step (only X sweeps
    // lie between the two, and those commute with it)
    ypair(a0, a1, p.te[J]);
    // closed lattice: the vertical-odd pair (yj-1, yj) does not exist at yj = 0 and yj = ny; the
    // ghost row is zero and stays zero (coupling 0), the real row takes 1/a per omitted sweep
    constexpr bool SLAB = BND >= 3;      // row 0 / ny-1 may be a cut with a neighbour behind it
    const bool yedge = XEDGE && ((yj == 0 && (!SLAB || p.edge_top)) ||
                                 (yj == p.ny && (!SLAB || p.edge_bot)));
    const T t_yo = yedge ? T(0) : th;
    ypair(h, a0, t_yo);
    {
        const bool lo_ok = !XEDGE || (c.xvalid && yj - 1 >= 0 && yj - 1 < p.ny);
        const bool hi_ok = !XEDGE || (c.xvalid && yj >= 0 && yj < p.ny);
        if (PM == 2) {
            // separable: the row factors come through L1 (one address per warp), the column
            // factors sit in registers; ghost rows are zero, so any finite factor will do there
            // py is indexed by the GLOBAL row: py_off = first row of a slab (0 for a whole
            // lattice), py_n = global height, py_wrap = the global lattice is periodic in y
            int ylo = yj - 1 + p.py_off, yhi = yj + p.py_off;
            if (p.py_wrap) {   // warm-up rows reach 2S + 1 rows above row 0: further than a
                               // very short ring is long, hence the looped form
                ylo = wrap_index(ylo, p.py_n);
                yhi = wrap_index(yhi, p.py_n);
            }
            else { ylo = min(max(ylo, 0), p.py_n - 1); yhi = min(max(yhi, 0), p.py_n - 1); }
            sep_phase_row(h, c.pxr, c.pxi, __ldg(p.py_re + ylo), __ldg(p.py_im + ylo));
            sep_phase_row(a0, c.pxr, c.pxi, __ldg(p.py_re + yhi), __ldg(p.py_im + yhi));
        } else {
            if (lo_ok) {
                T pr[4], pi[4];
                lds4(pot_yjm1 + c.lane_off, pr);
                lds4(pot_yjm1 + ROWB + c.lane_off, pi);
                phase_row(h, pr, pi);
            }
            if (hi_ok) {
                T pr[4], pi[4];
                lds4(pot_yj + c.lane_off, pr);
                lds4(pot_yj + ROWB + c.lane_off, pi);
                phase_row(a0, pr, pi);
            }
        }
    }
    ypair(h, a0, t_yo);
    if (XEDGE) {
        const T sy = yedge ? p.sec_o[J] * p.sec_o[J] : T(1);
        scale_row(h, sy); scale_row(a0, sy);
    }
    if (LAST) ypair(g, h, p.te[S]);
    xo<T, XEDGE>(g, th, p.sec_o[J], c.e); xo<T, XEDGE>(h, th, p.sec_o[J], c.e);
    if (LAST) { xe(g, p.te[S]); xe(h, p.te[S]); }
}

// The same sub-step WITHOUT a potential, regrouped.  Horizontal sweeps act inside a row and
// vertical sweeps act along a column with the same scalar coefficients, so every X sweep commutes
// with every Y sweep (tensor-product structure; pinned on the oracle by test_xy_regrouping and on
// dense matrices by test_stage_order...).  The step Xe Xo Ye Yo(f) Ye Xo Xe therefore equals
// [Xe(h) Xo(f) Xe(h)] [Ye(h) Yo(f) Ye(h)], and across chained sub-steps the adjacent half sweeps
// merge: per pass  X: Xe(h0) Xo(f0) {Xe(h_{j-1} + h_j) Xo(f_j)}_{j=1..S-1} Xe(h_{S-1}),  Y: likewise.
// 4S+2 sweeps instead of 7S.  Only the rounding differs from the literal sequence.
//   in : (a0, a1) = rows (yj, yj+1) entering step; (g, h) = rows (yj-2, yj-1), h waiting for Yo
//   out: (g, h) finished with this step; (a0, a1) held for the next iteration
template <typename T, int BND, bool XEDGE, int S, int J>
__device__ __forceinline__ void stream_stage_nopot(const StreamParams<T>& p,
                                                   const StreamCtx<T>& c, int yj, Row4<T>& a0,
                                                   Row4<T>& a1, Row4<T>& g, Row4<T>& h) {
    constexpr bool LAST = J == S - 1;
    xe(a0, p.te[J]); xe(a1, p.te[J]);
    xo<T, XEDGE>(a0, p.tox[J], p.sec_ox[J], c.e); xo<T, XEDGE>(a1, p.tox[J], p.sec_ox[J], c.e);
    if (LAST) { xe(a0, p.te[S]); xe(a1, p.te[S]); }
    ypair(a0, a1, p.te[J]);
    // closed lattice: the vertical-odd pair (yj-1, yj) does not exist at yj = 0 and yj = ny; the
    // real row of the two takes 1/a instead (the ghost row is zero and stays zero)
    constexpr bool SLAB = BND >= 3;      // row 0 / ny-1 may be a cut with a neighbour behind it
    const bool yedge = XEDGE && ((yj == 0 && (!SLAB || p.edge_top)) ||
                                 (yj == p.ny && (!SLAB || p.edge_bot)));
    const T t_yo = yedge ? T(0) : p.to[J];
    ypair(h, a0, t_yo);
    if (XEDGE) { const T sy = yedge ? p.sec_o[J] : T(1); scale_row(h, sy); scale_row(a0, sy); }
    if (LAST) ypair(g, h, p.te[S]);
}

// stages 0..S-1 of one iteration: the pair (x0, x1) flows through them, see the kernel
template <typename T, int PM, int BND, bool XEDGE, int S, int J>
struct Stages {
    static __device__ __forceinline__ void run(const StreamParams<T>& p, const StreamCtx<T>& c,
                                               int y, int cs, int nst, uint32_t slotb,
                                               Row4<T> (&W)[S][2][2], const int u, Row4<T>& x0,
                                               Row4<T>& x1) {
        constexpr uint32_t ROWB = kStripSites * sizeof(T);
        Row4<T>& a0 = W[J][u][0];
        Row4<T>& a1 = W[J][u][1];
        Row4<T>& g = W[J][u ^ 1][0];
        Row4<T>& h = W[J][u ^ 1][1];
        a0 = x0; a1 = x1;
        if (PM == 1) {
            int s0 = cs - J;      if (s0 < 0) s0 += nst;
            int s1 = s0 - 1;      if (s1 < 0) s1 += nst;
            // cs / nst / slotb here: the PHASE ring's slot of this iteration, its length, 4 rows
            const uint32_t pot_yj = c.pot_ring + s0 * slotb;
            const uint32_t pot_yjm1 = c.pot_ring + s1 * slotb + 2 * ROWB;
            stream_stage<T, 1, BND, XEDGE, S, J>(p, c, y - 2 * J, a0, a1, g, h, pot_yj, pot_yjm1);
        } else if (PM == 2) {
            stream_stage<T, 2, BND, XEDGE, S, J>(p, c, y - 2 * J, a0, a1, g, h, 0, 0);
        } else {
            stream_stage_nopot<T, BND, XEDGE, S, J>(p, c, y - 2 * J, a0, a1, g, h);
        }
        x0 = g; x1 = h;   // (g, h) left the sub-step and flows on; (a0, a1) now waits in stage J
        if constexpr (J + 1 < S)
            Stages<T, PM, BND, XEDGE, S, J + 1>::run(p, c, y, cs, nst, slotb, W, u, x0, x1);
    }
};

template <typename T, int S, int PM, int BND, int MINB>
__global__ void __launch_bounds__(kWarps * 32, MINB)
stream_kernel(const StreamParams<T> p) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // BND: 0 = closed on both axes, 1 = periodic on both, 2 = periodic in x and closed in y (a row
    // slab with stored halos, paper_1208_2407_b200/slab.py); 3 / 4 = closed / periodic in x, and in y
    // a slab whose neighbours' rows are fetched in place (ts_slab_pass).  The peer logic is
    // compiled in only there: as run-time branches it cost the closed kernels 13-18 %.
    constexpr bool PERX = BND == 1 || BND == 2 || BND == 4, PERY = BND == 1, SLAB = BND >= 3;
    const bool edge_top = !SLAB || p.edge_top, edge_bot = !SLAB || p.edge_bot;
    // Phase planes travel through a ring of their OWN (r2): a state row pair is consumed in the
    // iteration it arrives, its phase rows are needed for S + 1 iterations (stage j applies P to
    // rows that arrived j iterations ago).  In one ring every slot was 8 rows and lived S + 1
    // iterations: 112 KB per block in fp32 at S = 3 (2 blocks per SM), 224 KB in fp64 (1 block).
    // Split, the state ring is prefetch + 1 slots of 4 rows and the phase ring prefetch + S + 1.
    constexpr bool POT = PM == 1;
    constexpr int R = 1;                      // iterations a state slot stays live after its arrival
    constexpr uint32_t ROWB = kStripSites * sizeof(T);
    constexpr int NROW = POT ? 8 : 4;         // copies per iteration: re0 im0 re1 im1 [pr0 pi0 pr1 pi1]
    constexpr uint32_t SLOTB = 4 * ROWB;      // a slot of either ring: four rows

    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // warp-uniform
    // (strip, segment) pairs are numbered strip-fastest and dealt to warps in order, so a block
    // may hold the last strips of one segment and the first of the next: no warp slot idles when
    // n_strips is not a multiple of kWarps (4096^2 at S = 3: 37 strips, 48 segments = 1776 warps,
    // exactly one wave of 444 blocks; with a grid of (10, 44) three warps in forty were empty and
    // every warp had 8 more rows).  Warps share nothing (own ring, own barriers).
    // Warps that run the closed-edge variant (about 8 % more per row) would end every pass late:
    // they get shorter segments (StreamParams::seg_edge), the x-edge strips first in the numbering.
    const int wid = blockIdx.x * kWarps + warp;
    int segi, strip;
    bool x_short = false;
    {
        const int we = p.n_xe * p.n_seg_x;
        if (wid < we) {
            const int k = wid / p.n_seg_x;
            segi = wid - k * p.n_seg_x;
            strip = k == 0 ? 0 : p.n_strips - 1;
            x_short = true;
        } else {
            const int ni = p.n_strips - p.n_xe;
            if (ni <= 0) return;
            const int w2 = wid - we;
            segi = w2 / ni;
            strip = (p.n_xe > 0 ? 1 : 0) + (w2 - segi * ni);
            if (segi >= p.n_seg) return;
        }
    }
    const int NST = p.nst;
    const int NPH = POT ? p.nph : 0;
    const int DIST = NST - R;                 // prefetch distance in iterations

    const int x0 = strip * p.wi;
    const int xs = x0 - p.halo;               // first column of the strip window
    const int xb = xs + 4 * lane;
    StreamCtx<T> c;
    c.xvalid = PERX ? true : (xb >= 0 && xb < p.nx);
    c.xedge = !PERX && (xs < 0 || xs + kStripSites > p.nx);
    c.e.up = !PERX && (xb == 0 || xb == p.nx);
    c.e.dn = !PERX && (xb + 4 == p.nx || xb + 4 == 0);
    c.ring = smem_u32(smem_raw) + warp * (NST + NPH) * SLOTB;
    c.pot_ring = c.ring + NST * SLOTB;
    c.lane_off = lane * 4 * sizeof(T);
    const uint32_t bars = smem_u32(smem_raw) + kWarps * (NST + NPH) * SLOTB + warp * NST * 8;
    const bool store_ok = (4 * lane >= p.halo) && (4 * lane < kStripSites - p.halo) && (xb < p.nx);

    // the strip window [xs, xs+128) as at most two contiguous global pieces (warp-uniform);
    // piece B (periodic wrap) always starts at global column 0
    int gx_a, off_a, len_a, len_b;
    if (PERX) {
        gx_a = wrap_index(xs, p.nx);
        off_a = 0;
        len_a = min(kStripSites, p.nx - gx_a);
        len_b = kStripSites - len_a;
    } else {
        gx_a = max(xs, 0);
        off_a = gx_a - xs;
        len_a = min(xs + kStripSites, p.nx) - gx_a;
        len_b = 0;
    }
    const uint32_t bytes_a = len_a * sizeof(T), bytes_b = len_b * sizeof(T);
    const uint32_t slot_tx = NROW * (bytes_a + bytes_b);
    const uint32_t dst_a = off_a * sizeof(T), dst_b = bytes_a;

    int y_out0, y_out1;
    if (x_short) {
        y_out0 = segi * p.seg_edge;
        y_out1 = min(y_out0 + p.seg_edge, p.ny);
    } else if (p.y_short) {
        if (segi == 0) { y_out0 = 0; y_out1 = p.seg_edge; }
        else if (segi == p.n_seg - 1) { y_out0 = p.ny - p.seg_edge; y_out1 = p.ny; }
        else {
            y_out0 = p.seg_edge + (segi - 1) * p.seg_rows;
            y_out1 = min(y_out0 + p.seg_rows, p.ny - p.seg_edge);
        }
    } else {
        y_out0 = segi * p.seg_rows;
        y_out1 = min(y_out0 + p.seg_rows, p.ny);
    }
    const int y_in0 = y_out0 - 2 * S;
    // even, so that the two-iteration loop body has no conditional half (the extra iteration only
    // feeds the pipeline; its output row pair lies beyond the segment and is not stored)
    const int n_iter = ((y_out1 - y_out0) / 2 + 2 * S + 1) & ~1;

    const bool leader = elect_one();
    if (leader) {
        for (int s = 0; s < NST; ++s) mbar_init(bars + 8 * s, 1);
        mbar_fence_init();
    }
    __syncwarp();
    // Programmatic dependent launch: the passes of one ts_evolve are launched with stream
    // serialisation relaxed, so this grid's blocks may be scheduled (and get here) while the
    // previous pass is still draining; no global memory has been read and nothing has been
    // written before this point (the separable phase vectors, too, are read after the wait: the
    // caller may have produced them with a kernel just before on the same stream).
    // griddepcontrol.wait returns once the previous grid has completed and its writes are visible;
    // launch_dependents lets the next pass start its own prologue as early as possible.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;");

    if (PM == 2) {
        // the lane's four columns (wrapped when periodic; 1 + 0i on ghost columns, which hold zeros)
        const int xw = PERX ? wrap_index(xb, p.nx) : xb;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const bool ok = PERX || (xb >= 0 && xb < p.nx);
            c.pxr[i] = ok ? __ldg(p.px_re + xw + i) : T(1);
            c.pxi[i] = ok ? __ldg(p.px_im + xw + i) : T(0);
        }
    }

    // running row of the next fetch (warp-uniform): rows (fy, fy+1), element offset foff
    int fy = PERY ? wrap_index(y_in0, p.ny) : y_in0;
    int64_t foff = (int64_t)fy * p.nx;
    const int64_t plane_elems = (int64_t)p.nx * p.ny;

    int fps = 0;                // phase-ring slot of the next fetch
    // fetch the next row pair into ring slot `slot` (one elected lane issues all copies)
    auto issue = [&](int slot) {
        // where the row pair lives: own planes -- or, beyond the slab, a neighbour's (ts_slab_pass)
        bool rowok = PERY ? true : (fy >= 0 && fy < p.ny);
        const T* b_re = p.src_re;
        const T* b_im = p.src_im;
        int64_t off = foff;
        if (SLAB && !rowok) {
            if (fy < 0) {
                rowok = p.up_re != nullptr && fy + p.up_rows >= 0;
                b_re = p.up_re; b_im = p.up_im;
                off = (int64_t)(fy + p.up_rows) * p.nx;
            } else {
                rowok = p.dn_re != nullptr && fy - p.ny + 2 <= p.dn_rows;
                b_re = p.dn_re; b_im = p.dn_im;
                off = (int64_t)(fy - p.ny) * p.nx;
            }
        }
        if (leader) {
            const uint32_t bar = bars + 8 * slot;
            if (rowok) {
                mbar_arrive_expect_tx(bar, slot_tx);
                const uint32_t dst = c.ring + slot * SLOTB;
                const T* planes[8] = {b_re, b_im, b_re, b_im,
                                      p.pot_re, p.pot_im, p.pot_re, p.pot_im};
                const uint32_t dst_p = c.pot_ring + fps * SLOTB;
#pragma unroll
                for (int r = 0; r < NROW; ++r) {
                    const T* row = planes[r] + (r < 4 ? off : foff) + ((r >> 1) & 1) * p.nx;
                    const uint32_t d = (r < 4 ? dst + r * ROWB : dst_p + (r - 4) * ROWB);
                    bulk_g2s(d + dst_a, row + gx_a, bytes_a, bar);
                    if (bytes_b) bulk_g2s(d + dst_b, row, bytes_b, bar);
                }
            } else {
                mbar_arrive(bar);
            }
        }
        fy += 2;
        foff += 2 * (int64_t)p.nx;
        if (PERY && fy >= p.ny) { fy -= p.ny; foff -= plane_elems; }
        if (POT && ++fps == NPH) fps = 0;
    };

    for (int k = 0; k < DIST; ++k)
        if (k < n_iter) issue(k);

    int cs = 0;                 // ring slot of the current iteration
    int ps = 0;                 // phase-ring slot of the current iteration
    uint32_t cph = 0;           // its mbarrier phase parity
    int rs = DIST % NST;        // ring slot refilled at the top of the current iteration

    // Ping-pong form of the pipeline.  Stage j owns two register sets W[j][0], W[j][1]: in an
    // even iteration the incoming pair is written to set 0 and the pair that waited there since
    // the previous iteration for its vertical-odd partner is set 1, in an odd iteration the other
    // way round.  The pair that leaves stage j is handed to stage j+1 by value (the copy folds
    // into the first sweep of that stage), and a set is dead once its pair has left, so S+1 pairs
    // are live, exactly as in a rotation over S+1 sets -- but the loop repeats after TWO iterations
    // instead of S+1: the S+1-fold unrolled rotation of r1b was 41 KB of SASS at S = 4 and
    // overflowed the instruction cache beyond (no_instruction stalls, round-1 captures).
    // The whole loop exists twice for closed lattices: warps whose strip touches an edge in x or
    // whose segment touches one in y (the outer ring of the warp grid) carry per-lane couplings,
    // zero ghost sites and the 1/a factor of unpaired sites (XEDGE, branch-free selects); all
    // others run the unmodified sweeps.  Chosen once per warp: no branch inside the sweeps.
    auto run = [&](auto xedge_tag) {
    constexpr bool XEDGE = decltype(xedge_tag)::value;
    Row4<T> W[S][2][2];
#pragma unroll
    for (int s = 0; s < S; ++s) {
        zero_row(W[s][0][0]); zero_row(W[s][0][1]); zero_row(W[s][1][0]); zero_row(W[s][1][1]);
    }

#pragma unroll 1
    for (int it0 = 0; it0 < n_iter; it0 += 2) {
        auto half = [&](auto utag) {
            constexpr int U = decltype(utag)::value;
            const int it = it0 + U;
            {
                __syncwarp();   // every lane is done with the slot about to be refilled
                if (it + DIST < n_iter) issue(rs);
                mbar_wait(bars + 8 * cs, cph);
                const int y = y_in0 + 2 * it;
                const bool rowok = !XEDGE || (c.xvalid && (y >= 0 || !edge_top) &&
                                              (y < p.ny || !edge_bot));
                Row4<T> x0, x1;
                if (rowok) {
                    const uint32_t base = c.ring + cs * SLOTB + c.lane_off;
                    lds4(base, x0.re);
                    lds4(base + ROWB, x0.im);
                    lds4(base + 2 * ROWB, x1.re);
                    lds4(base + 3 * ROWB, x1.im);
                } else {
                    zero_row(x0);
                    zero_row(x1);
                }
                if (POT) Stages<T, PM, BND, XEDGE, S, 0>::run(p, c, y, ps, NPH, SLOTB, W, U, x0, x1);
                else Stages<T, PM, BND, XEDGE, S, 0>::run(p, c, y, cs, NST, SLOTB, W, U, x0, x1);
                if (it >= 2 * S && store_ok && y - 2 * S < y_out1) {
                    const int64_t off = (int64_t)(y - 2 * S) * p.nx + xb;
                    st4(p.dst_re + off, x0.re, p.out_scale);
                    st4(p.dst_im + off, x0.im, p.out_scale);
                    st4(p.dst_re + off + p.nx, x1.re, p.out_scale);
                    st4(p.dst_im + off + p.nx, x1.im, p.out_scale);
                }
                if (++cs == NST) { cs = 0; cph ^= 1; }
                if (++rs == NST) rs = 0;
                if (POT && ++ps == NPH) ps = 0;
            }
        };
        half(std::integral_constant<int, 0>{});
        half(std::integral_constant<int, 1>{});
    }
    };   // run
    const bool edge = c.xedge || (!PERY && ((y_in0 < 0 && edge_top) ||
                                            (y_in0 + 2 * n_iter >= p.ny && edge_bot)));
    if (edge) run(std::true_type{});
    else run(std::false_type{});
}

// programmatic dependent launch of consecutive passes (environment TS_NO_PDL=1 turns it off)
bool stream_pdl() {
    static const bool on = [] {
        const char* e = getenv("TS_NO_PDL");
        return !(e && e[0] == '1');
    }();
    return on;
}

template <typename T, int S, int PM, int BND>
int launch(const StreamParams<T>& p, cudaStream_t st) {
    constexpr uint32_t SLOTB = 4 * kStripSites * sizeof(T);
    const size_t smem = (size_t)kWarps * ((size_t)(p.nst + (PM == 1 ? p.nph : 0)) * SLOTB + p.nst * 8);
    // register budget: the ring (64 KB per block) admits 3 blocks per SM anyway, so fp32 gets 168
    // registers from S = 3 on (128 below); fp64 3 or 2 blocks (255)
    constexpr int MINB = sizeof(T) == 4 ? (S <= 2 ? 4 : 3) : (S <= 2 ? 3 : 2);
    auto kern = stream_kernel<T, S, PM, BND, MINB>;
    // the opt-in for > 48 KB of dynamic shared memory is a per-device, per-kernel attribute:
    // remembered per instantiation and device (atomics: plans on different threads may race here,
    // setting it twice is harmless)
    static std::atomic<size_t> configured[kMaxDevices];
    int dev = 0;
    TS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices || smem > configured[dev].load(std::memory_order_relaxed)) {
        TS_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem));
        if (dev >= 0 && dev < kMaxDevices) configured[dev].store(smem, std::memory_order_relaxed);
    }
    const int64_t n_warps = (int64_t)p.n_xe * p.n_seg_x + (int64_t)(p.n_strips - p.n_xe) * p.n_seg;
    dim3 grid((unsigned)((n_warps + kWarps - 1) / kWarps));
    // programmatic dependent launch pays where launch latency and the prologue are a visible part
    // of a pass, i.e. for grids of at most one wave (1024^2 +12 %, 2048^2 +17 %, 4096^2 +0-2 %);
    // on many-wave grids the next pass's blocks then start in lockstep and a 16384^2 pass gets
    // ~8 % slower (probe r1f pdl/pdl2), so those keep the ordinary launch
    if (stream_pdl() && (int64_t)grid.x <= 148 * 3) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid;
        cfg.blockDim = dim3(kWarps * 32);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        TS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, p));
    } else {
        kern<<<grid, kWarps * 32, smem, st>>>(p);
    }
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}

template <typename T, int S, int PM>
int launch_b(const StreamParams<T>& p, int bnd, cudaStream_t st) {
    if (bnd == 1) return launch<T, S, PM, 1>(p, st);
    if (bnd == 2) return launch<T, S, PM, 2>(p, st);
    if constexpr (PM != 1) {      // slabs with peer halos: no phase planes
        if (bnd == 3) return launch<T, S, PM, 3>(p, st);
        if (bnd == 4) return launch<T, S, PM, 4>(p, st);
    }
    return launch<T, S, PM, 0>(p, st);
}

template <typename T, int S>
int launch_s(const StreamParams<T>& p, int pm, int bnd, cudaStream_t st) {
    if (pm == 1) return launch_b<T, S, 1>(p, bnd, st);
    if (pm == 2) return launch_b<T, S, 2>(p, bnd, st);
    return launch_b<T, S, 0>(p, bnd, st);
}

template <typename T>
int pass_t(const LatticeDesc& L, const T* src_re, const T* src_im, T* dst_re, T* dst_im,
           const StepCoef* subs, const Phase& ph, int S, SegShape seg, int nst, cudaStream_t st,
           const Peers* peers) {
    StreamParams<T> p;
    p.up_re = p.up_im = p.dn_re = p.dn_im = nullptr;
    p.up_rows = p.dn_rows = 0;
    if (peers) {
        p.up_re = (const T*)peers->up_re; p.up_im = (const T*)peers->up_im;
        p.dn_re = (const T*)peers->dn_re; p.dn_im = (const T*)peers->dn_im;
        p.up_rows = (int)peers->up_rows; p.dn_rows = (int)peers->dn_rows;
    }
    p.edge_top = p.up_re == nullptr;
    p.edge_bot = p.dn_re == nullptr;
    p.src_re = src_re; p.src_im = src_im; p.dst_re = dst_re; p.dst_im = dst_im;
    const T* pot = ph.mode == 1 ? (const T*)ph.planes : nullptr;
    p.pot_re = pot;
    p.pot_im = pot ? pot + L.nx * L.ny : nullptr;
    p.px_re = p.px_im = p.py_re = p.py_im = nullptr;
    p.py_off = 0; p.py_n = (int)L.ny; p.py_wrap = L.periodic_y;
    if (ph.mode == 2) {
        p.px_re = (const T*)ph.px; p.px_im = p.px_re + L.nx;
        const int64_t ny_g = ph.py_n > 0 ? ph.py_n : L.ny;
        p.py_re = (const T*)ph.py; p.py_im = p.py_re + ny_g;
        p.py_off = (int)ph.py_off; p.py_n = (int)ny_g;
        p.py_wrap = ph.py_n > 0 ? ph.py_wrap : L.periodic_y;
    }
    const bool any = ph.mode != 0;        // the 6-sweeps-and-P stage, as opposed to the regrouped one
    p.nx = (int)L.nx; p.ny = (int)L.ny;
    p.halo = (2 * S + 3) / 4 * 4;
    p.wi = kStripSites - 2 * p.halo;
    p.n_strips = (int)((L.nx + p.wi - 1) / p.wi);
    p.seg_rows = seg.rows;
    p.n_seg = (int)((L.ny + seg.rows - 1) / seg.rows);
    p.seg_edge = seg.rows; p.n_seg_x = 0; p.n_xe = 0; p.y_short = 0;
    if (seg.edge > 0 && seg.edge < seg.rows) {
        p.seg_edge = seg.edge;
        if (!L.periodic_x) {
            p.n_xe = p.n_strips < 2 ? p.n_strips : 2;
            p.n_seg_x = (int)((L.ny + seg.edge - 1) / seg.edge);
        }
        // first and last segment short: only where rows are left for a segment between them
        if (!L.periodic_y && L.ny >= 2 * (int64_t)seg.edge + 2) {
            p.y_short = 1;
            p.n_seg = 2 + (int)((L.ny - 2 * seg.edge + seg.rows - 1) / seg.rows);
        }
    }
    // state ring: prefetch distance + 1 slots; phase ring (planes only): prefetch + S + 1
    if (nst <= 0) nst = stream_default_slots(L, S, pot != nullptr);   // separable: as without
    if (nst < 2) nst = 2;
    const size_t slotb = (size_t)4 * kStripSites * sizeof(T);
    auto smem_of = [&](int n) {
        return (size_t)kWarps * ((size_t)(n + (pot ? n - 1 + S + 1 : 0)) * slotb + n * 8);
    };
    while (nst > 2 && smem_of(nst) > 227u * 1024u) --nst;
    p.nst = nst;
    p.nph = pot ? nst - 1 + S + 1 : 0;
    // tangents and deferred cosines of the S sub-steps (all in double, rounded once).  The merged
    // even sweep between sub-steps j-1 and j rotates by the sum of their half angles:
    // cos = a a' - b b', sin = a b' + b a'.
    double scale = 1.0;
    {
        const StepCoef& f = subs[0];
        const StepCoef& l = subs[S - 1];
        p.te[0] = (T)(f.b_h / f.a_h);
        p.te[S] = (T)(l.b_h / l.a_h);
        const double ends = f.a_h * l.a_h;
        scale *= ends * ends;                        // X-even and Y-even
    }
    for (int j = 1; j < S; ++j) {
        const StepCoef& u = subs[j - 1];
        const StepCoef& v = subs[j];
        const double cm = u.a_h * v.a_h - u.b_h * v.b_h;
        const double sm = u.a_h * v.b_h + u.b_h * v.a_h;
        p.te[j] = (T)(sm / cm);
        scale *= cm * cm;
    }
    for (int j = 0; j < S; ++j) {
        const StepCoef& v = subs[j];
        if (any) {
            // Xo, Yo at the half angle, each twice per sub-step
            p.to[j] = (T)(v.b_h / v.a_h);
            p.sec_o[j] = (T)(1.0 / v.a_h);
            scale *= pow(v.a_h, 4);
        } else {
            // Yo once with the caller's full-angle coefficients (the "full middle sweep"); Xo once
            // by twice the half angle: the regrouped form of Xo(h) ... Xo(h)
            p.to[j] = (T)(v.b_f / v.a_f);
            p.sec_o[j] = (T)(1.0 / v.a_f);
            const double c2 = v.a_h * v.a_h - v.b_h * v.b_h, s2 = 2.0 * v.a_h * v.b_h;
            p.tox[j] = (T)(s2 / c2);
            p.sec_ox[j] = (T)(1.0 / c2);
            scale *= v.a_f * c2;
        }
    }
    for (int j = 0; j < TS_MAX_FUSE; ++j) {
        if (any || j >= S) { p.tox[j] = T(0); p.sec_ox[j] = T(1); }
        if (j >= S) { p.to[j] = T(0); p.sec_o[j] = T(1); p.te[j + 1] = T(0); }
    }
    p.out_scale = (T)scale;
    int per = L.periodic_x ? (L.periodic_y ? 1 : 2) : 0;
    if (peers) {
        if (L.periodic_y || ph.mode == 1) {
            set_error("stream_pass: peer halos need a closed-y plan and no phase planes");
            return TS_EINVAL;
        }
        per = L.periodic_x ? 4 : 3;
    }
    switch (S) {
        case 1: return launch_s<T, 1>(p, ph.mode, per, st);
        case 2: return launch_s<T, 2>(p, ph.mode, per, st);
        case 3: return launch_s<T, 3>(p, ph.mode, per, st);
        case 4: return launch_s<T, 4>(p, ph.mode, per, st);
    }
    // deeper temporal blocking only where the ALU budget allows it: fp32 without a potential
    if constexpr (sizeof(T) == 4) {
        if (!any) {
            if (S == 5) return launch_b<T, 5, false>(p, per, st);
            if (S == 6) return launch_b<T, 6, false>(p, per, st);
        }
    }
    set_error("stream_pass: steps per pass out of range");
    return TS_EINVAL;
}

}  // namespace

// This file is compiled twice (build.py): once for fp32 (-DTS_STREAM_TU=32: defines
// stream_pass_f32, the dispatcher and the defaults) and once for fp64 (-DTS_STREAM_TU=64: only
// stream_pass_f64), so that the ~110 kernel instantiations build in parallel.
#ifndef TS_STREAM_TU
#define TS_STREAM_TU 0          // one translation unit with everything
#endif

#if TS_STREAM_TU == 0 || TS_STREAM_TU == 64
int stream_pass_f64(const LatticeDesc& L, const void* src_re, const void* src_im, void* dst_re,
                    void* dst_im, const StepCoef* subs, const Phase& ph, int S, SegShape seg,
                    int nst, cudaStream_t st, const Peers* peers) {
    return pass_t<double>(L, (const double*)src_re, (const double*)src_im, (double*)dst_re,
                          (double*)dst_im, subs, ph, S, seg, nst, st, peers);
}
#endif

#if TS_STREAM_TU == 0 || TS_STREAM_TU == 32
int stream_pass_f64(const LatticeDesc& L, const void* src_re, const void* src_im, void* dst_re,
                    void* dst_im, const StepCoef* subs, const Phase& ph, int S, SegShape seg,
                    int nst, cudaStream_t st, const Peers* peers);

bool stream_supported(const LatticeDesc& L, const StepCoef& c) {
    // the strip window must split into at most two contiguous pieces of a row
    // (closed in x with periodic in y is not instantiated)
    // (periodic in x: the 128-wide window may wrap once, so the row must be at least that long;
    // closed in x: any width, columns beyond the lattice are ghost lanes)
    return fused_shape_ok(L, c) && (L.nx >= kStripSites || !L.periodic_x) &&
           (L.periodic_x || !L.periodic_y);
}

int stream_max_steps(const LatticeDesc& L, bool pot) {
    return (L.dtype == TS_F32 && !pot) ? 6 : 4;
}

int stream_default_steps_sep(const LatticeDesc& L) {
    // no phase rows in the ring: the occupancy of the potential-free kernel, the arithmetic of the
    // 6-sweeps-and-P stage (probe r1e)
    return L.dtype == TS_F32 ? 4 : 4;
}

int stream_default_slots(const LatticeDesc& L, int S, bool pot) {
    // measured on B200 (round-1 probes): 8 row-pair slots per warp keep ~7 iterations in
    // flight for fp32 without a potential (64 KB per block, 3 blocks per SM).  With phase planes
    // (own ring of prefetch + S + 1 slots) two state slots = one iteration in flight per warp, in
    // both types: fp32 at S = 3 14 KB per warp, 3 blocks per SM (register-limited); fp64 28 KB per
    // warp, 112 KB per block, 2 blocks per SM.  Measured (profiles/r2_probe_stream_pot.txt): C3
    // 5.34e11 with one ring of 8-row slots, 5.76e11 with 3 state slots, 5.96e11 with 2; C5 2.81e11
    // -> 3.05e11 with 2 (2.86e11 with 3: one block per SM again).
    if (pot) return 2;
    return L.dtype == TS_F32 ? 8 : 6;
}

SegShape stream_default_seg(const LatticeDesc& L, int S, int blocks_per_sm) {
    // As fused_default_seg_rows (a segment of r rows costs r/2 + 2S + 1 iterations; whole waves,
    // since a grid of 1.1 waves costs two), but counted in WARPS: the kernel deals (strip, segment)
    // pairs to warps without gaps, so the machine holds 148 * blocks_per_sm * kWarps of them per
    // wave whatever n_strips is.  Warps at a closed edge run the edge variant of the loop, which
    // costs kEdgeCost per row of the plain one (4096^2 at S = 3: 76.7 us per pass periodic, 82.6
    // closed with equal segments): their segments are shortened by that factor, and the smallest
    // plain height whose warp count still fits the waves is taken.
    constexpr double kEdgeCost = 1.08;
    const int halo = (2 * S + 3) / 4 * 4;
    const int64_t strips = (L.nx + (kStripSites - 2 * halo) - 1) / (kStripSites - 2 * halo);
    const int64_t slots = 148 * (int64_t)(blocks_per_sm > 0 ? blocks_per_sm : 3) * kWarps;
    const int64_t cap = S >= 5 ? 512 : 256;
    const int64_t min_segs = (L.ny + cap - 1) / cap;
    int64_t waves = (min_segs * strips + slots - 1) / slots;
    if (waves < 1) waves = 1;
    int64_t segs = waves * slots / strips;
    if (segs < 1) segs = 1;
    int64_t r = (L.ny + segs - 1) / segs;
    r += r % 2;
    if (r > cap) r = cap;
    if (r < 8) r = 8;     // small lattices: parallelism over warm-up redundancy
    if (r > L.ny) r = L.ny;
    SegShape out{(int)r, 0};
    const bool closed = !L.periodic_x || !L.periodic_y;
    static const bool no_short = getenv("TS_PROBE_NO_SHORT_EDGE") != nullptr;   // tuning probe only
    if (!closed || no_short || r < 32 || L.ny < 4 * r) return out;
    auto edge_of = [&](int64_t h) {
        int64_t e = (int64_t)(2.0 * ((h / 2 + 2 * S + 1) / kEdgeCost - (2 * S + 1)));
        e -= e % 2;
        if (e < 8) e = 8;
        return e < h ? e : h;
    };
    auto warps_of = [&](int64_t h, int64_t e) {
        const int64_t n_xe = L.periodic_x ? 0 : (strips < 2 ? strips : 2);
        const int64_t seg_x = (L.ny + e - 1) / e;
        int64_t seg_i = (L.ny + h - 1) / h;
        if (!L.periodic_y) seg_i = 2 + (L.ny - 2 * e + h - 1) / h;
        return n_xe * seg_x + (strips - n_xe) * seg_i;
    };
    // the equal-height choice r fits by construction; taller plain segments make room for the
    // extra (short) edge segments
    for (int64_t h = r; h <= cap; h += 2) {
        const int64_t e = edge_of(h);
        if (warps_of(h, e) <= waves * slots) return SegShape{(int)h, (int)e};
    }
    return out;
}

int stream_pass(const LatticeDesc& L, const void* src_re, const void* src_im, void* dst_re,
                void* dst_im, const StepCoef* subs, const Phase& ph, int S, SegShape seg, int nst,
                cudaStream_t st, const Peers* peers) {
    if (seg.rows <= 0 || seg.rows % 2 || seg.edge < 0 || seg.edge % 2 || seg.edge > seg.rows) {
        set_error("stream_pass: segment heights must be positive and even, edge <= rows");
        return TS_EINVAL;
    }
    if (L.dtype == TS_F32)
        return pass_t<float>(L, (const float*)src_re, (const float*)src_im, (float*)dst_re,
                             (float*)dst_im, subs, ph, S, seg, nst, st, peers);
    return stream_pass_f64(L, src_re, src_im, dst_re, dst_im, subs, ph, S, seg, nst, st,
                           peers);
}
#endif

}  // namespace ts
