// ts_internal.h -- declarations shared by the translation units of libts (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "ts.h"

namespace ts {

void set_error(const std::string& msg);
int cuda_fail(cudaError_t e, const char* what);   // records the CUDA string, returns TS_ECUDA

#define TS_CUDA_TRY(expr)                                             \
    do {                                                              \
        cudaError_t e_ = (expr);                                      \
        if (e_ != cudaSuccess) return ::ts::cuda_fail(e_, #expr);     \
    } while (0)

// Optional per-launch timing (plan option "timing"): CUDA events around every kernel or copy of
// one ts_evolve* call, on the launch stream; read back with ts_plan_get_launch_times.
enum LaunchKind {
    kKindGeneric = 1,   // the per-sweep kernels of one whole call (not split)
    kKindFused = 2,     // fused_kernel pass (register prefetch)
    kKindStream = 3,    // stream_kernel pass (TMA ring)
    kKindTiny = 4,      // tiny_kernel (whole evolution)
    kKindLineRows = 5,  // line_kernel along rows (resident lines, all sub-steps)
    kKindLineCols = 6,  // line_kernel along columns
    kKindXwin = 7,      // xwin_kernel pass (windowed rows)
    kKindYcol = 8,      // ycol_kernel pass (pipelined columns)
    kKindCopy = 9,      // device-to-device copy of a plane
    kKindExpand = 10,   // separable phase written out as planes
    kKindLineZ = 11     // line_kernel along z (3-D lattices)
};
struct LaunchTimer {
    struct Rec {
        int kind;
        cudaEvent_t a, b;
    };
    std::vector<Rec> recs;
    size_t used = 0;
    void reset() { used = 0; }
    void begin(int kind, cudaStream_t st);
    void end(cudaStream_t st);
    ~LaunchTimer();
};
// null-safe helpers
inline void timer_begin(LaunchTimer* t, int kind, cudaStream_t st) { if (t) t->begin(kind, st); }
inline void timer_end(LaunchTimer* t, cudaStream_t st) { if (t) t->end(st); }

// Double-precision description of one step; each path converts to its own arithmetic form.
struct StepCoef {
    double a_h, b_h, a_f, b_f;
};

// The diagonal step P of a sub-step: none, full phase planes [2][ny][nx], or separable factors
// px [2][nx], py [2][ny] with P(x, y) = px(x) * py(y) (device pointers of the plan's dtype).
struct Phase {
    int mode;             // 0 none, 1 planes, 2 separable
    const void* planes;
    const void* px;
    const void* py;
    // separable phase of a row slab: py covers the GLOBAL lattice (py_n rows, py_n = 0: the plan's
    // own ny), local row 0 is global row py_off, py_wrap = global lattice periodic in y
    int64_t py_off = 0;
    int64_t py_n = 0;
    int py_wrap = 0;
};

// Neighbours of a row slab (ts_slab_pass): their SOURCE planes of this pass and their row counts.
struct Peers {
    const void* up_re;
    const void* up_im;
    int64_t up_rows;
    const void* dn_re;
    const void* dn_im;
    int64_t dn_rows;
};

struct LatticeDesc {
    int64_t nx, ny;
    int dtype;      // TS_F32 / TS_F64
    int periodic_x, periodic_y;   // per axis: 0 closed, 1 periodic
};

// ---- generic per-sweep path (ts_generic.cu): in place, any nx, ny ------------------------------
// n_steps full second-order steps, 7 (pot == nullptr) or 9 launches per step.
int generic_evolve(const LatticeDesc& L, void* re, void* im, const StepCoef& c,
                   const void* pot, int64_t n_steps, cudaStream_t st, int64_t* launches);

// sum re^2 + im^2 in double -> *d_out (device double).  workspace: >= norm_workspace_doubles().
int norm2_device(const LatticeDesc& L, const void* re, const void* im, double* d_work,
                 cudaStream_t st);
size_t norm_workspace_doubles();

// ---- fused streaming path (ts_fused.cu): out of place, S steps per pass ------------------------
bool fused_shape_ok(const LatticeDesc& L, const StepCoef& c);   // alignment and angle range only
bool fused_supported(const LatticeDesc& L, const StepCoef& c);  // + same boundary on both axes
// One pass: dst <- U2^S src.  S in 1..TS_MAX_FUSE.  seg_rows even, > 0.
int fused_pass(const LatticeDesc& L, const void* src_re, const void* src_im, void* dst_re,
               void* dst_im, const StepCoef& c, const void* pot, int S, int seg_rows,
               cudaStream_t st);
int fused_default_seg_rows(const LatticeDesc& L, int S, int blocks_per_sm = 3);

// ---- on-chip-resident path for tiny lattices (ts_tiny.cu): the whole evolution in one launch -----
int tiny_rows_per_warp(const LatticeDesc& L, bool pot, int prefer);   // prefer 4: 4 rows if possible
bool tiny_supported(const LatticeDesc& L, const StepCoef& c, bool pot);
int tiny_evolve(const LatticeDesc& L, void* re, void* im, const StepCoef& c, const void* pot,
                int64_t n_steps, int rows_per_warp, cudaStream_t st);

// ---- fused streaming path v2 (ts_stream.cu): TMA bulk copies into a per-warp smem ring ---------
bool stream_supported(const LatticeDesc& L, const StepCoef& c);
int stream_max_steps(const LatticeDesc& L, bool pot);   // 6 for fp32 without potential, else 4
int stream_default_steps_sep(const LatticeDesc& L);     // sub-steps per pass, separable phase
int stream_default_slots(const LatticeDesc& L, int S, bool pot);
// Segment heights of one pass: `rows` for warps that run the plain loop, `edge` (<= rows; 0: as
// rows) for warps that run the closed-edge variant of it (x-edge strips, first / last segment of
// a lattice closed in y), which costs ~8 % more per row.
struct SegShape {
    int rows, edge;
};
SegShape stream_default_seg(const LatticeDesc& L, int S, int blocks_per_sm = 3);
// One pass: dst <- U2(subs[S-1]) ... U2(subs[0]) src; the S sub-steps may have different angles
// (fourth-order step, Eq. 4) but share one potential-phase array.
int stream_pass(const LatticeDesc& L, const void* src_re, const void* src_im, void* dst_re,
                void* dst_im, const StepCoef* subs, const Phase& ph, int S, SegShape seg, int nst,
                cudaStream_t st, const Peers* peers = nullptr);
// pot[2][ny][nx] <- px (x) py: the separable factors written out for paths that take planes
int expand_separable(const LatticeDesc& L, const void* px, const void* py, void* pot,
                     cudaStream_t st);
int fused_default_steps(const LatticeDesc& L, bool pot);


// ---- axis-split path for steps without a potential (ts_axis.cu) ------------------------------------
// U2^n = (row chain) x (column chain): whole lines resident in a warp's registers where they fit
// (one launch per axis for ALL sub-steps, in place), else windowed rows / pipelined columns with up
// to 16 sub-steps per pass (out of place, ping-pong with the scratch planes).
struct AxisInfo {
    int64_t passes, launches, chain_x, chain_y, seg_rows;
};
// Rows that arrive in pieces (ts_evolve_host: the host-to-device copy of rows [y_end[k-1],
// y_end[k]) of both planes has completed when ready[k] has): the row chain of a piece starts as
// soon as the piece is there, while the next one is still on the bus.
struct RowFeed {
    int n;
    const int64_t* y_end;
    const cudaEvent_t* ready;
};
bool axis_supported(const LatticeDesc& L, const StepCoef* pat, int period);
bool axis_needs_scratch(const LatticeDesc& L);
int axis_default_chain(const LatticeDesc& L);
// psi <- (U2(pat[period-1]) ... U2(pat[0]))^(n_sub / period) psi, n_sub sub-steps in pattern order.
// chain: sub-steps per windowed / pipelined pass (0 = default); seg_rows, nst: 0 = default.
int axis_evolve(const LatticeDesc& L, void* psi_re, void* psi_im, void* scr_re, void* scr_im,
                const StepCoef* pat, int period, int64_t n_sub, int chain, int seg_rows, int nst,
                cudaStream_t st, AxisInfo* info, LaunchTimer* timer = nullptr,
                const RowFeed* feed = nullptr);
// true if axis_evolve consumes a RowFeed piece by piece on this lattice (rows resident in
// registers); otherwise the caller waits for the last piece before the call
bool axis_takes_feed(const LatticeDesc& L);


// ---- three-dimensional lattices ------------------------------------------------------------------------
struct Lattice3 {
    int64_t nx, ny, nz;
    int dtype;
    int per[3];       // periodic flag of the x, y, z axis
};
// every axis resident in registers (even extents that fit a thread block), cos of every angle > 0.25
bool axis3_supported(const Lattice3& L, const StepCoef& c);
// n_steps steps on psi[nz][ny][nx], in place; pot = null or phase planes [2][nz][ny][nx]
int axis3_evolve(const Lattice3& L, void* re, void* im, const StepCoef& c, const void* pot,
                 int64_t n_steps, cudaStream_t st, AxisInfo* info, LaunchTimer* timer);
// per-sweep kernels (ts_generic.cu): 11 / 13 launches per step, any extents
int generic3_evolve(const Lattice3& L, void* re, void* im, const StepCoef& c, const void* pot,
                    int64_t n_steps, cudaStream_t st, int64_t* launches);

}  // namespace ts
