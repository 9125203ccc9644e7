/*
 * ts.h -- C ABI of libts: second-order Trotter-Suzuki time step for one particle on a 2-D (or 3-D:
 * ts_plan_create_3d) lattice, NVIDIA B200 (sm_100a).  Plain pointers and sizes only; no C++/torch
 * types.
 *
 * What it computes (PAPER.md = the paper's text; readings R1..R13 are listed in DESIGN.md):
 *   The lattice Hamiltonian is split into a diagonal part H0 and, per axis, an even-pair and an
 *   odd-pair part.  The exponential of a pair part is a set of
 *   independent 2x2 plane rotations M = [[a, i b],[i b, a]].  One time step is
 *   the symmetrised second-order product U2 = U1^T U1 (Eq. 3), here
 *
 *      Xe(h) Xo(h) Ye(h) [ Yo(f) | Yo(h) P Yo(h) ] Ye(h) Xo(h) Xe(h)       applied left to right,
 *
 *   X/Y = horizontal/vertical, e/o = even pairs (2k,2k+1) / odd pairs (2k+1,2k+2),
 *   (h) = half-angle coefficients (a_half, b_half), (f) = full-angle (a_full, b_full),
 *   P = multiplication by the unit-modulus potential phase exp(-i V dt).
 *
 * Data layout: the wavefunction is two dense planes psi_re[ny][nx], psi_im[ny][nx] (x fastest,
 * element (x, y) at y*nx + x) of the plan's dtype, in DEVICE memory, each 16-byte aligned and
 * non-overlapping.  pot_phase is 2*ny*nx elements of the same dtype in DEVICE memory: plane 0 =
 * Re = cos(V dt), plane 1 = Im = -sin(V dt).
 *
 * Every function returns TS_OK (0) or an error code; nothing is enqueued when an error is
 * returned by argument validation.  ts_last_error() gives a thread-local text for the last
 * failure on the calling thread.  No exceptions cross this boundary.
 */
#ifndef TS_H_
#define TS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ts_plan ts_plan;               /* opaque; owned by the library */

enum { TS_F32 = 0, TS_F64 = 1 };              /* dtype of psi planes and pot_phase */
enum { TS_CLOSED = 0, TS_PERIODIC = 1 };      /* boundary, same on both axes */
enum { TS_OK = 0, TS_EINVAL = 1, TS_EUNSUPPORTED = 2, TS_EALLOC = 3, TS_ECUDA = 4 };

/*
 * ts_plan_create -- describe a lattice (L x L mesh; here nx x ny).
 *   nx, ny    lattice extent, >= 1, nx*ny < 2^62.
 *   dtype     TS_F32 or TS_F64.
 *   boundary  TS_CLOSED: pairs crossing the edge are omitted, unpaired sites are unchanged in
 *             that sweep (the zero 1x1 blocks of the printed H1/H2);
 *             TS_PERIODIC: the wrap pair (n-1, 0) belongs to the odd sweep; needs nx, ny even.
 * Returns a plan bound to the CUDA device current at the call, or NULL (see ts_last_error()).
 * The plan owns all scratch (second state buffer for the double-buffered fused kernel,
 * PAPER.md:109; reduction workspace); scratch is allocated on first use and freed by
 * ts_plan_destroy.  A plan may be reused across calls and streams, but not concurrently.
 */
ts_plan* ts_plan_create(int64_t nx, int64_t ny, int dtype, int boundary);

/*
 * ts_plan_create_xy -- the same with one boundary type per axis.  (TS_PERIODIC, TS_CLOSED) is what
 * a row slab of a larger periodic lattice needs (domain decomposition: the
 * slab plus its halo rows is evolved as a lattice that is closed in y; the rows within 2 sites per
 * step of a cut are then wrong and are the halo that the next exchange overwrites).
 * (TS_CLOSED, TS_PERIODIC) with a potential runs on the per-sweep kernels only.
 */
ts_plan* ts_plan_create_xy(int64_t nx, int64_t ny, int dtype, int boundary_x, int boundary_y);

/*
 * ts_plan_create_3d -- a THREE-dimensional lattice nx x ny x nz, the extension the paper names as its
 * next direction along the lines it gives for more than one dimension ("the
 * diagonal energies, and two terms for each dimension").  One boundary type per
 * axis, as for ts_plan_create_xy; a periodic axis needs an even extent.  Layout: planes
 * psi[nz][ny][nx], x fastest, element (x, y, z) at (z*ny + y)*nx + x.  Such a plan is evolved with
 * ts_evolve_3d only (ts_norm works on it; the 2-D entry points return TS_EINVAL).
 */
ts_plan* ts_plan_create_3d(int64_t nx, int64_t ny, int64_t nz, int dtype,
                           int boundary_x, int boundary_y, int boundary_z);

/*
 * ts_evolve_3d -- psi <- U2^n_steps psi on a plan from ts_plan_create_3d, in place, with the step
 *
 *      Xe(h) Xo(h) Ye(h) Yo(h) Ze(h) [ Zo(f) | Zo(h) P Zo(h) ] Ze(h) Yo(h) Ye(h) Xo(h) Xe(h)
 *
 * (Eq. 3 with seven parts; reading R14: the 2-D order with the new axis innermost).
 * Arguments as for ts_evolve; pot_phase_or_null is 2*nz*ny*nx elements (Re plane, then Im plane).
 * Paths: sweeps along different axes commute, so without a potential the n_steps steps are three
 * chains (one launch per axis, every line resident in registers for all steps), and with one the
 * sweeps between two applications of the phase regroup per axis into O(h) E(2h) O(h): three
 * launches per step.  Both need even extents of at most 16384 (fp32) / 8192 (fp64) sites per axis
 * in a shape a thread block holds, and cos of every sweep angle > 0.25; other lattices run on the
 * per-sweep kernels (11 / 13 launches per step).  Option "path" = 1 forces those, "path" = 2 or
 * "variant" = 4 requires the fused path (TS_EUNSUPPORTED otherwise).  No scratch is used.
 */
int ts_evolve_3d(ts_plan* plan, void* psi_re, void* psi_im,
                 double a_half, double b_half, double a_full, double b_full,
                 const void* pot_phase_or_null, int64_t n_steps, void* cuda_stream);

/*
 * ts_evolve -- psi <- U2^n_steps psi, in place from the caller's view (Eq. 3).
 *   psi_re, psi_im   DEVICE pointers, ny*nx elements each, 16-byte aligned, caller-owned.
 *   a_half, b_half   cos, sin of theta/2, theta = dt*|V_tunnel|/hbar.
 *   a_full, b_full   cos, sin of theta; used by the middle sweep when pot_phase is NULL.
 *                    Both pairs must be finite with |a^2 + b^2 - 1| <= 1e-6.  The sign of b is
 *                    the caller's: (b -> -b, pot_phase -> conj) is the time-reversed step.
 *   pot_phase_or_null  NULL: 7-stage step.  Else DEVICE pointer to 2*ny*nx elements: 9-stage
 *                    step with the phase at the centre (a_full, b_full validated but unused).
 *   n_steps          >= 0; 0 is a no-op.
 *   cuda_stream      cudaStream_t passed as void* (NULL = legacy default stream).
 * Work is enqueued on the stream; the call does not synchronise.  The plan's scratch buffer is
 * in use until that work completes.
 * Errors: TS_EINVAL (NULL/misaligned/overlapping pointers, pointers to pageable host memory, bad
 * coefficients, n_steps < 0), TS_EALLOC (scratch allocation), TS_ECUDA (launch failure; text in
 * ts_last_error()).
 */
int ts_evolve(ts_plan* plan, void* psi_re, void* psi_im,
              double a_half, double b_half, double a_full, double b_full,
              const void* pot_phase_or_null, int64_t n_steps, void* cuda_stream);

/*
 * ts_evolve_u4 -- psi <- U4^n_steps psi, the fourth-order step of Eq. 4:
 *
 *      U4(dt) = U2(p dt) U2(p dt) U2((1-4p) dt) U2(p dt) U2(p dt),     p = (4 - 4^(1/3))^-1,
 *
 * every U2(f dt) being the second-order step of ts_evolve with angle f*theta (coefficients
 * cos/sin(f theta/2), cos/sin(f theta), computed in double inside the library).
 *   theta            full-step angle dt*|V_tunnel|/hbar in radians, finite; its sign is the caller's.
 *   pot_phase_p_or_null, pot_phase_q_or_null
 *                    both NULL (no potential) or both DEVICE pointers to 2*ny*nx elements laid out
 *                    like pot_phase of ts_evolve: the phases of the two distinct sub-steps,
 *                    exp(-i V p dt) and exp(-i V (1-4p) dt).
 * Other arguments, asynchrony, scratch use and errors as for ts_evolve.  The five sub-steps are
 * chained inside the fused kernel like ordinary steps (per-sub-step angle table), so a
 * fourth-order step costs five second-order sub-steps, not five passes over HBM.
 */
int ts_evolve_u4(ts_plan* plan, void* psi_re, void* psi_im, double theta,
                 const void* pot_phase_p_or_null, const void* pot_phase_q_or_null,
                 int64_t n_steps, void* cuda_stream);

/*
 * ts_u4_coefficients -- the coefficient table of ONE fourth-order step (Eq. 4), as
 * ts_evolve_u4 uses it: five rows (a_half, b_half, a_full, b_full) for the sub-step angles
 * p theta, p theta, (1-4p) theta, p theta, p theta with p = (4 - 4^(1/3))^-1, in order of
 * application.  For callers that schedule passes themselves (ts_slab_pass): the method's
 * constants come from the library, not from the binding.  Host arithmetic only; no device needed.
 *   out20   HOST array of 20 doubles.            Errors: TS_EINVAL (NULL, non-finite theta).
 */
int ts_u4_coefficients(double theta, double* out20);

/*
 * ts_evolve_sep -- ts_evolve for a SEPARABLE potential V(x, y) = Vx(x) + Vy(y) (the harmonic trap
 * of the benchmark configs is one): the phase of the diagonal step factorises,
 * exp(-i V dt) = px(x) * py(y), and is passed as two vectors instead of two planes
 * (the remark that a general potential "always adds a cost": this one adds
 * arithmetic but no memory traffic).
 *   phase_x   DEVICE pointer, 2*nx elements of the plan's dtype: Re px[0..nx), then Im px[0..nx).
 *   phase_y   DEVICE pointer, 2*ny elements: Re py, then Im py.   Both 16-byte aligned.
 * The step is the 9-stage step of ts_evolve with P(x, y) = px(x) py(y) (complex product, formed
 * in the plan's dtype).  The TMA ring kernel keeps px in registers and reads py through L1, so a
 * pass moves 16 B (fp32) per site like the potential-free step; other paths first write the
 * product out as planes into plan-owned scratch.  Other arguments and errors as for ts_evolve.
 */
int ts_evolve_sep(ts_plan* plan, void* psi_re, void* psi_im,
                  double a_half, double b_half, double a_full, double b_full,
                  const void* phase_x, const void* phase_y, int64_t n_steps, void* cuda_stream);

/*
 * ts_evolve_tdep -- ts_evolve for a TIME-DEPENDENT potential (the Hamiltonian may
 * depend on time): step k (k = 0 .. n_steps-1) uses the phase planes pot_phases[k].
 *   pot_phases   HOST array of n_steps DEVICE pointers, each laid out like pot_phase of ts_evolve
 *                (NULL entry = that step has no potential and is the 7-stage step).
 * Steps are fused into one pass only while they share the same phase array, so a potential that
 * changes every step costs one pass over HBM per step (24 B per site in fp32).  Other arguments,
 * asynchrony (the pointer list is read before the call returns) and errors as for ts_evolve.
 */
int ts_evolve_tdep(ts_plan* plan, void* psi_re, void* psi_im,
                   double a_half, double b_half, double a_full, double b_full,
                   const void* const* pot_phases, int64_t n_steps, void* cuda_stream);

/*
 * ts_slab_pass -- ONE fused pass over a row slab of a larger lattice, halos read in place from
 * the neighbouring slabs: dst <- U2(c[n_sub-1]) ... U2(c[0]) src on the plan's nx x ny rows, where
 * the rows above row 0 are the LAST up_rows rows of (up_re, up_im) and the rows below row ny-1
 * are the FIRST dn_rows rows of (dn_re, dn_im) -- the neighbours' source planes of this same
 * pass, in this GPU's memory or mapped from a peer GPU (NVLink).  This is the compute step and the
 * halo "exchange" of the distributed solver in one kernel: the bulk copies
 * that feed the pipeline simply take the rows beyond the slab from the neighbour's address.
 *   plan        from ts_plan_create_xy(nx, ny_slab, dtype, boundary_x, TS_CLOSED); ny_slab even.
 *   src, dst    DEVICE planes of the slab, distinct (out of place; the caller ping-pongs).
 *   up_*, dn_*  neighbour planes (pitch nx) or NULL for a real closed edge of the lattice;
 *               up_rows, dn_rows even and >= 2*n_sub.
 *   coef        HOST table, n_sub rows of (a_half, b_half, a_full, b_full): the sub-steps of this
 *               pass in order of application (equal rows: plain steps; the Eq. 4 pattern: U4).
 *   n_sub       sub-steps fused in this pass: 1..6 (fp32 without potential), else 1..4.
 *   phase_x, phase_y, y0, ny_global, periodic_y_global
 *               both NULL: no potential.  Else the separable phase of ts_evolve_sep, phase_y
 *               covering the GLOBAL lattice (2*ny_global elements); slab row y is global row
 *               y0 + y (y0 even), and rows beyond the global lattice wrap if periodic_y_global.
 * The caller must make sure that the neighbours have finished writing their source planes
 * (i.e. the previous pass) before this pass starts, and do not overwrite them before it ends:
 * one barrier over the ranks between passes (paper_1208_2407_b200/slab.py::PeerRank).
 * Errors: TS_EINVAL, TS_EUNSUPPORTED (shapes the TMA ring kernel does not take), TS_ECUDA.
 */
int ts_slab_pass(ts_plan* plan, const void* src_re, const void* src_im, void* dst_re, void* dst_im,
                 const void* up_re, const void* up_im, int64_t up_rows,
                 const void* dn_re, const void* dn_im, int64_t dn_rows,
                 const double* coef, int n_sub,
                 const void* phase_x, const void* phase_y, int64_t y0, int64_t ny_global,
                 int periodic_y_global, void* cuda_stream);

/*
 * ts_norm -- squared norm sum |psi|^2, accumulated in double for either dtype.
 *   psi_re, psi_im   DEVICE pointers as above (read only).
 *   out_norm2_host   HOST pointer to one double, written before the call returns.
 * Enqueues on cuda_stream and synchronises that stream.
 */
int ts_norm(ts_plan* plan, const void* psi_re, const void* psi_im,
            double* out_norm2_host, void* cuda_stream);

/*
 * ts_norm_static -- the same squared norm for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it): needs no plan,
 * allocates NOTHING (no cudaMalloc / cudaFree, no stream or event creation), never synchronises.
 * The per-chunk partial sums live in a 256 KB array in the library's device image (every GPU that
 * loads libts holds it until the process exits) instead of a plan-owned allocation.
 *   dtype              TS_F32 / TS_F64, the element type of both planes.
 *   psi_re, psi_im     DEVICE pointers to n_sites elements each (read only; any lattice shape,
 *                      planes contiguous).
 *   n_sites            0 <= n_sites <= 536870912 (2^29: 32768 partial sums of 16384 sites; C4's
 *                      16384^2 is 2^28).  Larger: TS_EUNSUPPORTED, nothing enqueued -- use ts_norm.
 *   out_norm2_device   DEVICE pointer to one double, written by the last kernel of the call
 *                      (stream-ordered: read it after the stream has reached that point).
 * Enqueues two kernels on cuda_stream (on the current device) and returns.  The sum is taken in a
 * fixed order, so equal inputs give bit-equal results.  The first call on each device looks up
 * the array's device address (make that call outside a graph capture).
 * Sharing: all calls on one device use the same array, which keeps the last call's contents;
 * nothing in it needs clearing (a call reads only what it has itself just written), but two
 * calls that OVERLAP on the GPU (different streams without a dependency) race -- order them.
 * Errors: TS_EINVAL (NULL / host pointers, bad dtype, n_sites < 0), TS_EUNSUPPORTED (n_sites
 * beyond the maximum), TS_ECUDA.
 */
int ts_norm_static(int dtype, const void* psi_re, const void* psi_im, int64_t n_sites,
                   double* out_norm2_device, void* cuda_stream);

/*
 * ts_evolve_host -- the same operation for HOST-resident planes (pageable or pinned): copies
 * psi (and pot_phase when given) to plan-owned device buffers, runs ts_evolve, copies psi
 * back, and synchronises.  This is the end-to-end entry measured by bench.py's "e2e".
 * Large lattices without a potential go up in 8 pieces of rows on a second plan-owned stream; where
 * the rows are evolved as resident lines (the axis-split path) the row chain of a piece runs while
 * the next piece is still on the bus, every other path waits for the last piece.  The result is
 * bit-identical to ts_evolve on device planes.  On an error nothing is left running.
 */
int ts_evolve_host(ts_plan* plan, void* psi_re_host, void* psi_im_host,
                   double a_half, double b_half, double a_full, double b_full,
                   const void* pot_phase_host_or_null, int64_t n_steps);

/*
 * ts_plan_set_option -- tuning knobs, all optional.  Unknown names give TS_EINVAL.
 *   "path"         0 = auto, 1 = generic per-sweep kernels only, 2 = fused kernel required
 *                  (ts_evolve then returns TS_EUNSUPPORTED for shapes the fused kernel cannot take).
 *   "fuse_steps"   steps fused per pass over HBM (1..TS_MAX_FUSE; 5 and 6 only fp32 without phase
 *                  planes on the TMA ring kernel), 0 = auto.
 *   "seg_rows"     rows of output per streaming segment of the fused kernel (even), 0 = auto;
 *                  for the on-chip kernel (variant 3): rows per warp, 2 / 4 / 8, 0 = auto.
 *   "variant"      0 = auto, 1 = register-prefetch kernel, 2 = TMA ring kernel (the default with a
 *                  potential wherever it applies: nx >= 128 or closed in x), 3 = on-chip-resident
 *                  kernel: the whole lattice in the registers of one thread block and all n_steps
 *                  in one launch (lattices up to 128 x 128 sites in fp32, 128 x 64 in fp64, half
 *                  that with a potential; the default there WITH a potential), 4 = axis-split path
 *                  (the default WITHOUT a potential, nx % 4 == 0, even ny): the step then
 *                  factorises exactly into a chain of sweeps along every row times a chain along
 *                  every column (X and Y sweeps commute); lines that fit a thread
 *                  block stay in registers for ALL n_steps (one launch per axis), longer rows are
 *                  cut into windows with a halo, longer columns stream through a register pipeline.
 *   "chain"        axis-split path: sub-steps per windowed / pipelined pass (<= 24 fp32, 12 fp64),
 *                  0 = auto.
 *   "ring_slots"   row-pair slots of the TMA ring per warp, 0 = auto (with phase planes: slots of the
 *                  state ring, i.e. prefetch distance + 1; the phase ring follows from it; the
 *                  column pipeline of the axis-split path holds two row pairs per slot and rounds
 *                  the count up to whole slots, at least two).
 *   "timing"       1: record CUDA events around every launch (ts_plan_get_launch_times), 0 = off.
 * Environment: TS_NO_PDL=1 turns off programmatic dependent launch between passes.
 */
int ts_plan_set_option(ts_plan* plan, const char* name, int64_t value);

/* ts_plan_get_info -- read back what the last ts_evolve* / ts_slab_pass used:
 *   "fused" (0/1), "fuse_steps", "passes", "launches" (kernels + copies enqueued), "seg_rows",
 *   "variant" (1 / 2 / 3 / 4, 0 on the per-sweep path), "chain_x", "chain_y" (axis-split path:
 *   sub-steps per launch along the rows / the columns). */
int ts_plan_get_info(const ts_plan* plan, const char* name, int64_t* out_value);

/*
 * ts_plan_reserve -- allocate now what ts_evolve* would allocate on first use (the second state
 * buffer for the double-buffered passes, and the reduction workspace of ts_norm), so
 * that no later call contains a device allocation.  with_host_staging != 0 also reserves the
 * device staging buffers of ts_evolve_host (state; plus phase planes if with_host_staging == 2).
 * Errors: TS_EINVAL (NULL plan, other device current), TS_EALLOC.
 */
int ts_plan_reserve(ts_plan* plan, int with_host_staging);

/*
 * ts_plan_get_launch_times -- device time of every launch of the LAST ts_evolve* call on this plan,
 * measured by CUDA events that the library records on the launch stream around each kernel (and
 * around the final plane copies) when the plan option "timing" is 1.  bench.py reports its
 * roofline from these (the dominant kernel's own time, not the call divided by the launch count).
 *   max_n      capacity of the two output arrays.
 *   kinds_out  HOST array: what was launched -- 1 per-sweep kernels of one whole call, 2 fused_kernel
 *              pass, 3 stream_kernel pass, 4 tiny_kernel, 5 line_kernel along rows, 6 line_kernel
 *              along columns, 7 xwin_kernel pass, 8 ycol_kernel pass, 9 plane copies, 10 separable
 *              phase expansion, 11 line_kernel along z, 12 phase kernel (3-D).
 *   ms_out     HOST array: milliseconds.
 *   n_out      HOST int: number of launches recorded (may exceed max_n; then only max_n are written).
 * Synchronises with the recorded events.  With "timing" 0 (the default) nothing is recorded and
 * *n_out is 0.  Errors: TS_EINVAL, TS_ECUDA.
 */
int ts_plan_get_launch_times(ts_plan* plan, int max_n, int* kinds_out, float* ms_out, int* n_out);

int ts_plan_destroy(ts_plan* plan);           /* NULL is accepted (no-op, TS_OK) */

const char* ts_last_error(void);              /* never NULL; "" if no failure yet */

#define TS_MAX_FUSE 6

#ifdef __cplusplus
}
#endif
#endif /* TS_H_ */
