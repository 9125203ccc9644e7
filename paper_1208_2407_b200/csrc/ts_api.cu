// ts_api.cu -- the C ABI of libts (include/ts.h): validation, plan-owned scratch, pass
// scheduling.  All arithmetic is in ts_fused.cu / ts_generic.cu.
#include <math.h>
#include <string.h>

#include <new>

#include "ts_internal.h"

namespace ts {

static thread_local std::string g_last_error;

void set_error(const std::string& msg) { g_last_error = msg; }

int cuda_fail(cudaError_t e, const char* what) {
    g_last_error = std::string("CUDA error: ") + cudaGetErrorString(e) + " in " + what;
    return TS_ECUDA;
}

void LaunchTimer::begin(int kind, cudaStream_t st) {
    if (used == recs.size()) {
        Rec r{kind, nullptr, nullptr};
        if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) {
            (void)cudaGetLastError();
            return;
        }
        recs.push_back(r);
    }
    recs[used].kind = kind;
    cudaEventRecord(recs[used].a, st);
}
void LaunchTimer::end(cudaStream_t st) {
    if (used < recs.size()) cudaEventRecord(recs[used++].b, st);
}
LaunchTimer::~LaunchTimer() {
    for (Rec& r : recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
}

}  // namespace ts

struct ts_plan {
    ts::LatticeDesc L;
    int64_t nz;               // 1: two-dimensional plan; else psi[nz][ny][nx] (ts_plan_create_3d)
    int periodic_z;
    int device;
    size_t elem;              // bytes per element
    // scratch state buffer for the double-buffered fused passes
    void* scratch_re;
    void* scratch_im;
    // norm workspace
    double* norm_work;
    // device staging for ts_evolve_host
    void* host_re;
    void* host_im;
    void* host_pot;
    void* sep_pot;            // separable phase written out as planes (paths without mode 2)
    cudaStream_t own_stream;
    // ts_evolve_host: the planes go up in kFeedPieces pieces on copy_stream, one event per piece;
    // feed is set for the duration of that call only
    cudaStream_t copy_stream;
    cudaEvent_t feed_ev[8];
    const ts::RowFeed* feed;
    // options
    int64_t opt_path, opt_fuse, opt_seg, opt_variant, opt_slots, opt_chain;
    // info on the last ts_evolve
    int64_t info_fused, info_fuse, info_passes, info_launches, info_seg, info_variant;
    int64_t info_chain_x, info_chain_y;
    int64_t opt_timing;
    ts::LaunchTimer* timer;   // allocated when option "timing" is first set
};

namespace {

using ts::set_error;

int fail(int code, const char* msg) {
    set_error(msg);
    return code;
}

int check_device(const ts_plan* plan) {
    int dev = -1;
    TS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != plan->device) return fail(TS_EINVAL, "plan was created on a different CUDA device");
    return TS_OK;
}

bool coef_ok(double a, double b) {
    return isfinite(a) && isfinite(b) && fabs(a * a + b * b - 1.0) <= 1e-6;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

bool overlap(const void* a, const void* b, size_t bytes) {
    const uintptr_t x = reinterpret_cast<uintptr_t>(a), y = reinterpret_cast<uintptr_t>(b);
    return x < y + bytes && y < x + bytes;
}

// a pointer the kernels can dereference: device or managed memory (or host memory registered with
// CUDA); plain pageable host memory would fault inside the kernel
bool device_accessible(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return a.type != cudaMemoryTypeUnregistered;
}

int ensure_alloc(void** p, size_t bytes) {
    if (*p) return TS_OK;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        *p = nullptr;
        (void)cudaGetLastError();
        set_error(std::string("scratch allocation failed: ") + cudaGetErrorString(e));
        return TS_EALLOC;
    }
    return TS_OK;
}

}  // namespace

extern "C" {

const char* ts_last_error(void) { return ts::g_last_error.c_str(); }

ts_plan* ts_plan_create(int64_t nx, int64_t ny, int dtype, int boundary) {
    return ts_plan_create_xy(nx, ny, dtype, boundary, boundary);
}

ts_plan* ts_plan_create_xy(int64_t nx, int64_t ny, int dtype, int boundary, int boundary_y) {
    if (nx < 1 || ny < 1) { set_error("nx and ny must be >= 1"); return nullptr; }
    if (nx > (int64_t(1) << 31) || ny > (int64_t(1) << 31) || nx * ny >= (int64_t(1) << 62) / 16) {
        set_error("lattice too large");
        return nullptr;
    }
    if (dtype != TS_F32 && dtype != TS_F64) { set_error("unknown dtype"); return nullptr; }
    if ((boundary != TS_CLOSED && boundary != TS_PERIODIC) ||
        (boundary_y != TS_CLOSED && boundary_y != TS_PERIODIC)) {
        set_error("unknown boundary");
        return nullptr;
    }
    if ((boundary == TS_PERIODIC && nx % 2) || (boundary_y == TS_PERIODIC && ny % 2)) {
        set_error("a periodic axis needs an even extent (an odd ring cannot be split into "
                  "disjoint pairs)");
        return nullptr;
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { ts::cuda_fail(e, "cudaGetDevice"); return nullptr; }
    ts_plan* p = new (std::nothrow) ts_plan();
    if (!p) { set_error("out of host memory"); return nullptr; }
    memset(p, 0, sizeof(*p));
    p->L.nx = nx; p->L.ny = ny; p->L.dtype = dtype; p->L.periodic_x = boundary == TS_PERIODIC; p->L.periodic_y = boundary_y == TS_PERIODIC;
    p->nz = 1;
    p->device = dev;
    p->elem = dtype == TS_F32 ? 4 : 8;
    return p;
}

ts_plan* ts_plan_create_3d(int64_t nx, int64_t ny, int64_t nz, int dtype, int boundary_x,
                           int boundary_y, int boundary_z) {
    if (nz < 1) { set_error("nz must be >= 1"); return nullptr; }
    if (boundary_z != TS_CLOSED && boundary_z != TS_PERIODIC) {
        set_error("unknown boundary");
        return nullptr;
    }
    if (boundary_z == TS_PERIODIC && nz % 2) {
        set_error("a periodic axis needs an even extent (an odd ring cannot be split into "
                  "disjoint pairs)");
        return nullptr;
    }
    if (nx < 1 || ny < 1 || nx > (int64_t(1) << 31) || ny > (int64_t(1) << 31) ||
        nz > (int64_t(1) << 31) ||
        (double)nx * (double)ny * (double)nz >= (double)((int64_t(1) << 62) / 16)) {
        set_error("lattice too large");
        return nullptr;
    }
    ts_plan* p = ts_plan_create_xy(nx, ny, dtype, boundary_x, boundary_y);
    if (!p) return nullptr;
    p->nz = nz;
    p->periodic_z = boundary_z == TS_PERIODIC;
    return p;
}

int ts_plan_destroy(ts_plan* plan) {
    if (!plan) return TS_OK;
    cudaFree(plan->scratch_re);
    cudaFree(plan->scratch_im);
    cudaFree(plan->norm_work);
    cudaFree(plan->host_re);
    cudaFree(plan->host_im);
    cudaFree(plan->host_pot);
    cudaFree(plan->sep_pot);
    if (plan->own_stream) cudaStreamDestroy(plan->own_stream);
    if (plan->copy_stream) cudaStreamDestroy(plan->copy_stream);
    for (cudaEvent_t e : plan->feed_ev)
        if (e) cudaEventDestroy(e);
    delete plan->timer;
    delete plan;
    return TS_OK;
}

int ts_plan_set_option(ts_plan* plan, const char* name, int64_t value) {
    if (!plan || !name) return fail(TS_EINVAL, "NULL plan or option name");
    if (!strcmp(name, "path")) {
        if (value < 0 || value > 2) return fail(TS_EINVAL, "path must be 0, 1 or 2");
        plan->opt_path = value;
    } else if (!strcmp(name, "fuse_steps")) {
        if (value < 0 || value > TS_MAX_FUSE) return fail(TS_EINVAL, "fuse_steps out of range");
        plan->opt_fuse = value;
    } else if (!strcmp(name, "seg_rows")) {
        if (value < 0 || value % 2) return fail(TS_EINVAL, "seg_rows must be even and >= 0");
        plan->opt_seg = value;
    } else if (!strcmp(name, "variant")) {
        if (value < 0 || value > 4) return fail(TS_EINVAL, "variant must be 0 .. 4");
        plan->opt_variant = value;
    } else if (!strcmp(name, "chain")) {
        if (value < 0 || value > 64) return fail(TS_EINVAL, "chain out of range");
        plan->opt_chain = value;
    } else if (!strcmp(name, "timing")) {
        if (value != 0 && value != 1) return fail(TS_EINVAL, "timing must be 0 or 1");
        if (value && !plan->timer) {
            plan->timer = new (std::nothrow) ts::LaunchTimer();
            if (!plan->timer) return fail(TS_EALLOC, "out of host memory");
        }
        plan->opt_timing = value;
    } else if (!strcmp(name, "ring_slots")) {
        if (value < 0 || value > 64) return fail(TS_EINVAL, "ring_slots out of range");
        plan->opt_slots = value;
    } else {
        return fail(TS_EINVAL, "unknown option");
    }
    return TS_OK;
}

int ts_plan_get_info(const ts_plan* plan, const char* name, int64_t* out) {
    if (!plan || !name || !out) return fail(TS_EINVAL, "NULL argument");
    if (!strcmp(name, "fused")) *out = plan->info_fused;
    else if (!strcmp(name, "fuse_steps")) *out = plan->info_fuse;
    else if (!strcmp(name, "passes")) *out = plan->info_passes;
    else if (!strcmp(name, "launches")) *out = plan->info_launches;
    else if (!strcmp(name, "seg_rows")) *out = plan->info_seg;
    else if (!strcmp(name, "variant")) *out = plan->info_variant;
    else if (!strcmp(name, "chain_x")) *out = plan->info_chain_x;
    else if (!strcmp(name, "chain_y")) *out = plan->info_chain_y;
    else return fail(TS_EINVAL, "unknown info name");
    return TS_OK;
}

}  // extern "C"

namespace {

struct SubStep {
    ts::StepCoef c;
    ts::Phase ph;      // the diagonal step of this sub-step
};

bool same_phase(const ts::Phase& a, const ts::Phase& b) {
    return a.mode == b.mode && a.planes == b.planes && a.px == b.px && a.py == b.py;
}

// psi <- (U2(pat[P-1]) ... U2(pat[0]))^n_repeat psi: the engine behind ts_evolve (P = 1) and
// ts_evolve_u4 (P = 5).  Consecutive sub-steps that share a potential-phase array are fused into
// passes of up to S sub-steps; passes ping-pong between the caller's planes and the scratch.
int evolve_pattern(ts_plan* plan, void* psi_re, void* psi_im, const SubStep* pat, int period,
                   int64_t n_repeat, void* cuda_stream) {
    if (!plan) return fail(TS_EINVAL, "NULL plan");
    if (plan->nz != 1) return fail(TS_EINVAL, "three-dimensional plan: use ts_evolve_3d");
    if (!psi_re || !psi_im) return fail(TS_EINVAL, "NULL psi plane");
    if (n_repeat < 0) return fail(TS_EINVAL, "n_steps < 0");
    const ts::LatticeDesc& L = plan->L;
    const size_t plane_bytes = (size_t)L.nx * (size_t)L.ny * plan->elem;
    if (!aligned16(psi_re) || !aligned16(psi_im))
        return fail(TS_EINVAL, "device pointers must be 16-byte aligned");
    if (overlap(psi_re, psi_im, plane_bytes)) return fail(TS_EINVAL, "psi_re and psi_im overlap");
    if (!device_accessible(psi_re) || !device_accessible(psi_im))
        return fail(TS_EINVAL, "psi planes must be device memory (ts_evolve_host takes host planes)");
    bool any_pot = false, any_sep = false, can_v1 = true, can_stream = true;
    for (int k = 0; k < period; ++k) {
        const ts::StepCoef& c = pat[k].c;
        if (!coef_ok(c.a_h, c.b_h) || !coef_ok(c.a_f, c.b_f))
            return fail(TS_EINVAL, "coefficients must be finite with |a^2 + b^2 - 1| <= 1e-6");
        const ts::Phase& ph = pat[k].ph;
        if (ph.mode == 1) {
            const void* pot = ph.planes;
            any_pot = true;
            if (!aligned16(pot)) return fail(TS_EINVAL, "device pointers must be 16-byte aligned");
            if (!device_accessible(pot)) return fail(TS_EINVAL, "pot_phase must be device memory");
            if (overlap(pot, psi_re, plane_bytes) || overlap(pot, psi_im, plane_bytes) ||
                overlap((const char*)pot + plane_bytes, psi_re, plane_bytes) ||
                overlap((const char*)pot + plane_bytes, psi_im, plane_bytes))
                return fail(TS_EINVAL, "pot_phase overlaps psi");
        } else if (ph.mode == 2) {
            any_pot = any_sep = true;
            if (!ph.px || !ph.py) return fail(TS_EINVAL, "NULL separable phase vector");
            if (!aligned16(ph.px) || !aligned16(ph.py))
                return fail(TS_EINVAL, "device pointers must be 16-byte aligned");
            if (!device_accessible(ph.px) || !device_accessible(ph.py))
                return fail(TS_EINVAL, "the separable phase vectors must be device memory");
        }
        can_v1 = can_v1 && ts::fused_supported(L, c);
        can_stream = can_stream && ts::stream_supported(L, c);
    }
    // sub-steps chained inside a pass merge their adjacent half sweeps: that angle, too, must
    // stay away from 90 degrees for the tangent form
    for (int k = 0; k < period && period > 1; ++k) {
        const ts::StepCoef& u = pat[k].c;
        const ts::StepCoef& v = pat[(k + 1) % period].c;
        if (u.a_h * v.a_h - u.b_h * v.b_h <= 0.25) can_v1 = can_stream = false;
    }
    const bool can_fuse = can_v1 || can_stream;
    // steps without a potential factorise into a row chain and a column chain (ts_axis.cu)
    ts::StepCoef axis_pat[8];
    bool can_axis = !any_pot && period <= 8;
    if (can_axis) {
        for (int k = 0; k < period; ++k) axis_pat[k] = pat[k].c;
        can_axis = ts::axis_supported(L, axis_pat, period);
    }
    int rc = check_device(plan);
    if (rc != TS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    ts::LaunchTimer* tm = plan->opt_timing ? plan->timer : nullptr;
    if (plan->timer) plan->timer->reset();

    plan->info_fused = plan->info_fuse = plan->info_passes = plan->info_launches = 0;
    plan->info_seg = plan->info_variant = plan->info_chain_x = plan->info_chain_y = 0;
    if (n_repeat == 0) return TS_OK;
    if (period > 1 && n_repeat > (int64_t(1) << 56)) return fail(TS_EINVAL, "n_steps too large");
    const int64_t n_sub = n_repeat * period;

    // ---- which path: every rejection comes before the first allocation or launch -----------------
    // tiny lattices: the whole evolution in one launch of the on-chip-resident kernel (uniform
    // steps, no or plane potential)
    const bool can_tiny = period == 1 && pat[0].ph.mode != 2 &&
                          ts::tiny_supported(L, pat[0].c, pat[0].ph.mode == 1);
    const int64_t variant = plan->opt_variant;
    if (variant == 3 && !can_tiny)
        return fail(TS_EUNSUPPORTED, "the on-chip kernel takes uniform steps on lattices of at most "
                                     "128 x 128 (fp32) / 128 x 64 (fp64) sites, half with a potential");
    if (variant == 4 && !can_axis)
        return fail(TS_EUNSUPPORTED, "the axis-split path takes steps without a potential, nx % 4 == 0, "
                                     "even ny, cos of every sweep angle > 0.25");
    if (plan->opt_path == 2 && !can_fuse && !can_axis)
        return fail(TS_EUNSUPPORTED,
                    "fused kernel needs nx % 4 == 0, even ny and cos(theta) > 0.25");
    if (variant == 2 && !can_stream)
        return fail(TS_EUNSUPPORTED, "the TMA ring kernel needs nx >= 128 on a lattice that is periodic in x");
    if (variant == 1 && !can_v1)
        return fail(TS_EUNSUPPORTED, "the register-prefetch kernel needs one boundary type on both axes");
    const bool generic = plan->opt_path == 1 || (!can_fuse && !can_axis);
    const bool use_axis = !generic && can_axis && (variant == 0 || variant == 4);
    const bool use_tiny = !generic && !use_axis && can_tiny && (variant == 0 || variant == 3);
    const bool use_stream = !generic && !use_axis && !use_tiny && can_stream && variant != 1;
    if (!generic && !use_axis && !use_tiny && !can_fuse)
        return fail(TS_EUNSUPPORTED, "the requested kernel variant does not take this lattice");
    const bool expand_sep = any_sep && !use_stream;
    if (expand_sep && period != 1)
        return fail(TS_EUNSUPPORTED, "separable phases of a multi-sub-step pattern need the TMA ring kernel");
    int S = 0, s_max = 0;
    if (!generic && !use_axis && !use_tiny) {
        S = plan->opt_fuse ? (int)plan->opt_fuse
                           : (any_sep && use_stream ? ts::stream_default_steps_sep(L)
                                                    : ts::fused_default_steps(L, any_pot));
        s_max = use_stream ? ts::stream_max_steps(L, any_pot) : 4;
        if (S > s_max) {
            if (plan->opt_fuse)
                return fail(TS_EUNSUPPORTED, "fuse_steps > 4 needs the TMA ring kernel, fp32, no potential");
            S = s_max;
        }
    }

    // host-fed planes (ts_evolve_host): only the axis-split path starts on a part of the rows
    if (plan->feed && !use_axis && plan->feed->n > 0)
        TS_CUDA_TRY(cudaStreamWaitEvent(st, plan->feed->ready[plan->feed->n - 1], 0));
    if (use_axis) {
        if (ts::axis_needs_scratch(L)) {
            rc = ensure_alloc(&plan->scratch_re, plane_bytes);
            if (rc == TS_OK) rc = ensure_alloc(&plan->scratch_im, plane_bytes);
            if (rc != TS_OK) return rc;
        }
        ts::AxisInfo ai;
        rc = ts::axis_evolve(L, psi_re, psi_im, plan->scratch_re, plan->scratch_im, axis_pat, period,
                             n_sub, (int)plan->opt_chain, (int)plan->opt_seg, (int)plan->opt_slots,
                             st, &ai, tm, plan->feed);
        plan->info_launches = ai.launches;
        if (rc != TS_OK) return rc;
        plan->info_fused = 1; plan->info_passes = ai.passes; plan->info_seg = ai.seg_rows;
        plan->info_chain_x = ai.chain_x; plan->info_chain_y = ai.chain_y;
        plan->info_fuse = ai.chain_y; plan->info_variant = 4;
        return TS_OK;
    }
    if (use_tiny) {
        ts::timer_begin(tm, ts::kKindTiny, st);
        rc = ts::tiny_evolve(L, psi_re, psi_im, pat[0].c, pat[0].ph.planes, n_repeat,
                             (int)plan->opt_seg, st);     // "seg_rows" = rows per warp here
        ts::timer_end(tm, st);
        if (rc != TS_OK) return rc;
        plan->info_fused = 1; plan->info_fuse = n_repeat; plan->info_passes = 1;
        plan->info_launches = 1; plan->info_seg = L.ny; plan->info_variant = 3;
        return TS_OK;
    }
    // separable factors are consumed directly only by the TMA ring kernel; every other path gets
    // them written out as planes (one array: period-1 patterns only)
    SubStep expanded;
    if (expand_sep) {
        rc = ensure_alloc(&plan->sep_pot, 2 * plane_bytes);
        if (rc != TS_OK) return rc;
        ts::timer_begin(tm, ts::kKindExpand, st);
        rc = ts::expand_separable(L, pat[0].ph.px, pat[0].ph.py, plan->sep_pot, st);
        ts::timer_end(tm, st);
        if (rc != TS_OK) return rc;
        ++plan->info_launches;
        expanded = pat[0];
        expanded.ph = ts::Phase{1, plan->sep_pot, nullptr, nullptr};
        pat = &expanded;
    }
    if (generic) {
        const int64_t l0 = plan->info_launches;
        if (period == 1) {
            ts::timer_begin(tm, ts::kKindGeneric, st);
            rc = ts::generic_evolve(L, psi_re, psi_im, pat[0].c, pat[0].ph.planes, n_repeat, st,
                                    &plan->info_launches);
            ts::timer_end(tm, st);
            plan->info_launches += l0;
            return rc;
        }
        for (int64_t i = 0; i < n_sub; ++i) {
            const SubStep& s = pat[i % period];
            int64_t launches = 0;
            rc = ts::generic_evolve(L, psi_re, psi_im, s.c, s.ph.planes, 1, st, &launches);
            if (rc != TS_OK) return rc;
            plan->info_launches += launches;
        }
        return TS_OK;
    }

    rc = ensure_alloc(&plan->scratch_re, plane_bytes);
    if (rc == TS_OK) rc = ensure_alloc(&plan->scratch_im, plane_bytes);
    if (rc != TS_OK) return rc;

    // resident blocks per SM of the kernel that will run: fp64 with phase planes (28 KB of rings per
    // warp) or beyond S = 2 (255 registers) two, everything else three
    const bool planes = any_pot && !(any_sep && use_stream);
    const int bpsm = (L.dtype == TS_F64 && (planes || S > 2)) ? 2 : 3;
    // an explicit "seg_rows" means equal segments; by default the tile kernel's edge warps get
    // shorter ones (stream_default_seg)
    const ts::SegShape sseg = plan->opt_seg ? ts::SegShape{(int)plan->opt_seg, 0}
                                            : ts::stream_default_seg(L, S, bpsm);
    const int seg = use_stream ? sseg.rows
                               : plan->opt_seg ? (int)plan->opt_seg
                                               : ts::fused_default_seg_rows(L, S, bpsm);
    plan->info_variant = use_stream ? 2 : 1;
    void* cur_re = psi_re; void* cur_im = psi_im;
    void* nxt_re = plan->scratch_re; void* nxt_im = plan->scratch_im;
    int64_t i = 0;
    while (i < n_sub) {
        // the run of sub-steps of this pass: same potential array; the register-prefetch kernel
        // (variant 1) also needs equal angles
        ts::StepCoef subs[TS_MAX_FUSE];
        const ts::Phase ph = pat[i % period].ph;
        int s = 0;
        while (s < S && i + s < n_sub) {
            const SubStep& x = pat[(i + s) % period];
            if (!same_phase(x.ph, ph)) break;
            if (!use_stream && s > 0 && memcmp(&x.c, &subs[0], sizeof(ts::StepCoef)) != 0) break;
            subs[s++] = x.c;
        }
        ts::timer_begin(tm, use_stream ? ts::kKindStream : ts::kKindFused, st);
        if (use_stream)
            rc = ts::stream_pass(L, cur_re, cur_im, nxt_re, nxt_im, subs, ph, s, sseg,
                                 (int)plan->opt_slots, st);
        else
            rc = ts::fused_pass(L, cur_re, cur_im, nxt_re, nxt_im, subs[0], ph.planes, s, seg, st);
        ts::timer_end(tm, st);
        if (rc != TS_OK) return rc;
        void* t;
        t = cur_re; cur_re = nxt_re; nxt_re = t;
        t = cur_im; cur_im = nxt_im; nxt_im = t;
        i += s;
        ++plan->info_passes;
        ++plan->info_launches;
    }
    if (cur_re != psi_re) {   // odd number of passes: the result sits in the scratch buffer
        ts::timer_begin(tm, ts::kKindCopy, st);
        TS_CUDA_TRY(cudaMemcpyAsync(psi_re, cur_re, plane_bytes, cudaMemcpyDeviceToDevice, st));
        TS_CUDA_TRY(cudaMemcpyAsync(psi_im, cur_im, plane_bytes, cudaMemcpyDeviceToDevice, st));
        ts::timer_end(tm, st);
        plan->info_launches += 2;
    }
    plan->info_fused = 1;
    plan->info_fuse = S;
    plan->info_seg = seg;
    return TS_OK;
}

}  // namespace

extern "C" {

int ts_evolve(ts_plan* plan, void* psi_re, void* psi_im, double a_half, double b_half,
              double a_full, double b_full, const void* pot, int64_t n_steps, void* cuda_stream) {
    const SubStep one{{a_half, b_half, a_full, b_full},
                      ts::Phase{pot ? 1 : 0, pot, nullptr, nullptr}};
    return evolve_pattern(plan, psi_re, psi_im, &one, 1, n_steps, cuda_stream);
}

int ts_evolve_3d(ts_plan* plan, void* psi_re, void* psi_im, double a_half, double b_half,
                 double a_full, double b_full, const void* pot, int64_t n_steps, void* cuda_stream) {
    if (!plan) return fail(TS_EINVAL, "NULL plan");
    if (!psi_re || !psi_im) return fail(TS_EINVAL, "NULL psi plane");
    if (n_steps < 0) return fail(TS_EINVAL, "n_steps < 0");
    const ts::Lattice3 L{plan->L.nx, plan->L.ny, plan->nz, plan->L.dtype,
                         {plan->L.periodic_x, plan->L.periodic_y, plan->periodic_z}};
    const size_t vol_bytes = (size_t)L.nx * (size_t)L.ny * (size_t)L.nz * plan->elem;
    if (!aligned16(psi_re) || !aligned16(psi_im) || (pot && !aligned16(pot)))
        return fail(TS_EINVAL, "device pointers must be 16-byte aligned");
    if (overlap(psi_re, psi_im, vol_bytes)) return fail(TS_EINVAL, "psi_re and psi_im overlap");
    if (!device_accessible(psi_re) || !device_accessible(psi_im) || (pot && !device_accessible(pot)))
        return fail(TS_EINVAL, "psi planes and pot_phase must be device memory");
    if (pot && (overlap(pot, psi_re, vol_bytes) || overlap(pot, psi_im, vol_bytes) ||
                overlap((const char*)pot + vol_bytes, psi_re, vol_bytes) ||
                overlap((const char*)pot + vol_bytes, psi_im, vol_bytes)))
        return fail(TS_EINVAL, "pot_phase overlaps psi");
    if (!coef_ok(a_half, b_half) || !coef_ok(a_full, b_full))
        return fail(TS_EINVAL, "coefficients must be finite with |a^2 + b^2 - 1| <= 1e-6");
    const ts::StepCoef c{a_half, b_half, a_full, b_full};
    const bool can_axis = ts::axis3_supported(L, c);
    if ((plan->opt_path == 2 || plan->opt_variant == 4) && !can_axis)
        return fail(TS_EUNSUPPORTED, "the fused 3-D path needs even extents that fit a thread block "
                                     "(<= 16384 sites fp32, 8192 fp64, per axis) and cos of every "
                                     "sweep angle > 0.25");
    if (plan->opt_variant != 0 && plan->opt_variant != 4)
        return fail(TS_EUNSUPPORTED, "3-D plans run on the axis path (variant 4) or the per-sweep kernels");
    int rc = check_device(plan);
    if (rc != TS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    ts::LaunchTimer* tm = plan->opt_timing ? plan->timer : nullptr;
    if (plan->timer) plan->timer->reset();
    plan->info_fused = plan->info_fuse = plan->info_passes = plan->info_launches = 0;
    plan->info_seg = plan->info_variant = plan->info_chain_x = plan->info_chain_y = 0;
    if (n_steps == 0) return TS_OK;
    if (can_axis && plan->opt_path != 1) {
        ts::AxisInfo ai;
        rc = ts::axis3_evolve(L, psi_re, psi_im, c, pot, n_steps, st, &ai, tm);
        plan->info_launches = ai.launches;
        if (rc != TS_OK) return rc;
        plan->info_fused = 1; plan->info_passes = ai.passes; plan->info_variant = 4;
        plan->info_chain_x = ai.chain_x; plan->info_chain_y = ai.chain_y;
        plan->info_fuse = pot ? 1 : n_steps;
        return TS_OK;
    }
    ts::timer_begin(tm, ts::kKindGeneric, st);
    rc = ts::generic3_evolve(L, psi_re, psi_im, c, pot, n_steps, st, &plan->info_launches);
    ts::timer_end(tm, st);
    return rc;
}

int ts_evolve_sep(ts_plan* plan, void* psi_re, void* psi_im, double a_half, double b_half,
                  double a_full, double b_full, const void* phase_x, const void* phase_y,
                  int64_t n_steps, void* cuda_stream) {
    if (!phase_x || !phase_y) return fail(TS_EINVAL, "NULL separable phase vector");
    const SubStep one{{a_half, b_half, a_full, b_full}, ts::Phase{2, nullptr, phase_x, phase_y}};
    return evolve_pattern(plan, psi_re, psi_im, &one, 1, n_steps, cuda_stream);
}

int ts_slab_pass(ts_plan* plan, const void* src_re, const void* src_im, void* dst_re,
                 void* dst_im, const void* up_re, const void* up_im, int64_t up_rows,
                 const void* dn_re, const void* dn_im, int64_t dn_rows, const double* coef,
                 int n_sub, const void* phase_x, const void* phase_y, int64_t y0,
                 int64_t ny_global, int periodic_y_global, void* cuda_stream) {
    if (!plan) return fail(TS_EINVAL, "NULL plan");
    if (plan->nz != 1) return fail(TS_EINVAL, "three-dimensional plan: use ts_evolve_3d");
    if (!src_re || !src_im || !dst_re || !dst_im) return fail(TS_EINVAL, "NULL psi plane");
    if (!coef) return fail(TS_EINVAL, "NULL coefficient table");
    if ((up_re == nullptr) != (up_im == nullptr) || (dn_re == nullptr) != (dn_im == nullptr))
        return fail(TS_EINVAL, "give both planes of a neighbour or neither");
    if ((phase_x == nullptr) != (phase_y == nullptr))
        return fail(TS_EINVAL, "give both separable phase vectors or neither");
    const ts::LatticeDesc& L = plan->L;
    if (L.periodic_y)
        return fail(TS_EINVAL, "a slab plan is closed in y (ts_plan_create_xy(.., bx, TS_CLOSED))");
    const size_t plane_bytes = (size_t)L.nx * (size_t)L.ny * plan->elem;
    const void* ptrs[10] = {src_re, src_im, dst_re, dst_im, up_re, up_im, dn_re, dn_im, phase_x,
                            phase_y};
    for (const void* q : ptrs) {
        if (q && !aligned16(q)) return fail(TS_EINVAL, "device pointers must be 16-byte aligned");
        if (q && !device_accessible(q)) return fail(TS_EINVAL, "planes must be device (or peer-mapped) memory");
    }
    if (overlap(src_re, dst_re, plane_bytes) || overlap(src_im, dst_im, plane_bytes) ||
        overlap(src_re, dst_im, plane_bytes) || overlap(src_im, dst_re, plane_bytes))
        return fail(TS_EINVAL, "ts_slab_pass works out of place: src and dst overlap");
    const bool sep = phase_x != nullptr;
    const int s_max = ts::stream_max_steps(L, sep);
    if (n_sub < 1 || n_sub > s_max) return fail(TS_EINVAL, "n_sub out of range for this dtype");
    ts::StepCoef subs[TS_MAX_FUSE];
    for (int j = 0; j < n_sub; ++j) {
        subs[j] = ts::StepCoef{coef[4 * j], coef[4 * j + 1], coef[4 * j + 2], coef[4 * j + 3]};
        if (!coef_ok(subs[j].a_h, subs[j].b_h) || !coef_ok(subs[j].a_f, subs[j].b_f))
            return fail(TS_EINVAL, "coefficients must be finite with |a^2 + b^2 - 1| <= 1e-6");
        bool ok = ts::stream_supported(L, subs[j]);
        if (ok && j > 0)   // the merged half sweeps between chained sub-steps
            ok = subs[j - 1].a_h * subs[j].a_h - subs[j - 1].b_h * subs[j].b_h > 0.25;
        if (!ok)
            return fail(TS_EUNSUPPORTED, "ts_slab_pass runs on the TMA ring kernel only: nx >= 128, "
                                         "nx % 4 == 0, even ny, cos of every sweep angle > 0.25");
    }
    // the halo a pass consumes: 2 rows per sub-step from each neighbour
    if ((up_re && up_rows < 2 * n_sub) || (dn_re && dn_rows < 2 * n_sub))
        return fail(TS_EINVAL, "a neighbour has fewer than 2 * n_sub rows");
    if (up_rows % 2 || dn_rows % 2) return fail(TS_EINVAL, "neighbour row counts must be even");
    ts::Phase ph{0, nullptr, nullptr, nullptr};
    if (sep) {
        if (ny_global < L.ny || y0 < 0 || y0 + L.ny > ny_global || y0 % 2)
            return fail(TS_EINVAL, "the slab [y0, y0 + ny) must lie inside the global lattice, y0 even");
        ph.mode = 2; ph.px = phase_x; ph.py = phase_y;
        ph.py_off = y0; ph.py_n = ny_global; ph.py_wrap = periodic_y_global != 0;
    }
    int rc = check_device(plan);
    if (rc != TS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const ts::Peers peers{up_re, up_im, up_rows, dn_re, dn_im, dn_rows};
    // slabs: equal segments (the cut rows of a slab are not lattice edges)
    const int seg = plan->opt_seg ? (int)plan->opt_seg : ts::stream_default_seg(L, n_sub, 3).rows;
    rc = ts::stream_pass(L, src_re, src_im, dst_re, dst_im, subs, ph, n_sub, ts::SegShape{seg, 0},
                         (int)plan->opt_slots, st, &peers);
    if (rc != TS_OK) return rc;
    plan->info_fused = 1; plan->info_fuse = n_sub; plan->info_passes = 1; plan->info_launches = 1;
    plan->info_seg = seg; plan->info_variant = 2;
    return TS_OK;
}

int ts_evolve_tdep(ts_plan* plan, void* psi_re, void* psi_im, double a_half, double b_half,
                   double a_full, double b_full, const void* const* pot_phases, int64_t n_steps,
                   void* cuda_stream) {
    if (n_steps < 0) return fail(TS_EINVAL, "n_steps < 0");
    if (n_steps > 0 && !pot_phases) return fail(TS_EINVAL, "NULL list of potential phases");
    if (n_steps > (int64_t(1) << 24)) return fail(TS_EINVAL, "n_steps too large for one call");
    // one sub-step per time step, each with its own phase array: consecutive steps that happen to
    // share an array are still fused into one pass
    SubStep* pat = n_steps ? new (std::nothrow) SubStep[(size_t)n_steps] : nullptr;
    if (n_steps && !pat) return fail(TS_EALLOC, "out of host memory");
    for (int64_t k = 0; k < n_steps; ++k) {
        pat[k].c = ts::StepCoef{a_half, b_half, a_full, b_full};
        pat[k].ph = ts::Phase{pot_phases[k] ? 1 : 0, pot_phases[k], nullptr, nullptr};
    }
    const SubStep none{{a_half, b_half, a_full, b_full}, ts::Phase{0, nullptr, nullptr, nullptr}};
    const int rc = n_steps ? evolve_pattern(plan, psi_re, psi_im, pat, (int)n_steps, 1, cuda_stream)
                           : evolve_pattern(plan, psi_re, psi_im, &none, 1, 0, cuda_stream);
    delete[] pat;
    return rc;
}

int ts_u4_coefficients(double theta, double* out20) {
    if (!out20) return fail(TS_EINVAL, "NULL output table");
    if (!isfinite(theta)) return fail(TS_EINVAL, "theta must be finite");
    // Eq. 4: U4(dt) = U2(p dt) U2(p dt) U2((1-4p) dt) U2(p dt) U2(p dt)
    const double p = 1.0 / (4.0 - cbrt(4.0));
    const double frac[5] = {p, p, 1.0 - 4.0 * p, p, p};
    for (int k = 0; k < 5; ++k) {
        const double th = frac[k] * theta;
        out20[4 * k] = cos(0.5 * th); out20[4 * k + 1] = sin(0.5 * th);
        out20[4 * k + 2] = cos(th); out20[4 * k + 3] = sin(th);
    }
    return TS_OK;
}

int ts_evolve_u4(ts_plan* plan, void* psi_re, void* psi_im, double theta, const void* pot_p,
                 const void* pot_q, int64_t n_steps, void* cuda_stream) {
    if ((pot_p == nullptr) != (pot_q == nullptr))
        return fail(TS_EINVAL, "give both potential-phase arrays of the fourth-order step or neither");
    if (!isfinite(theta)) return fail(TS_EINVAL, "theta must be finite");
    double coef[20];
    ts_u4_coefficients(theta, coef);
    SubStep pat[5];
    for (int k = 0; k < 5; ++k) {
        pat[k].c = ts::StepCoef{coef[4 * k], coef[4 * k + 1], coef[4 * k + 2], coef[4 * k + 3]};
        const void* pot = k == 2 ? pot_q : pot_p;
        pat[k].ph = ts::Phase{pot ? 1 : 0, pot, nullptr, nullptr};
    }
    return evolve_pattern(plan, psi_re, psi_im, pat, 5, n_steps, cuda_stream);
}

int ts_plan_reserve(ts_plan* plan, int with_host_staging) {
    if (!plan) return fail(TS_EINVAL, "NULL plan");
    int rc = check_device(plan);
    if (rc != TS_OK) return rc;
    const size_t plane_bytes = (size_t)plan->L.nx * (size_t)plan->L.ny * plan->elem;
    if (plan->nz == 1) {      // the 3-D paths work in place
        rc = ensure_alloc(&plan->scratch_re, plane_bytes);
        if (rc == TS_OK) rc = ensure_alloc(&plan->scratch_im, plane_bytes);
    }
    if (rc == TS_OK)
        rc = ensure_alloc(reinterpret_cast<void**>(&plan->norm_work),
                          ts::norm_workspace_doubles() * sizeof(double));
    if (rc == TS_OK && with_host_staging) {
        rc = ensure_alloc(&plan->host_re, plane_bytes);
        if (rc == TS_OK) rc = ensure_alloc(&plan->host_im, plane_bytes);
        if (rc == TS_OK && with_host_staging == 2) rc = ensure_alloc(&plan->host_pot, 2 * plane_bytes);
    }
    return rc;
}

int ts_plan_get_launch_times(ts_plan* plan, int max_n, int* kinds_out, float* ms_out, int* n_out) {
    if (!plan || !n_out || max_n < 0 || (max_n > 0 && (!kinds_out || !ms_out)))
        return fail(TS_EINVAL, "NULL argument");
    *n_out = 0;
    if (!plan->timer) return TS_OK;
    const ts::LaunchTimer& t = *plan->timer;
    *n_out = (int)t.used;
    for (size_t i = 0; i < t.used && (int)i < max_n; ++i) {
        TS_CUDA_TRY(cudaEventSynchronize(t.recs[i].b));
        float ms = 0.f;
        TS_CUDA_TRY(cudaEventElapsedTime(&ms, t.recs[i].a, t.recs[i].b));
        kinds_out[i] = t.recs[i].kind;
        ms_out[i] = ms;
    }
    return TS_OK;
}

int ts_norm(ts_plan* plan, const void* psi_re, const void* psi_im, double* out, void* cuda_stream) {
    if (!plan) return fail(TS_EINVAL, "NULL plan");
    if (!psi_re || !psi_im || !out) return fail(TS_EINVAL, "NULL argument");
    if (!device_accessible(psi_re) || !device_accessible(psi_im))
        return fail(TS_EINVAL, "psi planes must be device memory");
    int rc = check_device(plan);
    if (rc != TS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    rc = ensure_alloc(reinterpret_cast<void**>(&plan->norm_work),
                      ts::norm_workspace_doubles() * sizeof(double));
    if (rc != TS_OK) return rc;
    ts::LatticeDesc flat = plan->L;     // a 3-D state is nz * ny rows of nx sites
    flat.ny *= plan->nz;
    rc = ts::norm2_device(flat, psi_re, psi_im, plan->norm_work, st);
    if (rc != TS_OK) return rc;
    TS_CUDA_TRY(cudaMemcpyAsync(out, plan->norm_work, sizeof(double), cudaMemcpyDeviceToHost, st));
    TS_CUDA_TRY(cudaStreamSynchronize(st));
    return TS_OK;
}

int ts_evolve_host(ts_plan* plan, void* re_h, void* im_h, double a_half, double b_half,
                   double a_full, double b_full, const void* pot_h, int64_t n_steps) {
    if (!plan) return fail(TS_EINVAL, "NULL plan");
    if (!re_h || !im_h) return fail(TS_EINVAL, "NULL psi plane");
    int rc = check_device(plan);
    if (rc != TS_OK) return rc;
    const size_t plane_bytes = (size_t)plan->L.nx * (size_t)plan->L.ny * plan->elem;
    rc = ensure_alloc(&plan->host_re, plane_bytes);
    if (rc == TS_OK) rc = ensure_alloc(&plan->host_im, plane_bytes);
    if (rc == TS_OK && pot_h) rc = ensure_alloc(&plan->host_pot, 2 * plane_bytes);
    if (rc != TS_OK) return rc;
    if (!plan->own_stream)
        TS_CUDA_TRY(cudaStreamCreateWithFlags(&plan->own_stream, cudaStreamNonBlocking));
    cudaStream_t st = plan->own_stream;
    // Without a potential the step factorises into a row chain and a column chain (ts_axis.cu) and
    // rows are independent lines: the planes go up in pieces on a second stream and the row chain
    // of a piece runs while the next piece is on the bus (C4: the 8.6 ms of the row chain hidden
    // behind the 39 ms of the upload).  Paths that need the whole lattice wait for the last piece.
    constexpr int kFeedPieces = 8;
    const bool pieces = !pot_h && plan->nz == 1 && plan->L.ny >= 64 * kFeedPieces &&
                        plane_bytes >= (size_t(8) << 20);
    if (pieces) {
        if (!plan->copy_stream)
            TS_CUDA_TRY(cudaStreamCreateWithFlags(&plan->copy_stream, cudaStreamNonBlocking));
        for (int k = 0; k < kFeedPieces; ++k)
            if (!plan->feed_ev[k])
                TS_CUDA_TRY(cudaEventCreateWithFlags(&plan->feed_ev[k], cudaEventDisableTiming));
        cudaStream_t cs = plan->copy_stream;
        int64_t y_end[kFeedPieces];
        const size_t row_bytes = (size_t)plan->L.nx * plan->elem;
        int64_t y0 = 0;
        for (int k = 0; k < kFeedPieces; ++k) {
            int64_t y1 = plan->L.ny * (k + 1) / kFeedPieces;
            y1 -= y1 % 2;
            if (k == kFeedPieces - 1) y1 = plan->L.ny;
            y_end[k] = y1;
            const size_t off = (size_t)y0 * row_bytes, nb = (size_t)(y1 - y0) * row_bytes;
            cudaError_t e = cudaMemcpyAsync((char*)plan->host_re + off, (const char*)re_h + off, nb,
                                            cudaMemcpyHostToDevice, cs);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync((char*)plan->host_im + off, (const char*)im_h + off, nb,
                                    cudaMemcpyHostToDevice, cs);
            if (e == cudaSuccess) e = cudaEventRecord(plan->feed_ev[k], cs);
            if (e != cudaSuccess) {
                cudaStreamSynchronize(cs);
                return ts::cuda_fail(e, "ts_evolve_host: upload");
            }
            y0 = y1;
        }
        const ts::RowFeed feed{kFeedPieces, y_end, plan->feed_ev};
        plan->feed = &feed;
        rc = ts_evolve(plan, plan->host_re, plan->host_im, a_half, b_half, a_full, b_full, nullptr,
                       n_steps, st);
        plan->feed = nullptr;
        if (rc != TS_OK) {
            cudaStreamSynchronize(cs);
            cudaStreamSynchronize(st);
            return rc;
        }
        // (a call of zero steps enqueues nothing that waits for the upload)
        TS_CUDA_TRY(cudaStreamWaitEvent(st, plan->feed_ev[kFeedPieces - 1], 0));
    } else {
        TS_CUDA_TRY(cudaMemcpyAsync(plan->host_re, re_h, plane_bytes, cudaMemcpyHostToDevice, st));
        TS_CUDA_TRY(cudaMemcpyAsync(plan->host_im, im_h, plane_bytes, cudaMemcpyHostToDevice, st));
        if (pot_h)
            TS_CUDA_TRY(cudaMemcpyAsync(plan->host_pot, pot_h, 2 * plane_bytes,
                                        cudaMemcpyHostToDevice, st));
        rc = ts_evolve(plan, plan->host_re, plan->host_im, a_half, b_half, a_full, b_full,
                       pot_h ? plan->host_pot : nullptr, n_steps, st);
        if (rc != TS_OK) {
            cudaStreamSynchronize(st);      // the uploads still read the caller's planes
            return rc;
        }
    }
    TS_CUDA_TRY(cudaMemcpyAsync(re_h, plan->host_re, plane_bytes, cudaMemcpyDeviceToHost, st));
    TS_CUDA_TRY(cudaMemcpyAsync(im_h, plan->host_im, plane_bytes, cudaMemcpyDeviceToHost, st));
    TS_CUDA_TRY(cudaStreamSynchronize(st));
    return TS_OK;
}

}  // extern "C"
