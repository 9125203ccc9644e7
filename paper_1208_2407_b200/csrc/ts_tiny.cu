// ts_tiny.cu -- lattices small enough to LIVE ON CHIP for the whole evolution.
//
// One thread block holds the whole wavefunction in registers -- a warp owns R consecutive rows, a
// lane 4 consecutive sites of each of them (nx <= 128) -- and applies all n_steps second-order
// steps in ONE launch: horizontal sweeps in registers and warp shuffles, the vertical-even sweep
// and the interior pairs of the vertical-odd sweep in registers, and only the vertical-odd pairs
// that straddle two warps through shared memory (two block barriers per such sweep).  HBM is
// touched twice: load at the start, store at the end.  The streaming kernel needs a pass (a
// launch, a prologue and 2S warm-up iterations per segment) per S steps, which is what bounds it
// on a 64 x 64 lattice (C1: 7 us per pass of 4 steps).
//
// Stage list, coefficients and boundary rules are those of ts_evolve (include/ts.h); the
// arithmetic is the scaled rotation of ts_rows.cuh with the deferred cosines multiplied in once
// per step (a whole evolution's worth would leave the fp32 range).
#include <math.h>

#include "ts_internal.h"
#include "ts_rows.cuh"

namespace ts {
namespace {

using namespace rows;

template <typename T>
struct TinyParams {
    T* re;
    T* im;
    const T* pot_re;
    const T* pot_im;
    int nx, ny;
    int64_t n_steps;
    T t_h, t_f, sec_h, sec_f;
    T scale4;         // deferred cosines of FOUR steps, (a_h^6 a_f)^4 or a_h^32, rounded to T
    T final_scale;    // the steps after the last multiple of four, and the accumulated rounding
                      // of scale4 taken out again
};

// me <- me + i t other (one side of a pair rotation whose partner lives in another warp)
template <typename T>
__device__ __forceinline__ void half_pair(Row4<T>& me, const Row4<T>& other, T t) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        me.re[i] = fma(-t, other.im[i], me.re[i]);
        me.im[i] = fma(t, other.re[i], me.im[i]);
    }
}

// 16-byte shared-memory accesses of a lane's four sites (conflict-free in fp32)
__device__ __forceinline__ void put4(float* d, const float (&v)[4]) {
    *reinterpret_cast<float4*>(d) = make_float4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void put4(double* d, const double (&v)[4]) {
    reinterpret_cast<double2*>(d)[0] = make_double2(v[0], v[1]);
    reinterpret_cast<double2*>(d)[1] = make_double2(v[2], v[3]);
}
__device__ __forceinline__ void get4(const float* s, float (&v)[4]) {
    const float4 q = *reinterpret_cast<const float4*>(s);
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
}
__device__ __forceinline__ void get4(const double* s, double (&v)[4]) {
    const double2 a = reinterpret_cast<const double2*>(s)[0];
    const double2 b = reinterpret_cast<const double2*>(s)[1];
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}

// X-odd sweep on a ring shorter than the warp: the cross-lane partners come from explicit lanes
template <typename T>
__device__ __forceinline__ void xo_ring(Row4<T>& r, T t, int up_src, int dn_src) {
    const T up_re = __shfl_sync(0xffffffffu, r.re[3], up_src);
    const T up_im = __shfl_sync(0xffffffffu, r.im[3], up_src);
    const T dn_re = __shfl_sync(0xffffffffu, r.re[0], dn_src);
    const T dn_im = __shfl_sync(0xffffffffu, r.im[0], dn_src);
    rot(r.re[1], r.im[1], r.re[2], r.im[2], t);
    const T r0 = r.re[0], i0 = r.im[0], r3 = r.re[3], i3 = r.im[3];
    r.re[0] = fma(-t, up_im, r0);
    r.im[0] = fma(t, up_re, i0);
    r.re[3] = fma(-t, dn_im, r3);
    r.im[3] = fma(t, dn_re, i3);
}

// threads per block the register budget allows: fp32 rows cost 8 registers each, fp64 16
template <typename T, int R>
constexpr int tiny_max_threads() { return R >= 8 ? 256 : (sizeof(T) == 4 ? 1024 : 512); }

template <typename T, int R, bool POT, bool PER>
__global__ void __launch_bounds__(tiny_max_threads<T, R>(), 1) tiny_kernel(const TinyParams<T> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // per warp: its top row and its bottom row, [warp][top|bottom][re|im][lane][4]
    T* xch = reinterpret_cast<T*>(smem_raw);
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int nw = blockDim.x >> 5;
    const int nl = p.nx >> 2;                   // active lanes
    const bool active = lane < nl;
    const int xb = 4 * lane;
    const int y0 = warp * R;

    // per-lane coefficients: ghost lanes (beyond the row) hold zeros and must stay zero
    const T t_h = active ? p.t_h : T(0);
    XCut cut;
    cut.up = !PER && (xb == 0 || !active);
    cut.dn = !PER && (xb + 4 == p.nx || !active);
    const int up_src = lane == 0 ? nl - 1 : lane - 1;
    const int dn_src = lane == nl - 1 ? 0 : lane + 1;

    Row4<T> row[R];
    Row4<T> pot[POT ? R : 1];
#pragma unroll
    for (int i = 0; i < R; ++i) {
        if (active) {
            const int64_t off = (int64_t)(y0 + i) * p.nx + xb;
            ld4(p.re + off, row[i].re);
            ld4(p.im + off, row[i].im);
            if (POT) { ld4(p.pot_re + off, pot[i].re); ld4(p.pot_im + off, pot[i].im); }
        } else {
            zero_row(row[i]);
            if (POT) {
#pragma unroll
                for (int k = 0; k < 4; ++k) { pot[i].re[k] = T(1); pot[i].im[k] = T(0); }
            }
        }
    }

    auto x_even = [&](T t) {
#pragma unroll
        for (int i = 0; i < R; ++i) xe(row[i], t);
    };
    auto x_odd = [&]() {
#pragma unroll
        for (int i = 0; i < R; ++i) {
            if (PER) xo_ring(row[i], t_h, up_src, dn_src);
            else xo<T, true>(row[i], p.t_h, p.sec_h, cut);
        }
    };
    auto y_even = [&](T t) {
#pragma unroll
        for (int i = 0; i < R; i += 2) ypair(row[i], row[i + 1], t);
    };
    // vertical-odd sweep: interior pairs in registers, the two pairs that leave the warp through
    // shared memory (old values of both partners: written before any of them is touched)
    auto y_odd = [&](T t, T sec) {
        T* mine = xch + (size_t)warp * 2 * 2 * 128;
        auto put = [&](T* dst, const Row4<T>& r) {
            put4(dst + 4 * lane, r.re);
            put4(dst + 128 + 4 * lane, r.im);
        };
        auto get = [&](const T* src, Row4<T>& r) {
            get4(src + 4 * lane, r.re);
            get4(src + 128 + 4 * lane, r.im);
        };
        put(mine, row[0]);
        put(mine + 256, row[R - 1]);
        __syncthreads();
#pragma unroll
        for (int i = 1; i + 1 < R; i += 2) ypair(row[i], row[i + 1], t);
        const int wu = warp == 0 ? nw - 1 : warp - 1;
        const int wd = warp == nw - 1 ? 0 : warp + 1;
        Row4<T> other;
        if (PER || warp > 0) {
            get(xch + (size_t)wu * 512 + 256, other);        // bottom row of the warp above
            half_pair(row[0], other, t);
        } else {
            scale_row(row[0], sec);                          // row 0 of a closed lattice: unpaired
        }
        if (PER || warp < nw - 1) {
            get(xch + (size_t)wd * 512, other);              // top row of the warp below
            half_pair(row[R - 1], other, t);
        } else {
            scale_row(row[R - 1], sec);
        }
        __syncthreads();                                     // everybody has read: buffers free
    };

    for (int64_t s = 0; s < p.n_steps; ++s) {
        x_even(p.t_h);
        x_odd();
        y_even(p.t_h);
        if (!POT) {
            y_odd(p.t_f, p.sec_f);
        } else {
            y_odd(p.t_h, p.sec_h);
#pragma unroll
            for (int i = 0; i < R; ++i) phase_row(row[i], pot[i].re, pot[i].im);
            y_odd(p.t_h, p.sec_h);
        }
        y_even(p.t_h);
        x_odd();
        x_even(p.t_h);
        if ((s & 3) == 3) {     // every fourth step: keeps the scaled amplitudes in range
#pragma unroll
            for (int i = 0; i < R; ++i) scale_row(row[i], p.scale4);
        }
    }

    if (active) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int64_t off = (int64_t)(y0 + i) * p.nx + xb;
            st4(p.re + off, row[i].re, p.final_scale);
            st4(p.im + off, row[i].im, p.final_scale);
        }
    }
}

template <typename K, typename T>
int launch_one(K kern, const TinyParams<T>& p, int nw, cudaStream_t st) {
    const size_t smem = (size_t)nw * 512 * sizeof(T);
    TS_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<1, nw * 32, smem, st>>>(p);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}

template <typename T, int R>
int launch_r(const TinyParams<T>& p, bool pot, bool per, int nw, cudaStream_t st) {
    if (pot)
        return per ? launch_one(tiny_kernel<T, R, true, true>, p, nw, st)
                   : launch_one(tiny_kernel<T, R, true, false>, p, nw, st);
    return per ? launch_one(tiny_kernel<T, R, false, true>, p, nw, st)
               : launch_one(tiny_kernel<T, R, false, false>, p, nw, st);
}

template <typename T>
int evolve_t(const LatticeDesc& L, T* re, T* im, const StepCoef& c, const T* pot, int64_t n_steps,
             int prefer, cudaStream_t st) {
    const int R = tiny_rows_per_warp(L, pot != nullptr, prefer);
    TinyParams<T> p;
    p.re = re; p.im = im;
    p.pot_re = pot; p.pot_im = pot ? pot + L.nx * L.ny : nullptr;
    p.nx = (int)L.nx; p.ny = (int)L.ny; p.n_steps = n_steps;
    p.t_h = (T)(c.b_h / c.a_h); p.t_f = (T)(c.b_f / c.a_f);
    p.sec_h = (T)(1.0 / c.a_h); p.sec_f = (T)(1.0 / c.a_f);
    const double step = pot ? pow(c.a_h, 8) : pow(c.a_h, 6) * c.a_f;
    p.scale4 = (T)pow(step, 4);
    // the rounded factor is applied n_steps / 4 times: its relative error would add up linearly
    // (2e-4 in the fp32 norm after 1000 steps when applied per step); the store takes it out
    // again, together with the cosines of the last n_steps % 4 steps
    const int64_t groups = n_steps / 4;
    p.final_scale = (T)(pow(step, (double)(n_steps % 4)) *
                        exp((double)groups * log(pow(step, 4) / (double)p.scale4)));
    const int nw = (int)(L.ny / R);
    const bool per = L.periodic_x != 0;
    if (R == 2) return launch_r<T, 2>(p, pot != nullptr, per, nw, st);
    if (R == 4 && !pot)      // (with the phase rows in registers four rows per warp would spill)
        return per ? launch_one(tiny_kernel<T, 4, false, true>, p, nw, st)
                   : launch_one(tiny_kernel<T, 4, false, false>, p, nw, st);
    if (R == 8 && !pot)
        return per ? launch_one(tiny_kernel<T, 8, false, true>, p, nw, st)
                   : launch_one(tiny_kernel<T, 8, false, false>, p, nw, st);
    set_error("tiny_evolve: lattice does not fit one block");
    return TS_EUNSUPPORTED;
}

}  // namespace

int tiny_rows_per_warp(const LatticeDesc& L, bool pot, int prefer) {
    // rows per warp R: 2 (up to 32 warps in fp32, 16 in fp64: register budget at 1024 / 512
    // threads), and without a potential 4, or 8 with at most 8 warps.  More rows per warp mean
    // fewer vertical-odd pairs through shared memory: C1 runs 3.6 / 4.5 / 4.8e9 site-steps/s at
    // R = 2 / 4 / 8, so the largest R that fits is taken unless `prefer` (2, 4, 8) says otherwise.
    // Capacity: 128 x 128 sites in fp32, 128 x 64 in fp64; half of that with a potential.
    // 0 = the lattice does not fit one block.
    if (L.nx > kStripSites || L.nx % 4 || L.ny % 2 || L.periodic_x != L.periodic_y) return 0;
    const int max_warps = L.dtype == TS_F32 ? 32 : 16;
    const bool ok8 = !pot && L.ny % 8 == 0 && L.ny / 8 <= 8;
    const bool ok4 = !pot && L.ny % 4 == 0 && L.ny / 4 <= max_warps;
    const bool ok2 = L.ny / 2 <= max_warps;
    if (prefer == 2 && ok2) return 2;
    if (prefer == 4 && ok4) return 4;
    if (ok8) return 8;
    if (ok4) return 4;
    if (ok2) return 2;
    return 0;
}

bool tiny_supported(const LatticeDesc& L, const StepCoef& c, bool pot) {
    return tiny_rows_per_warp(L, pot, 0) != 0 && c.a_h > 0.25 && c.a_f > 0.25;
}

int tiny_evolve(const LatticeDesc& L, void* re, void* im, const StepCoef& c, const void* pot,
                int64_t n_steps, int rows_per_warp, cudaStream_t st) {
    if (L.dtype == TS_F32)
        return evolve_t<float>(L, (float*)re, (float*)im, c, (const float*)pot, n_steps,
                               rows_per_warp, st);
    return evolve_t<double>(L, (double*)re, (double*)im, c, (const double*)pot, n_steps,
                            rows_per_warp, st);
}

}  // namespace ts
