// ts_generic.cu -- generic per-sweep CUDA path: one launch per checkerboard sweep, in place.
//
// Works for every lattice shape and both boundaries; it is the in-library path for shapes the
// fused kernel does not take (nx % 4 != 0, odd ny, large angles) and the simple statement of
// SURVEY.md 8(a) rows a1-a7, a9 on the device.  It moves 16 B/site (fp32) per sweep, i.e. 7-9x
// the traffic of the fused kernel, so it is never the fast path.
//
// Pair rotation: (psi_p, psi_q) <- [[a, i b],[i b, a]] (psi_p, psi_q), both
// outputs from the old values.  fp32 uses the eps-form a*x = x - eps*x with eps = 1 - a computed
// in double: same two FMAs, but a^2 + b^2 = 1 is kept to ~1e-12 instead of
// the ~6e-8 that rounding cos(theta) to fp32 would give.
#include <math.h>

#include "ts_internal.h"

namespace ts {
namespace {

template <typename T>
struct RotCoef {
    T a;    // cos
    T b;    // sin (signed)
    T eps;  // 1 - a, rounded from double
};

template <typename T>
__device__ __forceinline__ T mul_a(T x, const RotCoef<T>& c);
template <>
__device__ __forceinline__ float mul_a<float>(float x, const RotCoef<float>& c) {
    return fmaf(-c.eps, x, x);
}
template <>
__device__ __forceinline__ double mul_a<double>(double x, const RotCoef<double>& c) {
    return c.a * x;
}

template <typename T>
__device__ __forceinline__ void rotate(T* __restrict__ re, T* __restrict__ im, int64_t p,
                                       int64_t q, const RotCoef<T>& c) {
    const T rp = re[p], ip = im[p], rq = re[q], iq = im[q];
    re[p] = fma(-c.b, iq, mul_a(rp, c));
    im[p] = fma(c.b, rq, mul_a(ip, c));
    re[q] = fma(-c.b, ip, mul_a(rq, c));
    im[q] = fma(c.b, rp, mul_a(iq, c));
}

// Horizontal sweep: pair i of row y couples x = parity + 2i and x + 1 (or the wrap pair).
template <typename T>
__global__ void __launch_bounds__(256)
sweep_x_kernel(T* __restrict__ re, T* __restrict__ im, int64_t nx, int64_t ny, int parity,
               int64_t pairs_per_row, int wrap, RotCoef<T> c) {
    const int64_t total = pairs_per_row * ny;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total;
         t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t y = t / pairs_per_row;
        const int64_t i = t - y * pairs_per_row;
        const int64_t x = parity + 2 * i;
        const int64_t p = y * nx + x;
        const int64_t q = (wrap && x == nx - 1) ? y * nx : p + 1;
        rotate(re, im, p, q, c);
    }
}

// Vertical sweep: pair k of column x couples y = parity + 2k and y + 1 (or the wrap pair).
template <typename T>
__global__ void __launch_bounds__(256)
sweep_y_kernel(T* __restrict__ re, T* __restrict__ im, int64_t nx, int64_t ny, int parity,
               int64_t pairs_per_col, int wrap, RotCoef<T> c) {
    const int64_t total = pairs_per_col * nx;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total;
         t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t k = t / nx;
        const int64_t x = t - k * nx;
        const int64_t y = parity + 2 * k;
        const int64_t p = y * nx + x;
        const int64_t q = (wrap && y == ny - 1) ? x : p + nx;
        rotate(re, im, p, q, c);
    }
}

// psi <- psi * (pr + i pi)   (e^{-i dt H0})
template <typename T>
__global__ void __launch_bounds__(256)
phase_kernel(T* __restrict__ re, T* __restrict__ im, const T* __restrict__ pr,
             const T* __restrict__ pi, int64_t n) {
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n;
         t += (int64_t)gridDim.x * blockDim.x) {
        const T r = re[t], m = im[t], cr = pr[t], ci = pi[t];
        re[t] = fma(-m, ci, r * cr);
        im[t] = fma(m, cr, r * ci);
    }
}

constexpr int kNormBlocks = 1184;   // 8 per SM on 148 SMs
constexpr int kNormThreads = 256;

template <typename T>
__global__ void __launch_bounds__(kNormThreads)
norm_partial_kernel(const T* __restrict__ re, const T* __restrict__ im, int64_t n,
                    double* __restrict__ partial) {
    double acc = 0.0;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n;
         t += (int64_t)gridDim.x * blockDim.x) {
        const double r = (double)re[t], m = (double)im[t];
        acc = fma(r, r, fma(m, m, acc));
    }
    __shared__ double sh[kNormThreads / 32];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < kNormThreads / 32 ? sh[threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) partial[blockIdx.x] = v;
    }
}

__global__ void __launch_bounds__(1024)
norm_final_kernel(const double* __restrict__ partial, int n, double* __restrict__ out) {
    __shared__ double sh[32];
    double acc = 0.0;
    for (int t = threadIdx.x; t < n; t += blockDim.x) acc += partial[t];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = sh[threadIdx.x];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) *out = v;
    }
}

inline int grid_for(int64_t total, int threads) {
    int64_t g = (total + threads - 1) / threads;
    const int64_t cap = 148 * 32;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

template <typename T>
RotCoef<T> make_rot(double a, double b) {
    RotCoef<T> c;
    c.a = (T)a;
    c.b = (T)b;
    // 1 - a without cancellation: b^2 / (1 + a) when a > 0 (a^2 + b^2 = 1)
    const double eps = a > 0.0 ? (b * b) / (1.0 + a) : 1.0 - a;
    c.eps = (T)eps;
    return c;
}

template <typename T>
int sweep(const LatticeDesc& L, T* re, T* im, int axis, int parity, double a, double b,
          cudaStream_t st, int64_t* launches) {
    const int64_t n = axis == 0 ? L.nx : L.ny;
    const int wrap = ((axis == 0 ? L.periodic_x : L.periodic_y) && parity == 1) ? 1 : 0;
    int64_t pairs = parity == 0 ? n / 2 : (n - 1) / 2;
    if (wrap) pairs += 1;   // n even when periodic: (n-1)/2 inner pairs + the wrap pair = n/2
    if (pairs <= 0) return TS_OK;
    const RotCoef<T> c = make_rot<T>(a, b);
    if (axis == 0) {
        const int64_t total = pairs * L.ny;
        sweep_x_kernel<T><<<grid_for(total, 256), 256, 0, st>>>(re, im, L.nx, L.ny, parity, pairs,
                                                                 wrap, c);
    } else {
        const int64_t total = pairs * L.nx;
        sweep_y_kernel<T><<<grid_for(total, 256), 256, 0, st>>>(re, im, L.nx, L.ny, parity, pairs,
                                                                 wrap, c);
    }
    ++*launches;
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}

template <typename T>
int evolve_t(const LatticeDesc& L, T* re, T* im, const StepCoef& c, const T* pot,
             int64_t n_steps, cudaStream_t st, int64_t* launches) {
    const int64_t n = L.nx * L.ny;
#define TS_SWEEP(axis, parity, a, b)                                               \
    do {                                                                           \
        int rc_ = sweep<T>(L, re, im, axis, parity, a, b, st, launches);           \
        if (rc_ != TS_OK) return rc_;                                              \
    } while (0)
    for (int64_t s = 0; s < n_steps; ++s) {
        TS_SWEEP(0, 0, c.a_h, c.b_h);
        TS_SWEEP(0, 1, c.a_h, c.b_h);
        TS_SWEEP(1, 0, c.a_h, c.b_h);
        if (pot == nullptr) {
            TS_SWEEP(1, 1, c.a_f, c.b_f);
        } else {
            TS_SWEEP(1, 1, c.a_h, c.b_h);
            phase_kernel<T><<<grid_for(n, 256), 256, 0, st>>>(re, im, pot, pot + n, n);
            ++*launches;
            TS_CUDA_TRY(cudaGetLastError());
            TS_SWEEP(1, 1, c.a_h, c.b_h);
        }
        TS_SWEEP(1, 0, c.a_h, c.b_h);
        TS_SWEEP(0, 1, c.a_h, c.b_h);
        TS_SWEEP(0, 0, c.a_h, c.b_h);
    }
#undef TS_SWEEP
    return TS_OK;
}

}  // namespace

int generic_evolve(const LatticeDesc& L, void* re, void* im, const StepCoef& c, const void* pot,
                   int64_t n_steps, cudaStream_t st, int64_t* launches) {
    if (L.dtype == TS_F32)
        return evolve_t<float>(L, (float*)re, (float*)im, c, (const float*)pot, n_steps, st,
                               launches);
    return evolve_t<double>(L, (double*)re, (double*)im, c, (const double*)pot, n_steps, st,
                            launches);
}

namespace {
template <typename T>
__global__ void expand_separable_kernel(const T* __restrict__ px, const T* __restrict__ py,
                                        T* __restrict__ pot, int64_t nx, int64_t ny) {
    const int64_t n = nx * ny;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t x = i % nx, y = i / nx;
        const T xr = px[x], xi = px[nx + x], yr = py[y], yi = py[ny + y];
        pot[i] = xr * yr - xi * yi;
        pot[n + i] = xr * yi + xi * yr;
    }
}
}  // namespace

int expand_separable(const LatticeDesc& L, const void* px, const void* py, void* pot,
                     cudaStream_t st) {
    const int64_t n = L.nx * L.ny;
    if (L.dtype == TS_F32)
        expand_separable_kernel<float><<<grid_for(n, 256), 256, 0, st>>>(
            (const float*)px, (const float*)py, (float*)pot, L.nx, L.ny);
    else
        expand_separable_kernel<double><<<grid_for(n, 256), 256, 0, st>>>(
            (const double*)px, (const double*)py, (double*)pot, L.nx, L.ny);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}


// ---- three-dimensional lattices: one launch per sweep ----------------------------------------------
// psi[nz][ny][nx]; a sweep along an axis of extent n whose sites are `m` elements apart (x: 1,
// y: nx, z: nx*ny) on `outer` repetitions (x: ny*nz, y: nz, z: 1): element (o, i, r) at
// (o*n + i)*m + r.  Pair k of a line couples i = parity + 2k and i + 1 (or the wrap pair).
namespace {
template <typename T>
__global__ void __launch_bounds__(256)
sweep3_kernel(T* __restrict__ re, T* __restrict__ im, int64_t m, int64_t n, int64_t outer,
              int parity, int64_t pairs, int wrap, RotCoef<T> c) {
    const int64_t total = pairs * m * outer;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total;
         t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = t % m;
        const int64_t q1 = t / m;
        const int64_t k = q1 % pairs;
        const int64_t o = q1 / pairs;
        const int64_t i = parity + 2 * k;
        const int64_t p = (o * n + i) * m + r;
        const int64_t q = (wrap && i == n - 1) ? (o * n) * m + r : p + m;
        rotate(re, im, p, q, c);
    }
}

template <typename T>
int sweep3(const Lattice3& L, T* re, T* im, int axis, int parity, double a, double b,
           cudaStream_t st, int64_t* launches) {
    const int64_t n = axis == 0 ? L.nx : (axis == 1 ? L.ny : L.nz);
    const int64_t m = axis == 0 ? 1 : (axis == 1 ? L.nx : L.nx * L.ny);
    const int64_t outer = axis == 0 ? L.ny * L.nz : (axis == 1 ? L.nz : 1);
    const int wrap = (L.per[axis] && parity == 1) ? 1 : 0;
    int64_t pairs = parity == 0 ? n / 2 : (n - 1) / 2;
    if (wrap) pairs += 1;
    if (pairs <= 0) return TS_OK;
    const RotCoef<T> c = make_rot<T>(a, b);
    const int64_t total = pairs * m * outer;
    sweep3_kernel<T><<<grid_for(total, 256), 256, 0, st>>>(re, im, m, n, outer, parity, pairs, wrap, c);
    ++*launches;
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}

// the literal stage list of the 3-D step (include/ts.h, ts_evolve_3d)
template <typename T>
int evolve3_t(const Lattice3& L, T* re, T* im, const StepCoef& c, const T* pot, int64_t n_steps,
              cudaStream_t st, int64_t* launches) {
    const int64_t sites = L.nx * L.ny * L.nz;
    int rc;
#define TS_SWEEP3(axis, parity, a, b)                                                        \
    if ((rc = sweep3<T>(L, re, im, axis, parity, a, b, st, launches)) != TS_OK) return rc
    for (int64_t s = 0; s < n_steps; ++s) {
        TS_SWEEP3(0, 0, c.a_h, c.b_h);
        TS_SWEEP3(0, 1, c.a_h, c.b_h);
        TS_SWEEP3(1, 0, c.a_h, c.b_h);
        TS_SWEEP3(1, 1, c.a_h, c.b_h);
        TS_SWEEP3(2, 0, c.a_h, c.b_h);
        if (pot == nullptr) {
            TS_SWEEP3(2, 1, c.a_f, c.b_f);
        } else {
            TS_SWEEP3(2, 1, c.a_h, c.b_h);
            phase_kernel<T><<<grid_for(sites, 256), 256, 0, st>>>(re, im, pot, pot + sites, sites);
            ++*launches;
            TS_CUDA_TRY(cudaGetLastError());
            TS_SWEEP3(2, 1, c.a_h, c.b_h);
        }
        TS_SWEEP3(2, 0, c.a_h, c.b_h);
        TS_SWEEP3(1, 1, c.a_h, c.b_h);
        TS_SWEEP3(1, 0, c.a_h, c.b_h);
        TS_SWEEP3(0, 1, c.a_h, c.b_h);
        TS_SWEEP3(0, 0, c.a_h, c.b_h);
    }
#undef TS_SWEEP3
    return TS_OK;
}
}  // namespace

int generic3_evolve(const Lattice3& L, void* re, void* im, const StepCoef& c, const void* pot,
                    int64_t n_steps, cudaStream_t st, int64_t* launches) {
    if (L.dtype == TS_F32)
        return evolve3_t<float>(L, (float*)re, (float*)im, c, (const float*)pot, n_steps, st, launches);
    return evolve3_t<double>(L, (double*)re, (double*)im, c, (const double*)pot, n_steps, st, launches);
}

size_t norm_workspace_doubles() { return kNormBlocks + 1; }

int norm2_device(const LatticeDesc& L, const void* re, const void* im, double* d_work,
                 cudaStream_t st) {
    const int64_t n = L.nx * L.ny;
    int blocks = grid_for(n, kNormThreads);
    if (blocks > kNormBlocks) blocks = kNormBlocks;
    if (L.dtype == TS_F32)
        norm_partial_kernel<float><<<blocks, kNormThreads, 0, st>>>((const float*)re,
                                                                    (const float*)im, n, d_work + 1);
    else
        norm_partial_kernel<double><<<blocks, kNormThreads, 0, st>>>(
            (const double*)re, (const double*)im, n, d_work + 1);
    TS_CUDA_TRY(cudaGetLastError());
    norm_final_kernel<<<1, 1024, 0, st>>>(d_work + 1, blocks, d_work);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}

}  // namespace ts
