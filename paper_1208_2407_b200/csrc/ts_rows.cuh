// ts_rows.cuh -- per-lane row arithmetic shared by the fused kernels (device code only).
//
// A lane owns 4 consecutive sites of a row (re[4], im[4]).  Every pair rotation
// [[a, i b],[i b, a]] is applied in the scaled form a * [[1, i t],[i t, 1]],
// t = b/a: two FMAs per site per sweep; the factors a are collected into one multiplication
// at the store.  At a closed edge the unpaired site is multiplied by 1/a instead, so that the
// deferred factor stays uniform over the lattice.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ts {
namespace rows {

constexpr int kStripSites = 128;   // 32 lanes x 4 sites

template <typename T>
struct Row4 {
    T re[4];
    T im[4];
};

__device__ __forceinline__ void ld4(const float* __restrict__ p, float (&v)[4]) {
    const float4 q = __ldg(reinterpret_cast<const float4*>(p));
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
}
__device__ __forceinline__ void ld4(const double* __restrict__ p, double (&v)[4]) {
    const double2 a = __ldg(reinterpret_cast<const double2*>(p));
    const double2 b = __ldg(reinterpret_cast<const double2*>(p) + 1);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}
__device__ __forceinline__ void mul2v(float& dx, float& dy, float ax, float ay, float bx,
                                      float by);
__device__ __forceinline__ void st4(float* __restrict__ p, const float (&v)[4], float s) {
    float4 q;
    mul2v(q.x, q.y, v[0], v[1], s, s);
    mul2v(q.z, q.w, v[2], v[3], s, s);
    *reinterpret_cast<float4*>(p) = q;
}
__device__ __forceinline__ void st4(double* __restrict__ p, const double (&v)[4], double s) {
    reinterpret_cast<double2*>(p)[0] = make_double2(v[0] * s, v[1] * s);
    reinterpret_cast<double2*>(p)[1] = make_double2(v[2] * s, v[3] * s);
}

template <typename T>
__device__ __forceinline__ void zero_row(Row4<T>& r) {
#pragma unroll
    for (int i = 0; i < 4; ++i) { r.re[i] = T(0); r.im[i] = T(0); }
}

// scaled pair rotation: (p, q) <- (p + i t q, q + i t p), from the old values of both
template <typename T>
__device__ __forceinline__ void rot(T& rp, T& ip, T& rq, T& iq, T t) {
    const T nrp = fma(-t, iq, rp);
    const T nip = fma(t, rq, ip);
    const T nrq = fma(-t, ip, rq);
    const T niq = fma(t, rp, iq);
    rp = nrp; ip = nip; rq = nrq; iq = niq;
}

// Packed fp32 arithmetic (sm_100: fma.rn.f32x2 / mul.rn.f32x2, SASS FFMA2 / FMUL2): two FMAs per
// issue slot on an aligned register pair.  The kernel is issue-limited before it is FMA-pipe
// limited (round-1 captures), so the sweeps whose pairs line up with adjacent sites use it.  ptxas
// folds the scalar broadcast, the negation and a swapped source pair into operand modifiers.
// (dx, dy) = s * (bx, by) + (cx, cy)
__device__ __forceinline__ void fma2(float& dx, float& dy, float s, float bx, float by, float cx,
                                     float cy) {
    unsigned long long rs, rb, rc, rd;
    asm("mov.b64 %0, {%1, %1};" : "=l"(rs) : "f"(s));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(bx), "f"(by));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rc) : "f"(cx), "f"(cy));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(rs), "l"(rb), "l"(rc));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(dx), "=f"(dy) : "l"(rd));
}
// (dx, dy) = (ax, ay) * (bx, by) + (cx, cy)
__device__ __forceinline__ void fma2v(float& dx, float& dy, float ax, float ay, float bx, float by,
                                      float cx, float cy) {
    unsigned long long ra, rb, rc, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(ax), "f"(ay));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(bx), "f"(by));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rc) : "f"(cx), "f"(cy));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(dx), "=f"(dy) : "l"(rd));
}
// (dx, dy) = (ax, ay) * (bx, by)
__device__ __forceinline__ void mul2v(float& dx, float& dy, float ax, float ay, float bx,
                                      float by) {
    unsigned long long ra, rb, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(ax), "f"(ay));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(bx), "f"(by));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(dx), "=f"(dy) : "l"(rd));
}

// X-even sweep on one row: pairs (0,1), (2,3) of the lane's four sites
template <typename T>
__device__ __forceinline__ void xe(Row4<T>& r, T t) {
    rot(r.re[0], r.im[0], r.re[1], r.im[1], t);
    rot(r.re[2], r.im[2], r.re[3], r.im[3], t);
}
#ifndef TS_SCALAR_F32   // -DTS_SCALAR_F32: A/B build without the packed forms
// fp32: (re_k, re_k+1) -= t (im_k+1, im_k); (im_k, im_k+1) += t (re_k+1, re_k)   [old values]
__device__ __forceinline__ void xe(Row4<float>& r, float t) {
#pragma unroll
    for (int k = 0; k < 4; k += 2) {
        float nr0, nr1, ni0, ni1;
        fma2(nr0, nr1, -t, r.im[k + 1], r.im[k], r.re[k], r.re[k + 1]);
        fma2(ni0, ni1, t, r.re[k + 1], r.re[k], r.im[k], r.im[k + 1]);
        r.re[k] = nr0; r.re[k + 1] = nr1; r.im[k] = ni0; r.im[k + 1] = ni1;
    }
}
#endif

// per-lane coefficients of the cross-lane X-odd pair; differ from (t, t, 1, 1) only in strips
// that touch a closed domain edge
template <typename T>
struct XEdge {
    T t_up;   // coupling of my site 0 to the previous lane's site 3
    T t_dn;   // coupling of my site 3 to the next lane's site 0
    T c0;     // factor on my site 0 (1/a when it is the unpaired edge site)
    T c3;     // factor on my site 3
};

// X-odd sweep on one row: pair (1,2) in-thread, pair (3, 0 of next lane) by shuffle.
template <typename T, bool EDGE>
__device__ __forceinline__ void xo(Row4<T>& r, T t, const XEdge<T>& e) {
    const T up_re = __shfl_up_sync(0xffffffffu, r.re[3], 1);
    const T up_im = __shfl_up_sync(0xffffffffu, r.im[3], 1);
    const T dn_re = __shfl_down_sync(0xffffffffu, r.re[0], 1);
    const T dn_im = __shfl_down_sync(0xffffffffu, r.im[0], 1);
    rot(r.re[1], r.im[1], r.re[2], r.im[2], t);
    if (EDGE) {
        const T r0 = r.re[0] * e.c0, i0 = r.im[0] * e.c0;
        const T r3 = r.re[3] * e.c3, i3 = r.im[3] * e.c3;
        r.re[0] = fma(-e.t_up, up_im, r0);
        r.im[0] = fma(e.t_up, up_re, i0);
        r.re[3] = fma(-e.t_dn, dn_im, r3);
        r.im[3] = fma(e.t_dn, dn_re, i3);
    } else {
        const T r0 = r.re[0], i0 = r.im[0], r3 = r.re[3], i3 = r.im[3];
        r.re[0] = fma(-t, up_im, r0);
        r.im[0] = fma(t, up_re, i0);
        r.re[3] = fma(-t, dn_im, r3);
        r.im[3] = fma(t, dn_re, i3);
    }
}

// The same with the coupling given per call (the angle may change from sub-step to sub-step):
// the lane only remembers WHERE its cross-lane pairs are cut by a closed edge.
struct XCut {
    bool up;   // pair (site 0, previous lane's site 3) straddles a closed edge (or is all ghost)
    bool dn;   // pair (site 3, next lane's site 0) does
};
template <typename T, bool EDGE>
__device__ __forceinline__ void xo(Row4<T>& r, T t, T sec, const XCut& m) {
    if (EDGE) {
        XEdge<T> e;
        e.t_up = m.up ? T(0) : t;  e.c0 = m.up ? sec : T(1);
        e.t_dn = m.dn ? T(0) : t;  e.c3 = m.dn ? sec : T(1);
        xo<T, true>(r, t, e);
    } else {
        XEdge<T> e;   // unused by the plain form
        xo<T, false>(r, t, e);
    }
}

// vertical pair sweep between two rows held by the same lane
template <typename T>
__device__ __forceinline__ void ypair(Row4<T>& a, Row4<T>& b, T t) {
#pragma unroll
    for (int i = 0; i < 4; ++i) rot(a.re[i], a.im[i], b.re[i], b.im[i], t);
}

#ifndef TS_SCALAR_F32
__device__ __forceinline__ void ypair(Row4<float>& a, Row4<float>& b, float t) {
#pragma unroll
    for (int k = 0; k < 4; k += 2) {
        float ar0, ar1, ai0, ai1, br0, br1, bi0, bi1;
        fma2(ar0, ar1, -t, b.im[k], b.im[k + 1], a.re[k], a.re[k + 1]);
        fma2(ai0, ai1, t, b.re[k], b.re[k + 1], a.im[k], a.im[k + 1]);
        fma2(br0, br1, -t, a.im[k], a.im[k + 1], b.re[k], b.re[k + 1]);
        fma2(bi0, bi1, t, a.re[k], a.re[k + 1], b.im[k], b.im[k + 1]);
        a.re[k] = ar0; a.re[k + 1] = ar1; a.im[k] = ai0; a.im[k + 1] = ai1;
        b.re[k] = br0; b.re[k + 1] = br1; b.im[k] = bi0; b.im[k + 1] = bi1;
    }
}
#endif

template <typename T>
__device__ __forceinline__ void scale_row(Row4<T>& r, T s) {
#pragma unroll
    for (int i = 0; i < 4; ++i) { r.re[i] *= s; r.im[i] *= s; }
}
#ifndef TS_SCALAR_F32
__device__ __forceinline__ void scale_row(Row4<float>& r, float s) {
#pragma unroll
    for (int k = 0; k < 4; k += 2) {
        mul2v(r.re[k], r.re[k + 1], r.re[k], r.re[k + 1], s, s);
        mul2v(r.im[k], r.im[k + 1], r.im[k], r.im[k + 1], s, s);
    }
}
#endif

// psi <- psi * (pr + i pi) on one row
template <typename T>
__device__ __forceinline__ void phase_row(Row4<T>& r, const T (&pr)[4], const T (&pi)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const T a = r.re[i], b = r.im[i];
        r.re[i] = fma(-b, pi[i], a * pr[i]);
        r.im[i] = fma(b, pr[i], a * pi[i]);
    }
}

#ifndef TS_SCALAR_F32
__device__ __forceinline__ void phase_row(Row4<float>& r, const float (&pr)[4],
                                          const float (&pi)[4]) {
#pragma unroll
    for (int k = 0; k < 4; k += 2) {
        float m0, m1, n0, n1, nr0, nr1, ni0, ni1;
        mul2v(m0, m1, r.re[k], r.re[k + 1], pr[k], pr[k + 1]);
        mul2v(n0, n1, r.re[k], r.re[k + 1], pi[k], pi[k + 1]);
        fma2v(nr0, nr1, -r.im[k], -r.im[k + 1], pi[k], pi[k + 1], m0, m1);
        fma2v(ni0, ni1, r.im[k], r.im[k + 1], pr[k], pr[k + 1], n0, n1);
        r.re[k] = nr0; r.re[k + 1] = nr1; r.im[k] = ni0; r.im[k + 1] = ni1;
    }
}
#endif

// separable potential: psi <- psi * (px + i px') * (py + i py') on one row; px per site of the
// lane (registers), py one value for the row
template <typename T>
__device__ __forceinline__ void sep_phase_row(Row4<T>& r, const T (&pxr)[4], const T (&pxi)[4],
                                              T pyr, T pyi) {
    T wr[4], wi[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        wr[i] = fma(-pxi[i], pyi, pxr[i] * pyr);
        wi[i] = fma(pxi[i], pyr, pxr[i] * pyi);
    }
    phase_row(r, wr, wi);
}
#ifndef TS_SCALAR_F32
__device__ __forceinline__ void sep_phase_row(Row4<float>& r, const float (&pxr)[4],
                                              const float (&pxi)[4], float pyr, float pyi) {
    float wr[4], wi[4];
#pragma unroll
    for (int k = 0; k < 4; k += 2) {
        float m0, m1, n0, n1;
        mul2v(m0, m1, pxr[k], pxr[k + 1], pyr, pyr);
        mul2v(n0, n1, pxr[k], pxr[k + 1], pyi, pyi);
        fma2(wr[k], wr[k + 1], -pyi, pxi[k], pxi[k + 1], m0, m1);
        fma2(wi[k], wi[k + 1], pyr, pxi[k], pxi[k + 1], n0, n1);
    }
    phase_row(r, wr, wi);
}
#endif

__device__ __forceinline__ int wrap_index(int v, int n) {
    while (v < 0) v += n;
    while (v >= n) v -= n;
    return v;
}


}  // namespace rows
}  // namespace ts
