// su3.cuh -- complex scalars, 3x3 colour algebra, half-spinor spin algebra (device only).
//
// Everything lives in registers: fixed-size arrays, fully unrolled loops.  T is double or float.
// Spin conventions: chiral basis, gamma_mu = [[0, sigma_mu],[sigma_mu^dag, 0]],
//   sigma_x = [[0,-i],[-i,0]], sigma_y = [[0,-1],[1,0]], sigma_z = [[-i,0],[0,i]], sigma_t = 1,
// so (1 +- gamma_mu) psi = (h, +- sigma_mu^dag h) with the half spinor h = psi_upper +- sigma_mu psi_lower.
#pragma once
#include <cuda_runtime.h>

namespace lgt {

template <class T> struct Vec2;
template <> struct Vec2<double> { typedef double2 type; };
template <> struct Vec2<float> { typedef float2 type; };

template <class T> struct cx {
    T re, im;
};

template <class T> __device__ __forceinline__ cx<T> mk(T re, T im) {
    cx<T> r;
    r.re = re;
    r.im = im;
    return r;
}
template <class T> __device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <class T> __device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <class T> __device__ __forceinline__ cx<T> operator*(cx<T> a, cx<T> b) {
    return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <class T> __device__ __forceinline__ cx<T> operator*(T s, cx<T> a) { return mk<T>(s * a.re, s * a.im); }
template <class T> __device__ __forceinline__ cx<T> conj(cx<T> a) { return mk<T>(a.re, -a.im); }
template <class T> __device__ __forceinline__ cx<T> times_i(cx<T> a) { return mk<T>(-a.im, a.re); }
template <class T> __device__ __forceinline__ cx<T> times_mi(cx<T> a) { return mk<T>(a.im, -a.re); }
template <class T> __device__ __forceinline__ T norm2(cx<T> a) { return a.re * a.re + a.im * a.im; }
// acc += a * b
template <class T> __device__ __forceinline__ void cfma(cx<T>& acc, cx<T> a, cx<T> b) {
    acc.re = fma(a.re, b.re, acc.re);
    acc.re = fma(-a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im);
    acc.im = fma(a.im, b.re, acc.im);
}
// acc += conj(a) * b
template <class T> __device__ __forceinline__ void cfma_cj(cx<T>& acc, cx<T> a, cx<T> b) {
    acc.re = fma(a.re, b.re, acc.re);
    acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im);
    acc.im = fma(-a.im, b.re, acc.im);
}
// acc += a * conj(b)
template <class T> __device__ __forceinline__ void cfma_jc(cx<T>& acc, cx<T> a, cx<T> b) {
    acc.re = fma(a.re, b.re, acc.re);
    acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(a.im, b.re, acc.im);
    acc.im = fma(-a.re, b.im, acc.im);
}

// vectorised global access of one complex number (128-bit in fp64, 64-bit in fp32)
template <class T> __device__ __forceinline__ cx<T> ldc(const typename Vec2<T>::type* p) {
    typename Vec2<T>::type v = __ldg(p);
    return mk<T>(v.x, v.y);
}
// the same without allocating the line in L1 (data no other thread of the block will ask for)
__device__ __forceinline__ cx<double> ldc_na(const double2* p) {
    cx<double> r;
    asm("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(r.re), "=d"(r.im) : "l"(p));
    return r;
}
__device__ __forceinline__ cx<float> ldc_na(const float2* p) {
    cx<float> r;
    asm("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(r.re), "=f"(r.im) : "l"(p));
    return r;
}
template <class T> __device__ __forceinline__ cx<T> ldc_rw(const typename Vec2<T>::type* p) {
    typename Vec2<T>::type v = *p;
    return mk<T>(v.x, v.y);
}
template <class T> __device__ __forceinline__ void stc(typename Vec2<T>::type* p, cx<T> a) {
    typename Vec2<T>::type v;
    v.x = a.re;
    v.y = a.im;
    *p = v;
}

// ---------------------------------------------------------------------------- 3x3 colour matrices, row-major m[3*i+j]
template <class T> __device__ __forceinline__ void mat_zero(cx<T> r[9]) {
#pragma unroll
    for (int k = 0; k < 9; k++) r[k] = mk<T>(0, 0);
}
// r = a b
template <class T> __device__ __forceinline__ void mul_nn(const cx<T> a[9], const cx<T> b[9], cx<T> r[9]) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cx<T> acc = a[3 * i] * b[j];
            cfma(acc, a[3 * i + 1], b[3 + j]);
            cfma(acc, a[3 * i + 2], b[6 + j]);
            r[3 * i + j] = acc;
        }
}
// r = a b^dag
template <class T> __device__ __forceinline__ void mul_nd(const cx<T> a[9], const cx<T> b[9], cx<T> r[9]) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cx<T> acc = mk<T>(0, 0);
#pragma unroll
            for (int k = 0; k < 3; k++) cfma_jc(acc, a[3 * i + k], b[3 * j + k]);
            r[3 * i + j] = acc;
        }
}
// r = a^dag b
template <class T> __device__ __forceinline__ void mul_dn(const cx<T> a[9], const cx<T> b[9], cx<T> r[9]) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cx<T> acc = mk<T>(0, 0);
#pragma unroll
            for (int k = 0; k < 3; k++) cfma_cj(acc, a[3 * k + i], b[3 * k + j]);
            r[3 * i + j] = acc;
        }
}

// Compact storage of a traceless anti-Hermitian matrix A (momenta and forces): 8 reals,
//   c[0] = Im A00, c[1] = Im A11, (c[2],c[3]) = A01, (c[4],c[5]) = A02, (c[6],c[7]) = A12;
//   Im A22 = -(c[0]+c[1]), A10 = -conj(A01), A20 = -conj(A02), A21 = -conj(A12).
// ta_compact: c = scale * P_su(3)[M],  P[M] = (M - M^dag)/2 - tr(M - M^dag)/6   (Eq. 7)
template <class T> __device__ __forceinline__ void ta_compact(const cx<T> m[9], T scale, T c[8]) {
    T tr3 = (m[0].im + m[4].im + m[8].im) * (T)(1.0 / 3.0);
    c[0] = scale * (m[0].im - tr3);
    c[1] = scale * (m[4].im - tr3);
    T h = (T)0.5 * scale;
    c[2] = h * (m[1].re - m[3].re);
    c[3] = h * (m[1].im + m[3].im);
    c[4] = h * (m[2].re - m[6].re);
    c[5] = h * (m[2].im + m[6].im);
    c[6] = h * (m[5].re - m[7].re);
    c[7] = h * (m[5].im + m[7].im);
}
template <class T> __device__ __forceinline__ void compact_expand(const T c[8], cx<T> m[9]) {
    m[0] = mk<T>(0, c[0]);
    m[4] = mk<T>(0, c[1]);
    m[8] = mk<T>(0, -(c[0] + c[1]));
    m[1] = mk<T>(c[2], c[3]);
    m[3] = mk<T>(-c[2], c[3]);
    m[2] = mk<T>(c[4], c[5]);
    m[6] = mk<T>(-c[4], c[5]);
    m[5] = mk<T>(c[6], c[7]);
    m[7] = mk<T>(-c[6], c[7]);
}

// ---------------------------------------------------------------------------- spin algebra
// Half-spinor projection h[t][c] = psi[t][c] + SG (sigma_MU psi_lower)[t][c], t = 0,1; psi[4][3] as p[3*alpha+c].
template <int MU, int SG, class T> __device__ __forceinline__ void spin_project(const cx<T> p[12], cx<T> h[6]) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        cx<T> s0, s1;  // (sigma psi_lower)_{0,1}
        if (MU == 0) {
            s0 = times_mi(p[9 + c]);
            s1 = times_mi(p[6 + c]);
        } else if (MU == 1) {
            s0 = mk<T>(-p[9 + c].re, -p[9 + c].im);
            s1 = p[6 + c];
        } else if (MU == 2) {
            s0 = times_mi(p[6 + c]);
            s1 = times_i(p[9 + c]);
        } else {
            s0 = p[6 + c];
            s1 = p[9 + c];
        }
        h[c] = (SG > 0) ? p[c] + s0 : p[c] - s0;
        h[3 + c] = (SG > 0) ? p[3 + c] + s1 : p[3 + c] - s1;
    }
}
// acc += (w, SG sigma_MU^dag w): the reconstruction of (1 + SG gamma_MU) from the half spinor w[2][3].
template <int MU, int SG, class T> __device__ __forceinline__ void spin_reconstruct_add(const cx<T> w[6], cx<T> acc[12]) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        acc[c] = acc[c] + w[c];
        acc[3 + c] = acc[3 + c] + w[3 + c];
        cx<T> l0, l1;  // (sigma^dag w)_{0,1}
        if (MU == 0) {
            l0 = times_i(w[3 + c]);
            l1 = times_i(w[c]);
        } else if (MU == 1) {
            l0 = w[3 + c];
            l1 = mk<T>(-w[c].re, -w[c].im);
        } else if (MU == 2) {
            l0 = times_i(w[c]);
            l1 = times_mi(w[3 + c]);
        } else {
            l0 = w[c];
            l1 = w[3 + c];
        }
        acc[6 + c] = (SG > 0) ? acc[6 + c] + l0 : acc[6 + c] - l0;
        acc[9 + c] = (SG > 0) ? acc[9 + c] + l1 : acc[9 + c] - l1;
    }
}
// w[t] = u h[t]  /  w[t] = u^dag h[t]   (colour multiplication of both spin components)
template <class T> __device__ __forceinline__ void su3_mul_half(const cx<T> u[9], const cx<T> h[6], cx<T> w[6]) {
#pragma unroll
    for (int t = 0; t < 2; t++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            cx<T> acc = u[3 * a] * h[3 * t];
            cfma(acc, u[3 * a + 1], h[3 * t + 1]);
            cfma(acc, u[3 * a + 2], h[3 * t + 2]);
            w[3 * t + a] = acc;
        }
}
template <class T> __device__ __forceinline__ void su3_dag_mul_half(const cx<T> u[9], const cx<T> h[6], cx<T> w[6]) {
#pragma unroll
    for (int t = 0; t < 2; t++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            cx<T> acc = mk<T>(0, 0);
#pragma unroll
            for (int b = 0; b < 3; b++) cfma_cj(acc, u[3 * b + a], h[3 * t + b]);
            w[3 * t + a] = acc;
        }
}

}  // namespace lgt
