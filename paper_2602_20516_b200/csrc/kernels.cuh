// kernels.cuh -- the CUDA kernels of the hot path (sm_100a, CUDA-core FMAs, no tensor cores:
// 3x3 complex products are not a dense contraction).  Included once by lgt_api.cu.
//
// NATIVE LAYOUT (structure of arrays, site-major):
//   spinor   psi[12][Vs]  complex, component k = 3*alpha + a   -> address (k*Vs + s)
//   links    U[4][9][Vs]  complex, k = 9*mu + 3*i + j          -> address (k*Vs + s)
//   momenta  P[4][4][Vs]  pairs of reals (8-real compact su(3)) k = 4*mu + q -> address (k*Vs + s)
// so that a warp's 32 consecutive sites read 32 consecutive 16-byte words (fp64) per component.
// s is the canonical lexicographic site index; Vs = V (field stride).
#pragma once
#include "su3.cuh"

namespace lgt {

struct Geom {
    int L[4];
    int stride[4];  // site-index stride of direction mu
    int V;
    int Vs;
    int bc[4];
};

// CG recurrence scalars, resident on the device so that iterations need no host round trip.
struct CgState {
    double rr;     // |r|^2
    double bb;     // |b|^2
    double pAp;    // |D p|^2 = <p, D^dag D p>
    double alpha;  // rr / pAp
    double beta;   // rr_new / rr
    double tol2;   // tol^2
    int iter;
    int max_iter;
    int done;
    int pad;
};

struct Site {
    int x[4];
};
__device__ __forceinline__ Site site_coords(const Geom& g, int s) {
    Site c;
    c.x[0] = s % g.L[0];
    int r = s / g.L[0];
    c.x[1] = r % g.L[1];
    r /= g.L[1];
    c.x[2] = r % g.L[2];
    c.x[3] = r / g.L[2];
    return c;
}
__device__ __forceinline__ int nbr_fwd(const Geom& g, const Site& c, int s, int mu) {
    return (c.x[mu] == g.L[mu] - 1) ? s - (g.L[mu] - 1) * g.stride[mu] : s + g.stride[mu];
}
__device__ __forceinline__ int nbr_bwd(const Geom& g, const Site& c, int s, int mu) {
    return (c.x[mu] == 0) ? s + (g.L[mu] - 1) * g.stride[mu] : s - g.stride[mu];
}

template <class T> __device__ __forceinline__ void load_link(const typename Vec2<T>::type* U, const Geom& g, int mu, int s, cx<T> u[9]) {
#pragma unroll
    for (int k = 0; k < 9; k++) u[k] = ldc<T>(U + (size_t)(9 * mu + k) * g.Vs + s);
}
template <class T> __device__ __forceinline__ void load_spinor(const typename Vec2<T>::type* f, const Geom& g, int s, cx<T> p[12]) {
#pragma unroll
    for (int k = 0; k < 12; k++) p[k] = ldc<T>(f + (size_t)k * g.Vs + s);
}

// ---------------------------------------------------------------------------- deterministic reductions
// Block sum (fixed shuffle tree), block partial to partials[blockIdx], and the last block to arrive sums
// the partials in a fixed order and calls fin(total).  Bitwise reproducible for a fixed launch shape.
template <class Fin>
__device__ __forceinline__ void block_reduce_finalize(double v, double* partials, unsigned* counter, Fin fin) {
    __shared__ double warp_sums[32];
    __shared__ bool is_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) warp_sums[warp] = v;
    __syncthreads();
    if (warp == 0) {
        double w = (lane < nwarp) ? warp_sums[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_down_sync(0xffffffffu, w, o);
        if (lane == 0) {
            partials[blockIdx.x] = w;
            __threadfence();
            unsigned ticket = atomicAdd(counter, 1u);
            is_last = (ticket == gridDim.x - 1);
        }
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double acc = 0.0;
        for (unsigned i = threadIdx.x; i < gridDim.x; i += blockDim.x) acc += __ldcg(partials + i);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        __syncthreads();
        if (lane == 0) warp_sums[warp] = acc;
        __syncthreads();
        if (warp == 0) {
            double w = (lane < nwarp) ? warp_sums[lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) w += __shfl_down_sync(0xffffffffu, w, o);
            if (lane == 0) {
                *counter = 0u;
                fin(w);
            }
        }
    }
}

// ---------------------------------------------------------------------------- A2: Wilson-Dirac operator
// Forward hop of direction MU: acc += (1 + SG gamma_MU) sign U_MU(s) psi(s+MU)
template <int MU, int SG, class T>
__device__ __forceinline__ void hop_fwd(const Geom& g, const typename Vec2<T>::type* U, const typename Vec2<T>::type* in,
                                        const Site& c, int s, cx<T> acc[12]) {
    const int sn = nbr_fwd(g, c, s, MU);
    cx<T> p[12], h[6], u[9], w[6];
    load_spinor<T>(in, g, sn, p);
    load_link<T>(U, g, MU, s, u);
    spin_project<MU, SG>(p, h);
    if (g.bc[MU] < 0 && c.x[MU] == g.L[MU] - 1) {
#pragma unroll
        for (int k = 0; k < 6; k++) h[k] = mk<T>(-h[k].re, -h[k].im);
    }
    su3_mul_half(u, h, w);
    spin_reconstruct_add<MU, SG>(w, acc);
}
// Backward hop: acc += (1 + SG gamma_MU) sign U_MU^dag(s-MU) psi(s-MU)
template <int MU, int SG, class T>
__device__ __forceinline__ void hop_bwd(const Geom& g, const typename Vec2<T>::type* U, const typename Vec2<T>::type* in,
                                        const Site& c, int s, cx<T> acc[12]) {
    const int sn = nbr_bwd(g, c, s, MU);
    cx<T> p[12], h[6], u[9], w[6];
    load_spinor<T>(in, g, sn, p);
    load_link<T>(U, g, MU, sn, u);
    spin_project<MU, SG>(p, h);
    if (g.bc[MU] < 0 && c.x[MU] == 0) {
#pragma unroll
        for (int k = 0; k < 6; k++) h[k] = mk<T>(-h[k].re, -h[k].im);
    }
    su3_dag_mul_half(u, h, w);
    spin_reconstruct_add<MU, SG>(w, acc);
}

// out = D in (DAG = 0) or D^dag in (DAG = 1).  MODE 0: plain.  MODE 1: CG step "t = D p" with the fused
// reduction pAp = |t|^2 and alpha = rr / pAp.  MODE 2: CG step "q = D^dag t" (only the done-flag check).
template <class T, int DAG, int MODE>
__global__ void __launch_bounds__(128) dslash_kernel(Geom g, const typename Vec2<T>::type* __restrict__ U,
                                                     const typename Vec2<T>::type* __restrict__ in,
                                                     typename Vec2<T>::type* __restrict__ out, T kappa, CgState* st,
                                                     double* partials, unsigned* counter) {
    if (MODE != 0 && st->done) return;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    double nrm = 0.0;
    if (s < g.V) {
        const Site c = site_coords(g, s);
        cx<T> acc[12];
#pragma unroll
        for (int k = 0; k < 12; k++) acc[k] = mk<T>(0, 0);
        constexpr int F = DAG ? +1 : -1;  // D: (1 - gamma) forward, (1 + gamma) backward; D^dag: swapped
        hop_fwd<0, F, T>(g, U, in, c, s, acc);
        hop_bwd<0, -F, T>(g, U, in, c, s, acc);
        hop_fwd<1, F, T>(g, U, in, c, s, acc);
        hop_bwd<1, -F, T>(g, U, in, c, s, acc);
        hop_fwd<2, F, T>(g, U, in, c, s, acc);
        hop_bwd<2, -F, T>(g, U, in, c, s, acc);
        hop_fwd<3, F, T>(g, U, in, c, s, acc);
        hop_bwd<3, -F, T>(g, U, in, c, s, acc);
#pragma unroll
        for (int k = 0; k < 12; k++) {
            cx<T> p = ldc<T>(in + (size_t)k * g.Vs + s);
            cx<T> o = mk<T>(fma(-kappa, acc[k].re, p.re), fma(-kappa, acc[k].im, p.im));
            stc<T>(out + (size_t)k * g.Vs + s, o);
            if (MODE == 1) nrm += (double)o.re * (double)o.re + (double)o.im * (double)o.im;
        }
    }
    if (MODE == 1) {
        block_reduce_finalize(nrm, partials, counter, [st](double sum) {
            st->pAp = sum;
            st->alpha = st->rr / sum;
        });
    }
}

// ---------------------------------------------------------------------------- A3: CG BLAS-1 (fused)
// r = b, p = b, x = 0, rr = bb = |b|^2
template <class T>
__global__ void __launch_bounds__(256) cg_init_kernel(size_t n, const typename Vec2<T>::type* __restrict__ b,
                                                      typename Vec2<T>::type* __restrict__ x, typename Vec2<T>::type* __restrict__ r,
                                                      typename Vec2<T>::type* __restrict__ p, CgState* st, double tol2, int max_iter,
                                                      double* partials, unsigned* counter) {
    double acc = 0.0;
    typename Vec2<T>::type zero;
    zero.x = 0;
    zero.y = 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        typename Vec2<T>::type v = __ldg(b + i);
        x[i] = zero;
        r[i] = v;
        p[i] = v;
        acc += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
    }
    block_reduce_finalize(acc, partials, counter, [=](double sum) {
        st->rr = sum;
        st->bb = sum;
        st->pAp = 0.0;
        st->alpha = 0.0;
        st->beta = 0.0;
        st->tol2 = tol2;
        st->iter = 0;
        st->max_iter = max_iter;
        st->done = (!(sum > tol2 * sum) || max_iter <= 0) ? 1 : 0;
    });
}

// x += alpha p ; r -= alpha q ; rr_new = |r|^2 ; beta = rr_new / rr ; convergence test
template <class T>
__global__ void __launch_bounds__(256) cg_update_xr_kernel(size_t n, typename Vec2<T>::type* __restrict__ x,
                                                           typename Vec2<T>::type* __restrict__ r,
                                                           const typename Vec2<T>::type* __restrict__ p,
                                                           const typename Vec2<T>::type* __restrict__ q, CgState* st,
                                                           double* partials, unsigned* counter) {
    if (st->done) return;
    const T alpha = (T)st->alpha;
    double acc = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        typename Vec2<T>::type xv = x[i], rv = r[i], pv = __ldg(p + i), qv = __ldg(q + i);
        xv.x = fma(alpha, pv.x, xv.x);
        xv.y = fma(alpha, pv.y, xv.y);
        rv.x = fma(-alpha, qv.x, rv.x);
        rv.y = fma(-alpha, qv.y, rv.y);
        x[i] = xv;
        r[i] = rv;
        acc += (double)rv.x * (double)rv.x + (double)rv.y * (double)rv.y;
    }
    block_reduce_finalize(acc, partials, counter, [st](double sum) {
        st->beta = sum / st->rr;
        st->rr = sum;
        st->iter += 1;
        st->done = (!(sum > st->tol2 * st->bb) || st->iter >= st->max_iter) ? 1 : 0;
    });
}

// p = r + beta p
template <class T>
__global__ void __launch_bounds__(256) cg_update_p_kernel(size_t n, typename Vec2<T>::type* __restrict__ p,
                                                          const typename Vec2<T>::type* __restrict__ r, const CgState* st) {
    if (st->done) return;
    const T beta = (T)st->beta;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        typename Vec2<T>::type pv = p[i], rv = __ldg(r + i);
        pv.x = fma(beta, pv.x, rv.x);
        pv.y = fma(beta, pv.y, rv.y);
        p[i] = pv;
    }
}

// result = Re <a, b>
template <class T>
__global__ void __launch_bounds__(256) redot_kernel(size_t n, const typename Vec2<T>::type* __restrict__ a,
                                                    const typename Vec2<T>::type* __restrict__ b, double* result, double* partials,
                                                    unsigned* counter) {
    double acc = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        typename Vec2<T>::type av = __ldg(a + i), bv = __ldg(b + i);
        acc += (double)av.x * (double)bv.x + (double)av.y * (double)bv.y;
    }
    block_reduce_finalize(acc, partials, counter, [result](double sum) { *result = sum; });
}

// ---------------------------------------------------------------------------- A5: fused fermion force
// One thread per link (s, MU):  C = sum_t h^-[X(s+mu)]_t (x) conj(h^-[Y(s)]_t) + h^+[Y(s+mu)]_t (x) conj(h^+[X(s)]_t)
// (the half-spinor form of the spin trace, tests pin P11), M = sign U C, F = -kappa P_su(3)[M];
// ACC: Pi -= eps F in place, else F written in compact form.  No spin-colour intermediate touches HBM.
template <class T, int MU, int ACC>
__device__ __forceinline__ void fermion_force_link(const Geom& g, const typename Vec2<T>::type* U,
                                                   const typename Vec2<T>::type* X, const typename Vec2<T>::type* Y,
                                                   typename Vec2<T>::type* P, T kappa, T eps, int s) {
    const Site c = site_coords(g, s);
    const int sn = nbr_fwd(g, c, s, MU);
    cx<T> C[9];
    mat_zero(C);
    {
        cx<T> p[12], a[6], b[6];
        load_spinor<T>(X, g, sn, p);
        spin_project<MU, -1>(p, a);
        load_spinor<T>(Y, g, s, p);
        spin_project<MU, -1>(p, b);
#pragma unroll
        for (int t = 0; t < 2; t++)
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) cfma_jc(C[3 * i + j], a[3 * t + i], b[3 * t + j]);
        load_spinor<T>(Y, g, sn, p);
        spin_project<MU, +1>(p, a);
        load_spinor<T>(X, g, s, p);
        spin_project<MU, +1>(p, b);
#pragma unroll
        for (int t = 0; t < 2; t++)
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = 0; j < 3; j++) cfma_jc(C[3 * i + j], a[3 * t + i], b[3 * t + j]);
    }
    cx<T> u[9], M[9];
    load_link<T>(U, g, MU, s, u);
    mul_nn(u, C, M);
    T sc = -kappa;
    if (g.bc[MU] < 0 && c.x[MU] == g.L[MU] - 1) sc = kappa;
    T f[8];
    ta_compact(M, sc, f);
#pragma unroll
    for (int q = 0; q < 4; q++) {
        typename Vec2<T>::type* addr = P + (size_t)(4 * MU + q) * g.Vs + s;
        typename Vec2<T>::type v;
        if (ACC) {
            v = *addr;
            v.x = fma(-eps, f[2 * q], v.x);
            v.y = fma(-eps, f[2 * q + 1], v.y);
        } else {
            v.x = f[2 * q];
            v.y = f[2 * q + 1];
        }
        *addr = v;
    }
}

template <class T, int ACC>
__global__ void __launch_bounds__(128) fermion_force_kernel(Geom g, const typename Vec2<T>::type* __restrict__ U,
                                                            const typename Vec2<T>::type* __restrict__ X,
                                                            const typename Vec2<T>::type* __restrict__ Y,
                                                            typename Vec2<T>::type* __restrict__ P, T kappa, T eps) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    switch (blockIdx.y) {
        case 0: fermion_force_link<T, 0, ACC>(g, U, X, Y, P, kappa, eps, s); break;
        case 1: fermion_force_link<T, 1, ACC>(g, U, X, Y, P, kappa, eps, s); break;
        case 2: fermion_force_link<T, 2, ACC>(g, U, X, Y, P, kappa, eps, s); break;
        default: fermion_force_link<T, 3, ACC>(g, U, X, Y, P, kappa, eps, s); break;
    }
}

// ---------------------------------------------------------------------------- A4: staple gauge force
// One thread per link (s, mu): V = sum_{nu != mu} [U_nu(s+mu) U_mu^dag(s+nu) U_nu^dag(s)
//                                               + U_nu^dag(s+mu-nu) U_mu^dag(s-nu) U_nu(s-nu)],
// F = (beta/6) P_su(3)[U_mu(s) V]; ACC: Pi -= eps F.
template <class T, int ACC>
__global__ void __launch_bounds__(128) gauge_force_kernel(Geom g, const typename Vec2<T>::type* __restrict__ U,
                                                          typename Vec2<T>::type* __restrict__ P, T beta_over_6, T eps) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    const int mu = blockIdx.y;
    const Site c = site_coords(g, s);
    const int smu = nbr_fwd(g, c, s, mu);
    cx<T> V[9];
    mat_zero(V);
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu) continue;
        cx<T> a[9], b[9], t[9], r[9];
        const int snu = nbr_fwd(g, c, s, nu);
        // up: U_nu(s+mu) (U_nu(s) U_mu(s+nu))^dag
        load_link<T>(U, g, nu, s, a);
        load_link<T>(U, g, mu, snu, b);
        mul_nn(a, b, t);
        load_link<T>(U, g, nu, smu, a);
        mul_nd(a, t, r);
#pragma unroll
        for (int k = 0; k < 9; k++) V[k] = V[k] + r[k];
        // down: (U_mu(s-nu) U_nu(s+mu-nu))^dag U_nu(s-nu)
        const int sdn = nbr_bwd(g, c, s, nu);
        Site cm = c;
        cm.x[mu] = (c.x[mu] == g.L[mu] - 1) ? 0 : c.x[mu] + 1;
        const int smudn = nbr_bwd(g, cm, smu, nu);
        load_link<T>(U, g, mu, sdn, a);
        load_link<T>(U, g, nu, smudn, b);
        mul_nn(a, b, t);
        load_link<T>(U, g, nu, sdn, a);
        mul_dn(t, a, r);
#pragma unroll
        for (int k = 0; k < 9; k++) V[k] = V[k] + r[k];
    }
    cx<T> u[9], M[9];
    load_link<T>(U, g, mu, s, u);
    mul_nn(u, V, M);
    T f[8];
    ta_compact(M, beta_over_6, f);
#pragma unroll
    for (int q = 0; q < 4; q++) {
        typename Vec2<T>::type* addr = P + (size_t)(4 * mu + q) * g.Vs + s;
        typename Vec2<T>::type v;
        if (ACC) {
            v = *addr;
            v.x = fma(-eps, f[2 * q], v.x);
            v.y = fma(-eps, f[2 * q + 1], v.y);
        } else {
            v.x = f[2 * q];
            v.y = f[2 * q + 1];
        }
        *addr = v;
    }
}

// ---------------------------------------------------------------------------- A6: link update
// U_mu(s) <- exp(eps Pi_mu(s)) U_mu(s) with exp(iQ), Q = -i eps Pi traceless Hermitian, by the Cayley-Hamilton
// form of the paper's ref. [6]: exp(iQ) = f0 + f1 Q + f2 Q^2.
template <class T> __device__ __forceinline__ void exp_iQ(const cx<T> Q[9], cx<T> E[9]) {
    cx<T> Q2[9];
    mul_nn(Q, Q, Q2);
    // c0 = det Q (real), c1 = tr Q^2 / 2
    cx<T> d0 = Q[4] * Q[8] - Q[5] * Q[7];
    cx<T> d1 = Q[3] * Q[8] - Q[5] * Q[6];
    cx<T> d2 = Q[3] * Q[7] - Q[4] * Q[6];
    T c0 = (Q[0] * d0 - Q[1] * d1 + Q[2] * d2).re;
    T c1 = (T)0.5 * (Q2[0].re + Q2[4].re + Q2[8].re);
    // |Q|^2 below the square of the working precision: exp(iQ) = 1 + iQ to rounding
    if (!(c1 > (sizeof(T) == 8 ? (T)1e-30 : (T)1e-12))) {
#pragma unroll
        for (int k = 0; k < 9; k++) E[k] = times_i(Q[k]);
        E[0].re += 1;
        E[4].re += 1;
        E[8].re += 1;
        return;
    }
    const bool neg = c0 < 0;
    c0 = fabs(c0);
    T c1_3 = c1 * (T)(1.0 / 3.0);
    T c0max = 2 * c1_3 * sqrt(c1_3);
    T ratio = c0 / c0max;
    T theta = acos(ratio > 1 ? (T)1 : ratio);
    T su, cu_;
    sincos(theta * (T)(1.0 / 3.0), &su, &cu_);
    T u = sqrt(c1_3) * cu_;
    T w = sqrt(c1) * su;
    T u2 = u * u, w2 = w * w;
    T sw, cw;
    sincos(w, &sw, &cw);
    T xi0;
    if (fabs(w) < (T)0.05)
        xi0 = 1 - w2 * (T)(1.0 / 6.0) * (1 - w2 * (T)(1.0 / 20.0) * (1 - w2 * (T)(1.0 / 42.0)));
    else
        xi0 = sw / w;
    T s2u, c2u, s1u, c1u;
    sincos(2 * u, &s2u, &c2u);
    sincos(u, &s1u, &c1u);
    cx<T> e2 = mk<T>(c2u, s2u);   // exp(2iu)
    cx<T> em = mk<T>(c1u, -s1u);  // exp(-iu)
    cx<T> h0 = (u2 - w2) * e2 + em * mk<T>(8 * u2 * cw, 2 * u * (3 * u2 + w2) * xi0);
    cx<T> h1 = (2 * u) * e2 - em * mk<T>(2 * u * cw, -(3 * u2 - w2) * xi0);
    cx<T> h2 = e2 - em * mk<T>(cw, 3 * u * xi0);
    T inv = 1 / (9 * u2 - w2);
    cx<T> f0 = inv * h0, f1 = inv * h1, f2 = inv * h2;
    if (neg) {
        f0 = conj(f0);
        f1 = mk<T>(-f1.re, f1.im);
        f2 = conj(f2);
    }
#pragma unroll
    for (int k = 0; k < 9; k++) E[k] = f1 * Q[k] + f2 * Q2[k];
    E[0] = E[0] + f0;
    E[4] = E[4] + f0;
    E[8] = E[8] + f0;
}

template <class T>
__global__ void __launch_bounds__(128) link_update_kernel(Geom g, typename Vec2<T>::type* __restrict__ U,
                                                          const typename Vec2<T>::type* __restrict__ P, T eps) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    const int mu = blockIdx.y;
    T c[8];
#pragma unroll
    for (int q = 0; q < 4; q++) {
        typename Vec2<T>::type v = __ldg(P + (size_t)(4 * mu + q) * g.Vs + s);
        c[2 * q] = v.x;
        c[2 * q + 1] = v.y;
    }
    // Q = -i eps Pi:  Pi_kk = i c_k -> Q_kk = eps c_k ;  Pi_01 = (re, im) -> Q_01 = eps (im, -re), Q_10 = conj(Q_01)
    cx<T> Q[9];
    Q[0] = mk<T>(eps * c[0], 0);
    Q[4] = mk<T>(eps * c[1], 0);
    Q[8] = mk<T>(-eps * (c[0] + c[1]), 0);
    Q[1] = mk<T>(eps * c[3], -eps * c[2]);
    Q[3] = conj(Q[1]);
    Q[2] = mk<T>(eps * c[5], -eps * c[4]);
    Q[6] = conj(Q[2]);
    Q[5] = mk<T>(eps * c[7], -eps * c[6]);
    Q[7] = conj(Q[5]);
    cx<T> E[9], u[9], r[9];
    exp_iQ(Q, E);
#pragma unroll
    for (int k = 0; k < 9; k++) u[k] = ldc_rw<T>(U + (size_t)(9 * mu + k) * g.Vs + s);
    mul_nn(E, u, r);
#pragma unroll
    for (int k = 0; k < 9; k++) stc<T>(U + (size_t)(9 * mu + k) * g.Vs + s, r[k]);
}

// ---------------------------------------------------------------------------- A1: actions
// result = sum_x sum_{mu<nu} Re tr U_P / 3
template <class T>
__global__ void __launch_bounds__(128) plaquette_kernel(Geom g, const typename Vec2<T>::type* __restrict__ U, double* result,
                                                        double* partials, unsigned* counter) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    double acc = 0.0;
    if (s < g.V) {
        const Site c = site_coords(g, s);
        for (int mu = 0; mu < 4; mu++) {
            const int smu = nbr_fwd(g, c, s, mu);
            for (int nu = mu + 1; nu < 4; nu++) {
                const int snu = nbr_fwd(g, c, s, nu);
                cx<T> a[9], b[9], t1[9], t2[9];
                load_link<T>(U, g, mu, s, a);
                load_link<T>(U, g, nu, smu, b);
                mul_nn(a, b, t1);  // U_mu(s) U_nu(s+mu)
                load_link<T>(U, g, nu, s, a);
                load_link<T>(U, g, mu, snu, b);
                mul_nn(a, b, t2);  // U_nu(s) U_mu(s+nu)
                // Re tr(t1 t2^dag)
                T tr = 0;
#pragma unroll
                for (int k = 0; k < 9; k++) tr += t1[k].re * t2[k].re + t1[k].im * t2[k].im;
                acc += (double)tr;
            }
        }
        acc *= (1.0 / 3.0);
    }
    block_reduce_finalize(acc, partials, counter, [result](double sum) { *result = sum; });
}

// result = sum ||Pi||_F^2 from the compact form
template <class T>
__global__ void __launch_bounds__(256) kinetic_kernel(Geom g, const typename Vec2<T>::type* __restrict__ P, double* result,
                                                      double* partials, unsigned* counter) {
    double acc = 0.0;
    const size_t nlinks = (size_t)4 * g.V;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nlinks; i += (size_t)gridDim.x * blockDim.x) {
        const int mu = (int)(i / g.V), s = (int)(i % g.V);
        typename Vec2<T>::type d = __ldg(P + (size_t)(4 * mu) * g.Vs + s);
        double d0 = d.x, d1 = d.y, d2 = -(d0 + d1);
        double off = 0.0;
#pragma unroll
        for (int q = 1; q < 4; q++) {
            typename Vec2<T>::type v = __ldg(P + (size_t)(4 * mu + q) * g.Vs + s);
            off += (double)v.x * v.x + (double)v.y * v.y;
        }
        acc += d0 * d0 + d1 * d1 + d2 * d2 + 2.0 * off;
    }
    block_reduce_finalize(acc, partials, counter, [result](double sum) { *result = sum; });
}

// ---------------------------------------------------------------------------- layout conversion
// DIR 0: canonical [V][ncomp] complex -> native [ncomp][Vs];  DIR 1: back.
template <class T, int DIR>
__global__ void __launch_bounds__(256) reorder_kernel(int V, int Vs, int ncomp, const typename Vec2<T>::type* __restrict__ src,
                                                      typename Vec2<T>::type* __restrict__ dst) {
    const size_t n = (size_t)V * ncomp;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        // i enumerates the native order (k, s): coalesced on the native side
        const int k = (int)(i / V), s = (int)(i % V);
        if (DIR == 0)
            dst[(size_t)k * Vs + s] = __ldg(src + (size_t)s * ncomp + k);
        else
            dst[(size_t)s * ncomp + k] = __ldg(src + (size_t)k * Vs + s);
    }
}

// canonical full 3x3 momenta [V][4][3][3] <-> compact native [4][4][Vs].  DIR 0 keeps the traceless
// anti-Hermitian part of the input (P_su(3)).
template <class T, int DIR>
__global__ void __launch_bounds__(256) momenta_reorder_kernel(int V, int Vs, const typename Vec2<T>::type* src,
                                                              typename Vec2<T>::type* dst) {
    const size_t n = (size_t)4 * V;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int mu = (int)(i / V), s = (int)(i % V);
        if (DIR == 0) {
            cx<T> m[9];
#pragma unroll
            for (int k = 0; k < 9; k++) m[k] = ldc<T>(src + ((size_t)s * 4 + mu) * 9 + k);
            T c[8];
            ta_compact(m, (T)1, c);
#pragma unroll
            for (int q = 0; q < 4; q++) {
                typename Vec2<T>::type v;
                v.x = c[2 * q];
                v.y = c[2 * q + 1];
                dst[(size_t)(4 * mu + q) * Vs + s] = v;
            }
        } else {
            T c[8];
#pragma unroll
            for (int q = 0; q < 4; q++) {
                typename Vec2<T>::type v = __ldg(src + (size_t)(4 * mu + q) * Vs + s);
                c[2 * q] = v.x;
                c[2 * q + 1] = v.y;
            }
            cx<T> m[9];
            compact_expand(c, m);
#pragma unroll
            for (int k = 0; k < 9; k++) stc<T>(dst + ((size_t)s * 4 + mu) * 9 + k, m[k]);
        }
    }
}

template <class T>
__global__ void __launch_bounds__(256) unit_links_kernel(int V, int Vs, typename Vec2<T>::type* U) {
    const size_t n = (size_t)36 * V;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int k = (int)(i / V) % 9, s = (int)(i % V);
        typename Vec2<T>::type v;
        v.x = (k == 0 || k == 4 || k == 8) ? 1 : 0;
        v.y = 0;
        U[(i / V) * (size_t)Vs + s] = v;
    }
}

}  // namespace lgt
