// nd_dirac.cuh - the spin / colour algebra of one hop of the Wilson-Dirac stencil (eq. 2.1-2.2), shared by
// the stencil kernels (wilson.cu: site-per-thread and hop-parallel kernels; wilson_tile.cu: tiled marching kernel).
//
// Chiral basis (R2): gamma_mu = [[0, A_mu], [A_mu^dagger, 0]], A_0 = -1, A_k = -i sigma_k, gamma5 = diag(1,1,-1,-1).
//   (1-gamma_mu) psi = (h, -A^dagger h),  h  = psi_up - A psi_low
//   (1+gamma_mu) psi = (h',  A^dagger h'), h' = psi_up + A psi_low
#pragma once
#include "nd_internal.cuh"
#include "nd_su3.cuh"

template <typename T>
__device__ __forceinline__ void load_spinor(const typename Prec<T>::Vec* __restrict__ f, long long V, long long s,
                                            cx<T> (&c)[12]) {
    typename Prec<T>::Vec w[Prec<T>::NV];
#pragma unroll
    for (int p = 0; p < Prec<T>::NV; p++) w[p] = ldg_vec(f + p * V + s);
    words_to_cx(w, c);
}

// g = U h (colour mat-vec for both spin components of the half-spinor)
template <typename T> __device__ __forceinline__ void mul_U(const cx<T> (&U)[3][3], const cx<T> (&h)[2][3], cx<T> (&g)[2][3]) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int i = 0; i < 3; i++) {
            cx<T> a = U[i][0] * h[s][0];
            cfma(a, U[i][1], h[s][1]);
            cfma(a, U[i][2], h[s][2]);
            g[s][i] = a;
        }
}
// g = U^dagger h
template <typename T> __device__ __forceinline__ void mul_Udag(const cx<T> (&U)[3][3], const cx<T> (&h)[2][3], cx<T> (&g)[2][3]) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int i = 0; i < 3; i++) {
            cx<T> a = cj(U[0][i]) * h[s][0];
            cfma_cj(a, U[1][i], h[s][1]);
            cfma_cj(a, U[2][i], h[s][2]);
            g[s][i] = a;
        }
}

// Spin projection: h = psi_up -/+ A_mu psi_low   (SGN = -1: (1-gamma_mu), forward hop; +1: (1+gamma_mu), backward hop)
template <typename T, int MU, int SGN>
__device__ __forceinline__ void project(const cx<T> (&p)[12], T phase, cx<T> (&h)[2][3]) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        cx<T> u0 = p[c], u1 = p[3 + c], l0 = p[6 + c], l1 = p[9 + c];
        cx<T> a, b;   // a = (A psi_low)_0, b = (A psi_low)_1
        if (MU == 0) { a = {-l0.re, -l0.im}; b = {-l1.re, -l1.im}; }
        else if (MU == 1) { a = times_mi(l1); b = times_mi(l0); }
        else if (MU == 2) { a = {-l1.re, -l1.im}; b = l0; }
        else { a = times_mi(l0); b = times_i(l1); }
        cx<T> h0 = (SGN < 0) ? (u0 - a) : (u0 + a);
        cx<T> h1 = (SGN < 0) ? (u1 - b) : (u1 + b);
        h[0][c] = {phase * h0.re, phase * h0.im};
        h[1][c] = {phase * h1.re, phase * h1.im};
    }
}

// acc += (g, -/+ A^dagger g)   (SGN = -1: lower = -A^dagger g; +1: lower = +A^dagger g)
template <typename T, int MU, int SGN>
__device__ __forceinline__ void accumulate(const cx<T> (&g)[2][3], cx<T> (&acc)[12]) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        acc[c] = acc[c] + g[0][c];
        acc[3 + c] = acc[3 + c] + g[1][c];
        cx<T> d0, d1;   // A^dagger g
        if (MU == 0) { d0 = {-g[0][c].re, -g[0][c].im}; d1 = {-g[1][c].re, -g[1][c].im}; }
        else if (MU == 1) { d0 = times_i(g[1][c]); d1 = times_i(g[0][c]); }
        else if (MU == 2) { d0 = g[1][c]; d1 = {-g[0][c].re, -g[0][c].im}; }
        else { d0 = times_i(g[0][c]); d1 = times_mi(g[1][c]); }
        if (SGN < 0) { acc[6 + c] = acc[6 + c] - d0; acc[9 + c] = acc[9 + c] - d1; }
        else { acc[6 + c] = acc[6 + c] + d0; acc[9 + c] = acc[9 + c] + d1; }
    }
}

// out(x) = gamma5 [ -1/2 acc ] (acc holds -2 (4+m) phi(x) + the eight hops), optionally followed by the fused vector update
// out = s0*Q(in) + s1*v1 + s2*v2 + s3*v3.  out may alias any v_i (the Clenshaw step passes v2 == out): neither out nor the
// v_i are __restrict__, every v_i(x) is read before out(x) is written, and no other thread touches site x.
template <typename T, bool EPI>
__device__ __forceinline__ void finish_site(typename Prec<T>::Vec* out, long long V, long long s,
                                            const cx<T> (&acc)[12], T s0, T s1,
                                            const typename Prec<T>::Vec* v1, T s2, const typename Prec<T>::Vec* v2, T s3,
                                            const typename Prec<T>::Vec* v3) {
    using Vec = typename Prec<T>::Vec;
    constexpr int NV = Prec<T>::NV;
    cx<T> res[12];
#pragma unroll
    for (int i = 0; i < 12; i++) {
        const T sg = (i < 6) ? T(-0.5) : T(0.5);
        res[i].re = sg * acc[i].re;
        res[i].im = sg * acc[i].im;
    }
    Vec w[NV];
    cx_to_words(res, w);
    if (EPI) {
        T* wr = reinterpret_cast<T*>(w);
        constexpr int NR = 24;
#pragma unroll
        for (int i = 0; i < NR; i++) wr[i] *= s0;
        const Vec* vs[3] = {v1, v2, v3};
        const T ss[3] = {s1, s2, s3};
#pragma unroll
        for (int j = 0; j < 3; j++) {
            if (vs[j]) {
#pragma unroll
                for (int p = 0; p < NV; p++) {
                    Vec a = vs[j][p * V + s];
                    const T* ar = reinterpret_cast<const T*>(&a);
#pragma unroll
                    for (int k = 0; k < NR / NV; k++) wr[p * (NR / NV) + k] = fma(ss[j], ar[k], wr[p * (NR / NV) + k]);
                }
            }
        }
    }
#pragma unroll
    for (int p = 0; p < NV; p++) out[p * V + s] = w[p];
}

