// nd_su3.cuh - loading an SU(3) link from its 18 / 12 / 8 stored reals and rebuilding the 3x3 matrix in registers
// (eq. 2.3; 8-parameter form: DESIGN.md R8).  Used by the stencil and by nd_get_gauge.
#pragma once
#include "nd_internal.cuh"

template <typename T> __device__ __forceinline__ T ldg_vec(const T* p) { return __ldg(p); }

// ------------------------------------------------------------------------------------- link reconstruction
template <typename T> __device__ __forceinline__ void unpack_reals(const float2& v, T* r) { r[0] = v.x; r[1] = v.y; }
template <typename T> __device__ __forceinline__ void unpack_reals(const float4& v, T* r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
template <typename T> __device__ __forceinline__ void unpack_reals(const double2& v, T* r) { r[0] = v.x; r[1] = v.y; }

// fp32: the special-function unit's sqrt / reciprocal (one MUFU instruction each, <= 1-2 ulp) - the 8-parameter form is bound by
// its reconstruction arithmetic, not by memory, and its rounding error is dominated by the 1/N amplification (R8),
// not by the last ulp of these two; the arguments are never denormal (N >= 1e-6 is enforced by nd_set_gauge, 1 + q^2 >= 1).
__device__ __forceinline__ float nd_sqrt(float x) { float r; asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float nd_rcp(float x) { float r; asm("rcp.approx.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
// fp64: correctly rounded reciprocal (rcp.rn): a handful of instructions instead of the general division routine
__device__ __forceinline__ double nd_rcp(double x) { return __drcp_rn(x); }
__device__ __forceinline__ double nd_sqrt(double x) { return sqrt(x); }
__device__ __forceinline__ float nd_max0(float x) { return fmaxf(x, 0.f); }
__device__ __forceinline__ double nd_max0(double x) { return fmax(x, 0.0); }

// (sin theta, cos theta) from q = tan(theta/4), |q| <= 1: half-angle rational form, then one angle doubling.  Exact up to
// a few roundings for every theta in [-pi, pi]; replaces an accurate sincos (R8) at a tenth of its instructions.
template <typename T> __device__ __forceinline__ void phase_from_quarter_tan(T q, T& s, T& c) {
    const T q2 = q * q;
    const T inv = nd_rcp(T(1) + q2);
    const T ch = (T(1) - q2) * inv;   // cos(theta/2)
    const T sh = (q + q) * inv;       // sin(theta/2)
    c = (ch - sh) * (ch + sh);
    s = (sh + sh) * ch;
}

// third row from the first two: c = (a x b)^*   (eq. 2.3 applied to rows; U^T is SU(3) too)
template <typename T> __device__ __forceinline__ void third_row(cx<T> (&U)[3][3]) {
    U[2][0] = cj(U[0][1] * U[1][2] - U[0][2] * U[1][1]);
    U[2][1] = cj(U[0][2] * U[1][0] - U[0][0] * U[1][2]);
    U[2][2] = cj(U[0][0] * U[1][1] - U[0][1] * U[1][0]);
}

// the NL stored words of link (mu, s), as they sit in memory
template <typename T, int RECON>
__device__ __forceinline__ void load_link_words(const typename LinkLayout<T, RECON>::LVec* __restrict__ g, long long V, int mu,
                                                long long s, typename LinkLayout<T, RECON>::LVec (&w)[LinkLayout<T, RECON>::NL]) {
    using LL = LinkLayout<T, RECON>;
    const typename LL::LVec* base = g + (long long)mu * LL::NL * V + s;
#pragma unroll
    for (int p = 0; p < LL::NL; p++) w[p] = ldg_vec(base + p * V);
}

// the 3x3 matrix from the stored words, in registers
template <typename T, int RECON>
__device__ __forceinline__ void reconstruct_link(const typename LinkLayout<T, RECON>::LVec (&w)[LinkLayout<T, RECON>::NL],
                                                 cx<T> (&U)[3][3]) {
    using LL = LinkLayout<T, RECON>;
    constexpr int W = sizeof(typename LL::LVec) / sizeof(T);
    T r[LL::NL * W];
#pragma unroll
    for (int p = 0; p < LL::NL; p++) unpack_reals<T>(w[p], r + p * W);
    if (RECON == 18) {
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int j = 0; j < 3; j++) U[i][j] = {r[2 * (3 * i + j)], r[2 * (3 * i + j) + 1]};
    } else if (RECON == 12) {
#pragma unroll
        for (int i = 0; i < 2; i++)
#pragma unroll
            for (int j = 0; j < 3; j++) U[i][j] = {r[2 * (3 * i + j)], r[2 * (3 * i + j) + 1]};
        third_row(U);
    } else {
        // 8 reals: a2, a3, b1, tan(theta1/4), tan(theta2/4) with theta1 = arg a1, theta2 = arg c1 (rows a, b, c; R8)
        cx<T> a2 = {r[0], r[1]}, a3 = {r[2], r[3]}, b1 = {r[4], r[5]};
        T N = a2.re * a2.re + a2.im * a2.im + a3.re * a3.re + a3.im * a3.im;
        T s1, c1, s2, c2;
        phase_from_quarter_tan(r[6], s1, c1);
        phase_from_quarter_tan(r[7], s2, c2);
        T ra = nd_sqrt(nd_max0(T(1) - N));
        T rc = nd_sqrt(nd_max0(N - (b1.re * b1.re + b1.im * b1.im)));
        cx<T> a1 = {ra * c1, ra * s1};
        cx<T> cc1 = {rc * c2, rc * s2};
        T inv = nd_rcp(N);
        // b2 = -(a1^* a2 b1 + a3^* c1^*)/N ,  b3 = (a2^* c1^* - a1^* a3 b1)/N
        cx<T> a1c_b1 = cj(a1) * b1;
        cx<T> t2 = a1c_b1 * a2 + cj(a3) * cj(cc1);
        cx<T> t3 = cj(a2) * cj(cc1) - a1c_b1 * a3;
        U[0][0] = a1; U[0][1] = a2; U[0][2] = a3;
        U[1][0] = b1; U[1][1] = {-t2.re * inv, -t2.im * inv}; U[1][2] = {t3.re * inv, t3.im * inv};
        U[2][0] = cc1;
        U[2][1] = cj(U[0][2] * U[1][0] - U[0][0] * U[1][2]);
        U[2][2] = cj(U[0][0] * U[1][1] - U[0][1] * U[1][0]);
    }
}


template <typename T, int RECON>
__device__ __forceinline__ void load_link(const typename LinkLayout<T, RECON>::LVec* __restrict__ g, long long V, int mu,
                                          long long s, cx<T> (&U)[3][3]) {
    typename LinkLayout<T, RECON>::LVec w[LinkLayout<T, RECON>::NL];
    load_link_words<T, RECON>(g, V, mu, s, w);
    reconstruct_link<T, RECON>(w, U);
}
