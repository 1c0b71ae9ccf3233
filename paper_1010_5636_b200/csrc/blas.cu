// blas.cu - BLAS-1 on spinor fields (BASELINE.json north_star; implied by PAPER.md:L66,L79) and the low-mode
// projection kernels  w_k = <u_k, x>  and  y <- y + sum_k a_k u_k  (eq. 2.7 / 2.11).
// All reductions accumulate in fp64 (both precisions): thread partials -> warp shuffle -> per-warp shared row ->
// per-block partial -> second-stage kernel.  No atomics: results are bitwise reproducible run to run.
#include <vector>

#include "nd_internal.cuh"

namespace {

constexpr int RED_THREADS = 128;
constexpr int RED_WARPS = RED_THREADS / 32;

template <typename T> struct Words;   // one site's words <-> 12 complex in fp64 for accumulation

template <typename T>
__device__ __forceinline__ void load_site(const typename Prec<T>::Vec* __restrict__ f, long long V, long long s, cx<T> (&c)[12]) {
    typename Prec<T>::Vec w[Prec<T>::NV];
#pragma unroll
    for (int p = 0; p < Prec<T>::NV; p++) w[p] = f[p * V + s];
    words_to_cx(w, c);
}
template <typename T>
__device__ __forceinline__ void store_site(typename Prec<T>::Vec* __restrict__ f, long long V, long long s, const cx<T> (&c)[12]) {
    typename Prec<T>::Vec w[Prec<T>::NV];
    cx_to_words(c, w);
#pragma unroll
    for (int p = 0; p < Prec<T>::NV; p++) f[p * V + s] = w[p];
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ------------------------------------------------------------------------------------------- elementwise
// y <- a x + y   (complex a)
template <typename T>
__global__ void axpy_kernel(typename Prec<T>::Vec* __restrict__ y, const typename Prec<T>::Vec* __restrict__ x, T ar, T ai, long long V) {
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < V; s += (long long)gridDim.x * blockDim.x) {
        cx<T> cxv[12], cy[12];
        load_site<T>(x, V, s, cxv);
        load_site<T>(y, V, s, cy);
        const cx<T> a = {ar, ai};
#pragma unroll
        for (int i = 0; i < 12; i++) cfma(cy[i], a, cxv[i]);
        store_site<T>(y, V, s, cy);
    }
}
template <typename T>
__global__ void scale_kernel(typename Prec<T>::Vec* __restrict__ x, T ar, T ai, long long V) {
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < V; s += (long long)gridDim.x * blockDim.x) {
        cx<T> c[12];
        load_site<T>(x, V, s, c);
        const cx<T> a = {ar, ai};
#pragma unroll
        for (int i = 0; i < 12; i++) c[i] = a * c[i];
        store_site<T>(x, V, s, c);
    }
}
// y <- gamma5 x : negate spin components 2, 3 (chiral basis, gamma5 = diag(1,1,-1,-1))
template <typename T>
__global__ void gamma5_kernel(typename Prec<T>::Vec* y, const typename Prec<T>::Vec* x, long long V) {
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < V; s += (long long)gridDim.x * blockDim.x) {
        cx<T> c[12];
        load_site<T>(x, V, s, c);
#pragma unroll
        for (int i = 6; i < 12; i++) c[i] = {-c[i].re, -c[i].im};
        store_site<T>(y, V, s, c);
    }
}

// y <- P_sigma u + c y,  P_sigma = (1 + sigma gamma5)/2: keep the spin components of chirality sigma of u (0, 1 for +1; 2, 3 for -1),
// zero the others (index by zero-mode counting: D_N^dagger D_N commutes with gamma5 and is diagonalised sector
// by sector).  c == 0: y is not read.
template <typename T>
__global__ void chiral_combine_kernel(typename Prec<T>::Vec* y, const typename Prec<T>::Vec* u, int sigma, T c, long long V) {
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < V; s += (long long)gridDim.x * blockDim.x) {
        cx<T> cu[12], cy[12];
        load_site<T>(u, V, s, cu);
        if (c != T(0)) load_site<T>(y, V, s, cy);
        const int lo = (sigma > 0) ? 0 : 6;
#pragma unroll
        for (int i = 0; i < 12; i++) {
            const bool keep = (i >= lo && i < lo + 6);
            cx<T> r = keep ? cu[i] : cx<T>{T(0), T(0)};
            if (c != T(0)) { r.re = fma(c, cy[i].re, r.re); r.im = fma(c, cy[i].im, r.im); }
            cy[i] = r;
        }
        store_site<T>(y, V, s, cy);
    }
}

// --------------------------------------------------------------------------------------- block dot product
// <v_k, x_c> for k < l vectors of a block and up to NC columns x_c given by pointer (eq. 2.7 / 2.11: V^dagger psi; the
// eigen-solver's Gram matrices).  Both operands move through HBM exactly once:
//   a CTA takes ranges of DOT_RANGE consecutive sites; the NC columns of the range are staged in shared memory ONCE, then
//   the block's vectors are streamed: for every k each thread reads its sites of v_k (coalesced, each element of the block
//   is read by exactly one thread of the grid), multiplies with the staged columns and accumulates in fp64 registers; one
//   warp reduction per (k, column) and RANGE, accumulated per CTA in shared memory;
//   partial[((c*l + k)*2 + {re,im})][cta]  ->  reduce_partials_kernel.  No atomics: bitwise reproducible.
//   On small lattices with many vectors (16^3x32, l = 50) grid.y splits the block's vectors into chunks so that the machine is
//   filled through l as well (fp64: 532 -> 287 us).
struct ColPtrs {
    const void* p[8];
};
constexpr int DOT_SITES_PER_THREAD = 2;
constexpr int DOT_RANGE = RED_THREADS * DOT_SITES_PER_THREAD;

template <typename T, int NC>
__global__ void __launch_bounds__(RED_THREADS) block_dot_cols_kernel(double* __restrict__ partial, int l, int nc,
                                                                     const typename Prec<T>::Vec* __restrict__ v, ColPtrs cols, long long V) {
    using Vec = typename Prec<T>::Vec;
    constexpr int NV = Prec<T>::NV;
    extern __shared__ __align__(16) unsigned char dsm[];
    Vec* xs = reinterpret_cast<Vec*>(dsm);                                              // [NC][NV][DOT_RANGE]
    double* acc = reinterpret_cast<double*>(dsm + (size_t)NC * NV * DOT_RANGE * sizeof(Vec));   // [nc*l*2] CTA totals
    double* wred = acc + (size_t)2 * NC * l;                                            // [RED_WARPS][2*NC]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // blockIdx.y = chunk of the block's vectors [kb, ke): small lattices with many vectors fill the machine through l as well
    const int kchunk = (l + (int)gridDim.y - 1) / (int)gridDim.y;
    const int kb = (int)blockIdx.y * kchunk, ke = (kb + kchunk < l) ? kb + kchunk : l;
    for (int i = threadIdx.x; i < 2 * nc * l; i += blockDim.x) acc[i] = 0.0;
    const long long nranges = (V + DOT_RANGE - 1) / DOT_RANGE;
    for (long long rg = blockIdx.x; rg < nranges; rg += gridDim.x) {
        const long long base = rg * DOT_RANGE;
        __syncthreads();   // the previous range's columns are no longer read; acc initialised
        for (int c = 0; c < nc; c++) {
            const Vec* xc = reinterpret_cast<const Vec*>(cols.p[c]);
#pragma unroll
            for (int p = 0; p < NV; p++)
#pragma unroll
                for (int j = 0; j < DOT_SITES_PER_THREAD; j++) {
                    const long long s = base + j * RED_THREADS + threadIdx.x;
                    Vec w;
                    T* wr = reinterpret_cast<T*>(&w);
#pragma unroll
                    for (int q = 0; q < (int)(sizeof(Vec) / sizeof(T)); q++) wr[q] = T(0);
                    if (s < V) w = xc[p * V + s];
                    xs[(c * NV + p) * DOT_RANGE + j * RED_THREADS + threadIdx.x] = w;
                }
        }
        __syncthreads();
        for (int k = kb; k < ke; k++) {
            const Vec* vk = v + (long long)k * NV * V;
            double re[NC], im[NC];
#pragma unroll
            for (int c = 0; c < NC; c++) re[c] = im[c] = 0.0;
            // fp64: the loads of both sites are issued before the first multiply (853 -> 722 us at 32^3x64, l = 8); fp32: one site
            // at a time (the same change costs registers there: 325 -> 397 us)
            cx<T> bb[DOT_SITES_PER_THREAD][12];
            if (sizeof(T) == 8) {
#pragma unroll
                for (int j = 0; j < DOT_SITES_PER_THREAD; j++) {
                    const long long s = base + j * RED_THREADS + threadIdx.x;
                    if (s < V) load_site<T>(vk, V, s, bb[j]);
                }
            }
#pragma unroll
            for (int j = 0; j < DOT_SITES_PER_THREAD; j++) {
                const long long s = base + j * RED_THREADS + threadIdx.x;
                if (s < V) {
                    cx<T> (&b)[12] = bb[j];
                    if (sizeof(T) != 8) load_site<T>(vk, V, s, b);
#pragma unroll
                    for (int c = 0; c < NC; c++) {
                        if (c < nc) {
                            Vec w[NV];
#pragma unroll
                            for (int p = 0; p < NV; p++) w[p] = xs[(c * NV + p) * DOT_RANGE + j * RED_THREADS + threadIdx.x];
                            cx<T> a[12];
                            words_to_cx(w, a);
#pragma unroll
                            for (int i = 0; i < 12; i++) {
                                const double br = (double)b[i].re, bi = (double)b[i].im, xr = (double)a[i].re, xi = (double)a[i].im;
                                re[c] = fma(br, xr, re[c]);
                                re[c] = fma(bi, xi, re[c]);
                                im[c] = fma(br, xi, im[c]);
                                im[c] = fma(-bi, xr, im[c]);
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int c = 0; c < NC; c++) {
                re[c] = warp_sum(re[c]);
                im[c] = warp_sum(im[c]);
                if (lane == 0) { wred[warp * 2 * NC + 2 * c] = re[c]; wred[warp * 2 * NC + 2 * c + 1] = im[c]; }
            }
            __syncthreads();
            if (threadIdx.x < 2 * nc) {
                double t = 0.0;
#pragma unroll
                for (int w = 0; w < RED_WARPS; w++) t += wred[w * 2 * NC + threadIdx.x];
                acc[((threadIdx.x >> 1) * l + k) * 2 + (threadIdx.x & 1)] += t;
            }
            __syncthreads();
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * nc * l; i += blockDim.x) {
        const int k = (i >> 1) % l;
        if (k >= kb && k < ke) partial[(long long)i * gridDim.x + blockIdx.x] = acc[i];
    }
}

// out[i] = sum_b partial[i][b]; one block per i
__global__ void reduce_partials_kernel(double* __restrict__ out, const double* __restrict__ partial, int nblocks) {
    __shared__ double sm[RED_WARPS];
    const int i = blockIdx.x;
    double t = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) t += partial[(long long)i * nblocks + b];
    t = warp_sum(t);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double r = 0.0;
#pragma unroll
        for (int w = 0; w < RED_WARPS; w++) r += sm[w];
        out[i] = r;
    }
}

// ------------------------------------------------------------------------------------------- block axpy
// MODE 0: y <- y + sum_k a_k v_k
// MODE 1: y <- pa * eta + pb * gamma5 ( y + sum_k a_k v_k )       (D_N assembly, eq. 2.4 + 2.11: pa = pb = 1/abar;
//                                                                   massive operator: pa = 1/abar + m/2, pb = 1/abar - m/2)
template <typename T, int MODE>
__global__ void __launch_bounds__(RED_THREADS) block_axpy_kernel(typename Prec<T>::Vec* y, int l, const double* __restrict__ coef,
                                                                 const typename Prec<T>::Vec* __restrict__ v,
                                                                 const typename Prec<T>::Vec* eta, T pa, T pb, long long V) {
    extern __shared__ double sm[];   // [2l]
    for (int i = threadIdx.x; i < 2 * l; i += blockDim.x) sm[i] = coef[i];
    __syncthreads();
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < V; s += (long long)gridDim.x * blockDim.x) {
        cx<T> c[12];
        load_site<T>(y, V, s, c);
        for (int k = 0; k < l; k++) {
            cx<T> b[12];
            load_site<T>(v + (long long)k * Prec<T>::NV * V, V, s, b);
            const cx<T> a = {(T)sm[2 * k], (T)sm[2 * k + 1]};
#pragma unroll
            for (int i = 0; i < 12; i++) cfma(c[i], a, b[i]);
        }
        if (MODE == 1) {
            cx<T> e[12];
            load_site<T>(eta, V, s, e);
#pragma unroll
            for (int i = 0; i < 12; i++) {
                const T sg = (i < 6) ? T(1) : T(-1);
                c[i] = {fma(pa, e[i].re, pb * sg * c[i].re), fma(pa, e[i].im, pb * sg * c[i].im)};
            }
        }
        store_site<T>(y, V, s, c);
    }
}

// the same for NB right-hand sides at once (nd_apply_DN_multi): y_j, eta_j are batches (stride = one spinor), coef[(j*l + k)*2];
// the block v is streamed once for all of them
template <typename T, int NB, int MODE>
__global__ void __launch_bounds__(RED_THREADS) block_axpy_batch_kernel(typename Prec<T>::Vec* y, int l, int nb, const double* __restrict__ coef,
                                                                       const typename Prec<T>::Vec* __restrict__ v,
                                                                       const typename Prec<T>::Vec* eta, T pa, T pb, long long V) {
    extern __shared__ double sm[];   // [nb][2l]
    for (int i = threadIdx.x; i < 2 * l * nb; i += blockDim.x) sm[i] = coef[i];
    __syncthreads();
    const long long bs = (long long)Prec<T>::NV * V;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < V; s += (long long)gridDim.x * blockDim.x) {
        cx<T> c[NB][12];
#pragma unroll
        for (int j = 0; j < NB; j++)
            if (j < nb) load_site<T>(y + j * bs, V, s, c[j]);
        for (int k = 0; k < l; k++) {
            cx<T> b[12];
            load_site<T>(v + (long long)k * bs, V, s, b);
#pragma unroll
            for (int j = 0; j < NB; j++)
                if (j < nb) {
                    const cx<T> a = {(T)sm[(j * l + k) * 2], (T)sm[(j * l + k) * 2 + 1]};
#pragma unroll
                    for (int i = 0; i < 12; i++) cfma(c[j][i], a, b[i]);
                }
        }
#pragma unroll
        for (int j = 0; j < NB; j++)
            if (j < nb) {
                if (MODE == 1) {
                    cx<T> e[12];
                    load_site<T>(eta + j * bs, V, s, e);
#pragma unroll
                    for (int i = 0; i < 12; i++) {
                        const T sg = (i < 6) ? T(1) : T(-1);
                        c[j][i] = {fma(pa, e[i].re, pb * sg * c[j][i].re), fma(pa, e[i].im, pb * sg * c[j][i].im)};
                    }
                }
                store_site<T>(y + j * bs, V, s, c[j]);
            }
    }
}

// ------------------------------------------------------------------------------------------- block rotation
// The eigen-solver needs X C for blocks of k vectors (lowmodes.cu): NG output columns at a time, so X is streamed k/NG times.
// rotate: y_j = sum_{i < l} coef[j*l + i] v_i for j < ng <= NG output columns (y_j at y + j*NV*V), one pass over v
template <typename T, int NG>
__global__ void __launch_bounds__(RED_THREADS) block_rotate_kernel(typename Prec<T>::Vec* __restrict__ y, int l, int ng,
                                                                   const double* __restrict__ coef,
                                                                   const typename Prec<T>::Vec* __restrict__ v, long long V) {
    extern __shared__ double sm[];   // [NG][2l]
    for (int i = threadIdx.x; i < 2 * l * ng; i += blockDim.x) sm[i] = coef[i];
    __syncthreads();
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < V; s += (long long)gridDim.x * blockDim.x) {
        cx<T> acc[NG][12];
#pragma unroll
        for (int j = 0; j < NG; j++)
#pragma unroll
            for (int i = 0; i < 12; i++) acc[j][i] = {T(0), T(0)};
        for (int k = 0; k < l; k++) {
            cx<T> b[12];
            load_site<T>(v + (long long)k * Prec<T>::NV * V, V, s, b);
#pragma unroll
            for (int j = 0; j < NG; j++) {
                if (j < ng) {
                    const cx<T> a = {(T)sm[(j * l + k) * 2], (T)sm[(j * l + k) * 2 + 1]};
#pragma unroll
                    for (int i = 0; i < 12; i++) cfma(acc[j][i], a, b[i]);
                }
            }
        }
#pragma unroll
        for (int j = 0; j < NG; j++)
            if (j < ng) store_site<T>(y + (long long)j * Prec<T>::NV * V, V, s, acc[j]);
    }
}

// ---------------------------------------------------------------------------------------- block residual
// partial[j][block] = sum over the block's sites of |y_j - nu_j x_j|^2   (blockIdx.y = j): the residues of eq. 2.8 for a
// whole block of Ritz pairs in one launch (differences formed in fp64)
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) block_resid_kernel(double* __restrict__ partial, const double* __restrict__ nu,
                                                                  const typename Prec<T>::Vec* __restrict__ x,
                                                                  const typename Prec<T>::Vec* __restrict__ y, long long V) {
    __shared__ double sm[RED_WARPS];
    const int j = blockIdx.y;
    const double nj = nu[j];
    const typename Prec<T>::Vec* xj = x + (long long)j * Prec<T>::NV * V;
    const typename Prec<T>::Vec* yj = y + (long long)j * Prec<T>::NV * V;
    double acc = 0.0;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < V; s += (long long)gridDim.x * blockDim.x) {
        cx<T> a[12], b[12];
        load_site<T>(xj, V, s, a);
        load_site<T>(yj, V, s, b);
#pragma unroll
        for (int i = 0; i < 12; i++) {
            const double dr = (double)b[i].re - nj * (double)a[i].re, di = (double)b[i].im - nj * (double)a[i].im;
            acc = fma(dr, dr, acc);
            acc = fma(di, di, acc);
        }
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < RED_WARPS; w++) t += sm[w];
        partial[(long long)j * gridDim.x + blockIdx.x] = t;
    }
}

// --------------------------------------------------------------------------------------------- gaussian
__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1,
                                              unsigned (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const unsigned n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
// word index w -> 4 (fp32) or 2 (fp64) standard normals by Box-Muller
template <typename T>
__global__ void gaussian_kernel(typename Prec<T>::Vec* __restrict__ x, unsigned long long seed, long long nwords, unsigned shard) {
    for (long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x; w < nwords; w += (long long)gridDim.x * blockDim.x) {
        unsigned r[4];
        philox4x32_10((unsigned)w, (unsigned)(w >> 32), shard, 0u, (unsigned)seed, (unsigned)(seed >> 32), r);   // counter = (word, shard rank)
        typename Prec<T>::Vec o;
        T* po = reinterpret_cast<T*>(&o);
        if (sizeof(T) == 4) {
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const float u1 = ((float)(r[2 * h] >> 8) + 0.5f) * (1.0f / 16777216.0f);
                const float u2 = ((float)(r[2 * h + 1] >> 8) + 0.5f) * (1.0f / 16777216.0f);
                const float rad = sqrtf(-2.0f * logf(u1));
                float sn, cs;
                sincospif(2.0f * u2, &sn, &cs);
                po[2 * h] = (T)(rad * cs);
                po[2 * h + 1] = (T)(rad * sn);
            }
        } else {
            const double u1 = ((double)(((unsigned long long)r[0] << 21) ^ (r[1] >> 11)) + 0.5) * (1.0 / 9007199254740992.0);
            const double u2 = ((double)(((unsigned long long)r[2] << 21) ^ (r[3] >> 11)) + 0.5) * (1.0 / 9007199254740992.0);
            const double rad = sqrt(-2.0 * log(u1));
            double sn, cs;
            sincospi(2.0 * u2, &sn, &cs);
            po[0] = (T)(rad * cs);
            po[1] = (T)(rad * sn);
        }
        x[w] = o;
    }
}

inline unsigned grid_for(long long n, int threads, int cap = ND_MAX_RED_BLOCKS) {
    long long b = (n + threads - 1) / threads;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (unsigned)b;
}

// <v_k, x_c>, k < l, for nc columns (pointers) -> d_out[(c*l + k)*2 + {re, im}] (device), NC columns per pass over the block
template <typename T>
int block_dot_cols_t(nd_ctx* ctx, int l, const void* v, int nc, const void* const* cols, double* d_out) {
    using Vec = typename Prec<T>::Vec;
    // staged columns: NC * 24 reals * DOT_RANGE sites of shared memory (fp32: 24 KB, fp64: 48 KB per column)
    constexpr int NCMAX = sizeof(T) == 4 ? 4 : 2;
    auto smem_for = [](int NC, int ll) {
        return (size_t)NC * Prec<T>::NV * DOT_RANGE * sizeof(Vec) + ((size_t)2 * NC * ll + (size_t)RED_WARPS * 2 * NC) * sizeof(double);
    };
    if (!ctx->dot_configured) {   // once per context (both precisions' instantiations are cheap to configure)
        ND_CUDA(ctx, cudaFuncSetAttribute(block_dot_cols_kernel<T, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_for(1, ND_MAX_BLOCK_L)));
        ND_CUDA(ctx, cudaFuncSetAttribute(block_dot_cols_kernel<T, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_for(2, ND_MAX_BLOCK_L)));
        ND_CUDA(ctx, cudaFuncSetAttribute(block_dot_cols_kernel<T, NCMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_for(NCMAX, ND_MAX_BLOCK_L)));
        ctx->dot_configured = true;
    }
    const long long nranges = (ctx->V + DOT_RANGE - 1) / DOT_RANGE;
    for (int c0 = 0; c0 < nc; c0 += NCMAX) {
        const int n = nc - c0 < NCMAX ? nc - c0 : NCMAX;
        ColPtrs cp;
        for (int i = 0; i < 8; i++) cp.p[i] = (i < n) ? cols[c0 + i] : nullptr;
        // the partial-sum scratch holds ND_RESULT_DOUBLES x ND_MAX_RED_BLOCKS doubles: rows (2 l n) x CTAs must fit
        long long cap = (long long)ND_RESULT_DOUBLES * ND_MAX_RED_BLOCKS / ((long long)2 * l * n);
        if (cap > 8LL * ctx->num_sms) cap = 8LL * ctx->num_sms;
        const unsigned blocks = (unsigned)(nranges < cap ? nranges : cap);
        // few ranges (small lattice) and many vectors: split the vectors over grid.y until there are ~4 CTAs per SM
        int nkc = 1;
        while ((long long)blocks * nkc < 4LL * ctx->num_sms && (l + nkc) / (nkc + 1) >= 2) nkc++;
        const dim3 grid(blocks, (unsigned)nkc, 1);
        if (n == 1) block_dot_cols_kernel<T, 1><<<grid, RED_THREADS, smem_for(1, l), ctx->stream>>>(ctx->d_partial, l, n, (const Vec*)v, cp, ctx->V);
        else if (n == 2) block_dot_cols_kernel<T, 2><<<grid, RED_THREADS, smem_for(2, l), ctx->stream>>>(ctx->d_partial, l, n, (const Vec*)v, cp, ctx->V);
        else block_dot_cols_kernel<T, NCMAX><<<grid, RED_THREADS, smem_for(NCMAX, l), ctx->stream>>>(ctx->d_partial, l, n, (const Vec*)v, cp, ctx->V);
        ND_LAUNCHED(ctx);
        reduce_partials_kernel<<<n * l * 2, RED_THREADS, 0, ctx->stream>>>(d_out + (size_t)2 * l * c0, ctx->d_partial, (int)blocks);
        ND_LAUNCHED(ctx);
    }
    return ndi_allreduce(ctx, d_out, 2 * l * nc);   // domain decomposition: the local sums become global ones
}

}  // namespace

// ------------------------------------------------------------------------------------ internal entry points
int ndi_read_result(nd_ctx* ctx, const double* d_src, double* h_dst, int n) {
    ND_CUDA(ctx, cudaMemcpyAsync(ctx->h_result, d_src, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < n; i++) h_dst[i] = ctx->h_result[i];
    return ND_OK;
}

int ndi_block_dot_cols_dev(nd_ctx* ctx, int l, const void* v, int nc, const void* const* cols, double* d_out) {
    return (ctx->prec == 32) ? block_dot_cols_t<float>(ctx, l, v, nc, cols, d_out) : block_dot_cols_t<double>(ctx, l, v, nc, cols, d_out);
}
int ndi_block_dot_dev(nd_ctx* ctx, int l, const void* v, const void* x, double* d_out) {
    const void* cols[1] = {x};
    return ndi_block_dot_cols_dev(ctx, l, v, 1, cols, d_out);
}
int ndi_block_dot2_dev(nd_ctx* ctx, int l, const void* v, const void* x0, const void* x1, double* d_out) {
    const void* cols[2] = {x0, x1};
    return ndi_block_dot_cols_dev(ctx, l, v, 2, cols, d_out);
}
// y <- y + sum_k coef_k v_k (mode 0) or the D_N assembly (mode 1); coef on the device
int ndi_block_axpy_dev(nd_ctx* ctx, int l, const double* d_coef, const void* v, void* y, int mode, const void* eta, double pa,
                       double pb) {
    const unsigned blocks = grid_for(ctx->V, RED_THREADS, 1 << 30);
    const size_t smem = (size_t)2 * (l > 0 ? l : 1) * sizeof(double);
    if (ctx->prec == 32) {
        using Vec = float4;
        if (mode == 0) block_axpy_kernel<float, 0><<<blocks, RED_THREADS, smem, ctx->stream>>>((Vec*)y, l, d_coef, (const Vec*)v, nullptr, 0.f, 0.f, ctx->V);
        else block_axpy_kernel<float, 1><<<blocks, RED_THREADS, smem, ctx->stream>>>((Vec*)y, l, d_coef, (const Vec*)v, (const Vec*)eta, (float)pa, (float)pb, ctx->V);
    } else {
        using Vec = double2;
        if (mode == 0) block_axpy_kernel<double, 0><<<blocks, RED_THREADS, smem, ctx->stream>>>((Vec*)y, l, d_coef, (const Vec*)v, nullptr, 0.0, 0.0, ctx->V);
        else block_axpy_kernel<double, 1><<<blocks, RED_THREADS, smem, ctx->stream>>>((Vec*)y, l, d_coef, (const Vec*)v, (const Vec*)eta, pa, pb, ctx->V);
    }
    ND_LAUNCHED(ctx);
    return ND_OK;
}

// rho_j = ||y_j - nu_j x_j||, j < k (host nu in, host rho out; synchronises)
int ndi_block_resid(nd_ctx* ctx, int k, const void* x, const void* y, const double* nu, double* rho) {
    ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < k; i++) ctx->h_result[i] = nu[i];
    ND_CUDA(ctx, cudaMemcpyAsync(ctx->d_coef, ctx->h_result, (size_t)k * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    long long bx = (ctx->V + 8 * RED_THREADS - 1) / (8 * RED_THREADS);
    if (bx > ctx->num_sms) bx = ctx->num_sms;
    const dim3 grid((unsigned)bx, (unsigned)k, 1);
    if (ctx->prec == 32) block_resid_kernel<float><<<grid, RED_THREADS, 0, ctx->stream>>>(ctx->d_partial, ctx->d_coef, (const float4*)x, (const float4*)y, ctx->V);
    else block_resid_kernel<double><<<grid, RED_THREADS, 0, ctx->stream>>>(ctx->d_partial, ctx->d_coef, (const double2*)x, (const double2*)y, ctx->V);
    ND_LAUNCHED(ctx);
    reduce_partials_kernel<<<k, RED_THREADS, 0, ctx->stream>>>(ctx->d_result, ctx->d_partial, (int)bx);
    ND_LAUNCHED(ctx);
    int rc = ndi_allreduce(ctx, ctx->d_result, k);
    if (rc == ND_OK) rc = ndi_read_result(ctx, ctx->d_result, rho, k);
    for (int i = 0; i < k && rc == ND_OK; i++) rho[i] = sqrt(rho[i] > 0.0 ? rho[i] : 0.0);
    return rc;
}

// G[k][j] = <v_k, x_j>, k < l, j < nx, into d_out[(j*l + k)*2 + {re, im}] (device); x_j at x + j*spinor_bytes
int ndi_block_gram_dev(nd_ctx* ctx, int l, const void* v, int nx, const void* x, double* d_out) {
    const size_t sb = nd_spinor_bytes(ctx);
    std::vector<const void*> cols(nx);
    for (int j = 0; j < nx; j++) cols[j] = (const char*)x + (size_t)j * sb;
    return ndi_block_dot_cols_dev(ctx, l, v, nx, cols.data(), d_out);
}
// batched block axpy (nb right-hand sides, coef[(j*l + k)*2] on the device); mode as ndi_block_axpy_dev
int ndi_block_axpy_batch_dev(nd_ctx* ctx, int l, int nb, const double* d_coef, const void* v, void* y, int mode, const void* eta,
                             double pa, double pb) {
    const size_t sb = nd_spinor_bytes(ctx);
    const int NB = ctx->prec == 32 ? 4 : 2;
    const unsigned blocks = grid_for(ctx->V, RED_THREADS, 1 << 30);
    for (int j0 = 0; j0 < nb; j0 += NB) {
        const int n = nb - j0 < NB ? nb - j0 : NB;
        char* yj = (char*)y + (size_t)j0 * sb;
        const char* ej = eta ? (const char*)eta + (size_t)j0 * sb : nullptr;
        const double* cj = d_coef + (size_t)2 * l * j0;
        const size_t smem = (size_t)2 * (l > 0 ? l : 1) * n * sizeof(double);
        if (ctx->prec == 32) {
            if (mode == 0) block_axpy_batch_kernel<float, 4, 0><<<blocks, RED_THREADS, smem, ctx->stream>>>((float4*)yj, l, n, cj, (const float4*)v, nullptr, 0.f, 0.f, ctx->V);
            else block_axpy_batch_kernel<float, 4, 1><<<blocks, RED_THREADS, smem, ctx->stream>>>((float4*)yj, l, n, cj, (const float4*)v, (const float4*)ej, (float)pa, (float)pb, ctx->V);
        } else {
            if (mode == 0) block_axpy_batch_kernel<double, 2, 0><<<blocks, RED_THREADS, smem, ctx->stream>>>((double2*)yj, l, n, cj, (const double2*)v, nullptr, 0.0, 0.0, ctx->V);
            else block_axpy_batch_kernel<double, 2, 1><<<blocks, RED_THREADS, smem, ctx->stream>>>((double2*)yj, l, n, cj, (const double2*)v, (const double2*)ej, pa, pb, ctx->V);
        }
        ND_LAUNCHED(ctx);
    }
    return ND_OK;
}
// y_j = sum_i coef[j*l + i] v_i for j < ny (coef: ny*l complex doubles on the device, y_j at y + j*spinor_bytes)
int ndi_block_rotate_dev(nd_ctx* ctx, int l, const double* d_coef, const void* v, int ny, void* y) {
    const size_t sb = nd_spinor_bytes(ctx);
    const int NG = ctx->prec == 32 ? 4 : 2;
    const unsigned blocks = grid_for(ctx->V, RED_THREADS, 1 << 30);
    for (int j0 = 0; j0 < ny; j0 += NG) {
        const int ng = ny - j0 < NG ? ny - j0 : NG;
        char* yj = (char*)y + (size_t)j0 * sb;
        const size_t smem = (size_t)2 * l * ng * sizeof(double);
        if (ctx->prec == 32) block_rotate_kernel<float, 4><<<blocks, RED_THREADS, smem, ctx->stream>>>((float4*)yj, l, ng, d_coef + (size_t)2 * l * j0, (const float4*)v, ctx->V);
        else block_rotate_kernel<double, 2><<<blocks, RED_THREADS, smem, ctx->stream>>>((double2*)yj, l, ng, d_coef + (size_t)2 * l * j0, (const double2*)v, ctx->V);
        ND_LAUNCHED(ctx);
    }
    return ND_OK;
}

// ------------------------------------------------------------------------------------------------ C ABI
#define ND_ENTER(ctx)                                   \
    if (!(ctx)) return ND_ERR_BAD_ARG;                  \
    ND_CUDA(ctx, cudaSetDevice((ctx)->device))

extern "C" int nd_axpy(nd_ctx* ctx, const double a[2], const void* x, void* y) {
    ND_ENTER(ctx);
    if (!a || !x || !y) return nd_fail(ctx, ND_ERR_BAD_ARG, "axpy: null argument");
    const unsigned blocks = grid_for(ctx->V, 128, 1 << 30);
    if (ctx->prec == 32) axpy_kernel<float><<<blocks, 128, 0, ctx->stream>>>((float4*)y, (const float4*)x, (float)a[0], (float)a[1], ctx->V);
    else axpy_kernel<double><<<blocks, 128, 0, ctx->stream>>>((double2*)y, (const double2*)x, a[0], a[1], ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
extern "C" int nd_scale(nd_ctx* ctx, const double a[2], void* x) {
    ND_ENTER(ctx);
    if (!a || !x) return nd_fail(ctx, ND_ERR_BAD_ARG, "scale: null argument");
    const unsigned blocks = grid_for(ctx->V, 128, 1 << 30);
    if (ctx->prec == 32) scale_kernel<float><<<blocks, 128, 0, ctx->stream>>>((float4*)x, (float)a[0], (float)a[1], ctx->V);
    else scale_kernel<double><<<blocks, 128, 0, ctx->stream>>>((double2*)x, a[0], a[1], ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
extern "C" int nd_copy(nd_ctx* ctx, void* y, const void* x) {
    ND_ENTER(ctx);
    if (!x || !y) return nd_fail(ctx, ND_ERR_BAD_ARG, "copy: null argument");
    ND_CUDA(ctx, cudaMemcpyAsync(y, x, nd_spinor_bytes(ctx), cudaMemcpyDeviceToDevice, ctx->stream));
    return ND_OK;
}
extern "C" int nd_gamma5(nd_ctx* ctx, void* y, const void* x) {
    ND_ENTER(ctx);
    if (!x || !y) return nd_fail(ctx, ND_ERR_BAD_ARG, "gamma5: null argument");
    const unsigned blocks = grid_for(ctx->V, 128, 1 << 30);
    if (ctx->prec == 32) gamma5_kernel<float><<<blocks, 128, 0, ctx->stream>>>((float4*)y, (const float4*)x, ctx->V);
    else gamma5_kernel<double><<<blocks, 128, 0, ctx->stream>>>((double2*)y, (const double2*)x, ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
int ndi_chiral_combine(nd_ctx* ctx, int sigma, void* y, const void* u, double c) {
    const unsigned blocks = (unsigned)std::min<long long>((ctx->V + 127) / 128, 8LL * ctx->num_sms);
    if (ctx->prec == 32) chiral_combine_kernel<float><<<blocks, 128, 0, ctx->stream>>>((float4*)y, (const float4*)u, sigma, (float)c, ctx->V);
    else chiral_combine_kernel<double><<<blocks, 128, 0, ctx->stream>>>((double2*)y, (const double2*)u, sigma, c, ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

extern "C" int nd_block_dot(nd_ctx* ctx, int l, const void* v, const void* x, double* out2l) {
    ND_ENTER(ctx);
    if (l < 1 || l > ND_MAX_BLOCK_L || !v || !x || !out2l) return nd_fail(ctx, ND_ERR_BAD_ARG, "block_dot: bad argument (1 <= l <= %d)", ND_MAX_BLOCK_L);
    int rc = ndi_block_dot_dev(ctx, l, v, x, ctx->d_result);
    if (rc != ND_OK) return rc;
    return ndi_read_result(ctx, ctx->d_result, out2l, 2 * l);
}
extern "C" int nd_dot(nd_ctx* ctx, const void* x, const void* y, double out[2]) { return nd_block_dot(ctx, 1, x, y, out); }
// results left in the caller's DEVICE memory, no synchronisation (SURVEY 8(b) `_dev` variants)
extern "C" int nd_block_dot_dev(nd_ctx* ctx, int l, const void* v, const void* x, double* d_out2l) {
    ND_ENTER(ctx);
    if (l < 1 || l > ND_MAX_BLOCK_L || !v || !x || !d_out2l) return nd_fail(ctx, ND_ERR_BAD_ARG, "block_dot_dev: bad argument (1 <= l <= %d)", ND_MAX_BLOCK_L);
    return ndi_block_dot_dev(ctx, l, v, x, d_out2l);
}
extern "C" int nd_dot_dev(nd_ctx* ctx, const void* x, const void* y, double* d_out2) { return nd_block_dot_dev(ctx, 1, x, y, d_out2); }
extern "C" int nd_norm2_dev(nd_ctx* ctx, const void* x, double* d_out2) { return nd_block_dot_dev(ctx, 1, x, x, d_out2); }

extern "C" int nd_norm2(nd_ctx* ctx, const void* x, double* out) {
    double t[2];
    int rc = nd_block_dot(ctx, 1, x, x, t);
    if (rc == ND_OK && out) *out = t[0];
    return rc;
}
extern "C" int nd_block_axpy(nd_ctx* ctx, int l, const double* a2l, const void* v, void* y) {
    ND_ENTER(ctx);
    if (l < 1 || l > ND_MAX_BLOCK_L || !a2l || !v || !y) return nd_fail(ctx, ND_ERR_BAD_ARG, "block_axpy: bad argument (1 <= l <= %d)", ND_MAX_BLOCK_L);
    // stage through the pinned buffer so the async copy is well defined, then order it on the stream
    ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < 2 * l; i++) ctx->h_result[i] = a2l[i];
    ND_CUDA(ctx, cudaMemcpyAsync(ctx->d_coef, ctx->h_result, (size_t)2 * l * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    return ndi_block_axpy_dev(ctx, l, ctx->d_coef, v, y, 0, nullptr, 0.0, 0.0);
}
extern "C" int nd_block_axpy_dev(nd_ctx* ctx, int l, const double* d_a2l, const void* v, void* y) {
    ND_ENTER(ctx);
    if (l < 1 || l > ND_MAX_BLOCK_L || !d_a2l || !v || !y) return nd_fail(ctx, ND_ERR_BAD_ARG, "block_axpy_dev: bad argument (1 <= l <= %d)", ND_MAX_BLOCK_L);
    return ndi_block_axpy_dev(ctx, l, d_a2l, v, y, 0, nullptr, 0.0, 0.0);
}
extern "C" int nd_gaussian(nd_ctx* ctx, void* x, unsigned long long seed) {
    ND_ENTER(ctx);
    if (!x) return nd_fail(ctx, ND_ERR_BAD_ARG, "gaussian: null argument");
    const long long nwords = ctx->V * (ctx->prec == 32 ? 6 : 12);
    const unsigned blocks = grid_for(nwords, 256, 1 << 30);
    if (ctx->prec == 32) gaussian_kernel<float><<<blocks, 256, 0, ctx->stream>>>((float4*)x, seed, nwords, (unsigned)ctx->shard_rank);
    else gaussian_kernel<double><<<blocks, 256, 0, ctx->stream>>>((double2*)x, seed, nwords, (unsigned)ctx->shard_rank);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
