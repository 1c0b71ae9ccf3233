// blas.cu - BLAS-1 on spinor fields (BASELINE.json north_star; implied by PAPER.md:L66,L79) and the low-mode
// projection kernels  w_k = <u_k, x>  and  y <- y + sum_k a_k u_k  (eq. 2.7 / 2.11).
// All reductions accumulate in fp64 (both precisions): thread partials -> warp shuffle -> per-warp shared row ->
// per-block partial -> second-stage kernel.  No atomics: results are bitwise reproducible run to run.
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

// --------------------------------------------------------------------------------------- block dot product
// partial[(j*l + k)*2 + {0,1}][block] = sum over this block's sites of conj(v_k) x_j ,  j < NX
template <typename T, int NX>
__global__ void __launch_bounds__(RED_THREADS) block_dot_kernel(double* __restrict__ partial, int l,
                                                                const typename Prec<T>::Vec* __restrict__ v,
                                                                const typename Prec<T>::Vec* __restrict__ x0,
                                                                const typename Prec<T>::Vec* __restrict__ x1, long long V) {
    extern __shared__ double sm[];   // [RED_WARPS][NX*l*2]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int row = NX * l * 2;
    for (int i = threadIdx.x; i < RED_WARPS * row; i += blockDim.x) sm[i] = 0.0;
    __syncthreads();
    const long long nchunks = (V + blockDim.x - 1) / blockDim.x;
    for (long long ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
        const long long s = ch * blockDim.x + threadIdx.x;
        const bool valid = s < V;
        const long long sc = valid ? s : V - 1;
        cx<T> a[NX][12];
        load_site<T>(x0, V, sc, a[0]);
        if (NX > 1) load_site<T>(x1, V, sc, a[NX - 1]);
        if (!valid) {
#pragma unroll
            for (int j = 0; j < NX; j++)
#pragma unroll
                for (int i = 0; i < 12; i++) a[j][i] = {T(0), T(0)};
        }
        for (int k = 0; k < l; k++) {
            cx<T> b[12];
            load_site<T>(v + (long long)k * Prec<T>::NV * V, V, sc, b);
#pragma unroll
            for (int j = 0; j < NX; j++) {
                double re = 0.0, im = 0.0;
#pragma unroll
                for (int i = 0; i < 12; i++) {
                    // conj(b) * a, products in T (exact in fp64 for fp32 inputs would need widening: widen)
                    const double br = (double)b[i].re, bi = (double)b[i].im, xr = (double)a[j][i].re, xi = (double)a[j][i].im;
                    re = fma(br, xr, re);
                    re = fma(bi, xi, re);
                    im = fma(br, xi, im);
                    im = fma(-bi, xr, im);
                }
                re = warp_sum(re);
                im = warp_sum(im);
                if (lane == 0) {
                    sm[warp * row + (j * l + k) * 2] += re;
                    sm[warp * row + (j * l + k) * 2 + 1] += im;
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < row; i += blockDim.x) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < RED_WARPS; w++) t += sm[w * row + i];
        partial[(long long)i * gridDim.x + blockIdx.x] = t;
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

// ----------------------------------------------------------------------------------- grouped Gram / rotation
// The eigen-solver needs X^dagger Y and X C for blocks of k vectors (lowmodes.cu).  Column by column (block_dot /
// block_axpy) the block X is re-read k times.  These two kernels take NG columns at a time, so X is streamed k/NG times.
//
// gram: partial[((j*l + k)*2 + c)][block] = sum over the block's sites of conj(v_k) x_j, j < ng <= NG.  The loop over
// k is OUTSIDE the loop over the CTA's sites: the NG x-columns of those sites are re-read from L1/L2, v_k is streamed
// once, and the accumulators of one k fit in registers, so there is one warp reduction per k and not one per chunk.
template <typename T, int NG>
__global__ void __launch_bounds__(RED_THREADS) block_gram_kernel(double* __restrict__ partial, int l, int ng,
                                                                 const typename Prec<T>::Vec* __restrict__ v,
                                                                 const typename Prec<T>::Vec* __restrict__ x, long long V) {
    __shared__ double sm[RED_WARPS][2 * NG];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long nchunks = (V + blockDim.x - 1) / blockDim.x;
    for (int k = 0; k < l; k++) {
        double re[NG], im[NG];
#pragma unroll
        for (int j = 0; j < NG; j++) re[j] = im[j] = 0.0;
        const typename Prec<T>::Vec* vk = v + (long long)k * Prec<T>::NV * V;
        for (long long ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
            const long long s = ch * blockDim.x + threadIdx.x;
            if (s >= V) continue;
            cx<T> b[12];
            load_site<T>(vk, V, s, b);
#pragma unroll
            for (int j = 0; j < NG; j++) {
                if (j < ng) {
                    cx<T> a[12];
                    load_site<T>(x + (long long)j * Prec<T>::NV * V, V, s, a);
#pragma unroll
                    for (int i = 0; i < 12; i++) {
                        const double br = (double)b[i].re, bi = (double)b[i].im, xr = (double)a[i].re, xi = (double)a[i].im;
                        re[j] = fma(br, xr, re[j]);
                        re[j] = fma(bi, xi, re[j]);
                        im[j] = fma(br, xi, im[j]);
                        im[j] = fma(-bi, xr, im[j]);
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < NG; j++) {
            re[j] = warp_sum(re[j]);
            im[j] = warp_sum(im[j]);
            if (lane == 0) { sm[warp][2 * j] = re[j]; sm[warp][2 * j + 1] = im[j]; }
        }
        __syncthreads();
        if (threadIdx.x < 2 * ng) {
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < RED_WARPS; w++) t += sm[w][threadIdx.x];
            const int j = threadIdx.x >> 1, c = threadIdx.x & 1;
            partial[((long long)(j * l + k) * 2 + c) * gridDim.x + blockIdx.x] = t;
        }
        __syncthreads();
    }
}

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
__global__ void gaussian_kernel(typename Prec<T>::Vec* __restrict__ x, unsigned long long seed, long long nwords) {
    for (long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x; w < nwords; w += (long long)gridDim.x * blockDim.x) {
        unsigned r[4];
        philox4x32_10((unsigned)w, (unsigned)(w >> 32), 0u, 0u, (unsigned)seed, (unsigned)(seed >> 32), r);
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

template <typename T>
int block_dot_t(nd_ctx* ctx, int l, int nx, const void* v, const void* x0, const void* x1, double* d_out) {
    using Vec = typename Prec<T>::Vec;
    const unsigned blocks = grid_for(ctx->V, RED_THREADS);
    const size_t smem = (size_t)RED_WARPS * nx * l * 2 * sizeof(double);
    if (nx == 1)
        block_dot_kernel<T, 1><<<blocks, RED_THREADS, smem, ctx->stream>>>(ctx->d_partial, l, (const Vec*)v, (const Vec*)x0, nullptr, ctx->V);
    else
        block_dot_kernel<T, 2><<<blocks, RED_THREADS, smem, ctx->stream>>>(ctx->d_partial, l, (const Vec*)v, (const Vec*)x0, (const Vec*)x1, ctx->V);
    ND_LAUNCHED(ctx);
    reduce_partials_kernel<<<nx * l * 2, RED_THREADS, 0, ctx->stream>>>(d_out, ctx->d_partial, (int)blocks);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------ internal entry points
int ndi_read_result(nd_ctx* ctx, const double* d_src, double* h_dst, int n) {
    ND_CUDA(ctx, cudaMemcpyAsync(ctx->h_result, d_src, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < n; i++) h_dst[i] = ctx->h_result[i];
    return ND_OK;
}

int ndi_block_dot_dev(nd_ctx* ctx, int l, const void* v, const void* x, double* d_out) {
    return (ctx->prec == 32) ? block_dot_t<float>(ctx, l, 1, v, x, nullptr, d_out) : block_dot_t<double>(ctx, l, 1, v, x, nullptr, d_out);
}
int ndi_block_dot2_dev(nd_ctx* ctx, int l, const void* v, const void* x0, const void* x1, double* d_out) {
    return (ctx->prec == 32) ? block_dot_t<float>(ctx, l, 2, v, x0, x1, d_out) : block_dot_t<double>(ctx, l, 2, v, x0, x1, d_out);
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
    int rc = ndi_read_result(ctx, ctx->d_result, rho, k);
    for (int i = 0; i < k && rc == ND_OK; i++) rho[i] = sqrt(rho[i] > 0.0 ? rho[i] : 0.0);
    return rc;
}

// G[k][j] = <v_k, x_j>, k < l, j < nx, into d_out[(j*l + k)*2 + {re, im}] (device); x_j at x + j*spinor_bytes
int ndi_block_gram_dev(nd_ctx* ctx, int l, const void* v, int nx, const void* x, double* d_out) {
    const size_t sb = nd_spinor_bytes(ctx);
    const int NG = ctx->prec == 32 ? 8 : 4;
    // the partial-sum scratch holds ND_RESULT_DOUBLES x ND_MAX_RED_BLOCKS doubles: rows (2 l NG) x blocks must fit
    long long cap = (long long)ND_RESULT_DOUBLES * ND_MAX_RED_BLOCKS / ((long long)2 * l * NG);
    if (cap > 4 * ctx->num_sms) cap = 4 * ctx->num_sms;
    const unsigned blocks = grid_for(ctx->V, RED_THREADS, (int)cap);
    for (int j0 = 0; j0 < nx; j0 += NG) {
        const int ng = nx - j0 < NG ? nx - j0 : NG;
        const char* xj = (const char*)x + (size_t)j0 * sb;
        if (ctx->prec == 32) block_gram_kernel<float, 8><<<blocks, RED_THREADS, 0, ctx->stream>>>(ctx->d_partial, l, ng, (const float4*)v, (const float4*)xj, ctx->V);
        else block_gram_kernel<double, 4><<<blocks, RED_THREADS, 0, ctx->stream>>>(ctx->d_partial, l, ng, (const double2*)v, (const double2*)xj, ctx->V);
        ND_LAUNCHED(ctx);
        reduce_partials_kernel<<<ng * l * 2, RED_THREADS, 0, ctx->stream>>>(d_out + (size_t)2 * l * j0, ctx->d_partial, (int)blocks);
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
extern "C" int nd_gaussian(nd_ctx* ctx, void* x, unsigned long long seed) {
    ND_ENTER(ctx);
    if (!x) return nd_fail(ctx, ND_ERR_BAD_ARG, "gaussian: null argument");
    const long long nwords = ctx->V * (ctx->prec == 32 ? 6 : 12);
    const unsigned blocks = grid_for(nwords, 256, 1 << 30);
    if (ctx->prec == 32) gaussian_kernel<float><<<blocks, 256, 0, ctx->stream>>>((float4*)x, seed, nwords);
    else gaussian_kernel<double><<<blocks, 256, 0, ctx->stream>>>((double2*)x, seed, nwords);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
