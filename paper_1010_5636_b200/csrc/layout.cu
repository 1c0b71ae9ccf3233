// layout.cu - canonical AoS <-> device plane-SoA reordering of spinors, and SU(3) link checking, compression to
// 18 / 12 / 8 reals and reordering (section 2.1, eq. 2.3; 8-parameter form DESIGN.md R8).
#include "nd_internal.cuh"
#include "nd_su3.cuh"

namespace {

// ------------------------------------------------------------------------------------------------- spinors
// thread = (site, plane): AoS reals [s][24] -> word (p, s)
template <typename T, typename Tin>
__global__ void pack_spinor_kernel(typename Prec<T>::Vec* __restrict__ soa, const Tin* __restrict__ aos, long long V) {
    constexpr int NV = Prec<T>::NV;
    constexpr int W = 24 / NV;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V * NV) return;
    int p = (int)(i / V);
    long long s = i - (long long)p * V;
    T r[W];
#pragma unroll
    for (int k = 0; k < W; k++) r[k] = (T)aos[s * 24 + p * W + k];
    typename Prec<T>::Vec w;
    T* wr = reinterpret_cast<T*>(&w);
#pragma unroll
    for (int k = 0; k < W; k++) wr[k] = r[k];
    soa[(long long)p * V + s] = w;
}

template <typename T, typename Tout>
__global__ void unpack_spinor_kernel(Tout* __restrict__ aos, const typename Prec<T>::Vec* __restrict__ soa, long long V) {
    constexpr int NV = Prec<T>::NV;
    constexpr int W = 24 / NV;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V * NV) return;
    int p = (int)(i / V);
    long long s = i - (long long)p * V;
    typename Prec<T>::Vec w = soa[(long long)p * V + s];
    const T* wr = reinterpret_cast<const T*>(&w);
#pragma unroll
    for (int k = 0; k < W; k++) aos[s * 24 + p * W + k] = (Tout)wr[k];
}

// device SoA of one precision -> device SoA of the other (mixed-precision solver): thread = site
template <typename Td, typename Ts>
__global__ void convert_spinor_kernel(typename Prec<Td>::Vec* __restrict__ dst, const typename Prec<Ts>::Vec* __restrict__ src, long long V) {
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= V) return;
    typename Prec<Ts>::Vec ws[Prec<Ts>::NV];
#pragma unroll
    for (int p = 0; p < Prec<Ts>::NV; p++) ws[p] = src[p * V + s];
    cx<Ts> cs[12];
    words_to_cx(ws, cs);
    cx<Td> cd[12];
#pragma unroll
    for (int i = 0; i < 12; i++) cd[i] = {(Td)cs[i].re, (Td)cs[i].im};
    typename Prec<Td>::Vec wd[Prec<Td>::NV];
    cx_to_words(cd, wd);
#pragma unroll
    for (int p = 0; p < Prec<Td>::NV; p++) dst[p * V + s] = wd[p];
}

// --------------------------------------------------------------------------------------------------- links
__device__ __forceinline__ void atomic_max_nonneg(double* addr, double v) {
    atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}
__device__ __forceinline__ void atomic_min_nonneg(double* addr, double v) {
    atomicMin(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

// thread = (mu, site).  stats[0] = max |U^dag U - 1|, stats[1] = max |det U - 1|, stats[2] = min N
template <typename T, int RECON, typename Tin>
__global__ void compress_gauge_kernel(typename LinkLayout<T, RECON>::LVec* __restrict__ g, const Tin* __restrict__ aos,
                                      long long V, double* stats) {
    using LL = LinkLayout<T, RECON>;
    constexpr int W = sizeof(typename LL::LVec) / sizeof(T);
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < 4 * V;
    if (!valid) i = 4 * V - 1;   // keep the whole warp alive for the shuffles below; the store is predicated
    int mu = (int)(i / V);
    long long s = i - (long long)mu * V;
    cx<double> U[3][3];
    const Tin* src = aos + i * 18;
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++) U[a][b] = {(double)src[2 * (3 * a + b)], (double)src[2 * (3 * a + b) + 1]};
    // checks in fp64 on the values as given
    double dev = 0.0;
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++) {
            cx<double> acc = {a == b ? -1.0 : 0.0, 0.0};
#pragma unroll
            for (int k = 0; k < 3; k++) cfma_cj(acc, U[k][a], U[k][b]);
            dev = fmax(dev, fmax(fabs(acc.re), fabs(acc.im)));
        }
    cx<double> det = U[0][0] * (U[1][1] * U[2][2] - U[1][2] * U[2][1]) - U[0][1] * (U[1][0] * U[2][2] - U[1][2] * U[2][0]) +
                     U[0][2] * (U[1][0] * U[2][1] - U[1][1] * U[2][0]);
    double ddev = fmax(fabs(det.re - 1.0), fabs(det.im));
    double N = U[0][1].re * U[0][1].re + U[0][1].im * U[0][1].im + U[0][2].re * U[0][2].re + U[0][2].im * U[0][2].im;
    // warp-level reduce before the atomics
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dev = fmax(dev, __shfl_xor_sync(0xffffffffu, dev, o));
        ddev = fmax(ddev, __shfl_xor_sync(0xffffffffu, ddev, o));
        N = fmin(N, __shfl_xor_sync(0xffffffffu, N, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomic_max_nonneg(stats + 0, dev);
        atomic_max_nonneg(stats + 1, ddev);
        atomic_min_nonneg(stats + 2, N);
    }
    T r[LL::NL * W];
    if (RECON == 18) {
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) { r[2 * (3 * a + b)] = (T)U[a][b].re; r[2 * (3 * a + b) + 1] = (T)U[a][b].im; }
    } else if (RECON == 12) {
#pragma unroll
        for (int a = 0; a < 2; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) { r[2 * (3 * a + b)] = (T)U[a][b].re; r[2 * (3 * a + b) + 1] = (T)U[a][b].im; }
    } else {
        r[0] = (T)U[0][1].re; r[1] = (T)U[0][1].im;
        r[2] = (T)U[0][2].re; r[3] = (T)U[0][2].im;
        r[4] = (T)U[1][0].re; r[5] = (T)U[1][0].im;
        // the two phases are stored as tan(theta/4) in [-1, 1]: rebuilt with one reciprocal, no sincos (nd_su3.cuh)
        r[6] = (T)tan(0.25 * atan2(U[0][0].im, U[0][0].re));
        r[7] = (T)tan(0.25 * atan2(U[2][0].im, U[2][0].re));
    }
    if (!valid) return;
    typename LL::LVec* dst = g + (long long)mu * LL::NL * V + s;
#pragma unroll
    for (int p = 0; p < LL::NL; p++) {
        typename LL::LVec w;
        T* wr = reinterpret_cast<T*>(&w);
#pragma unroll
        for (int k = 0; k < W; k++) wr[k] = r[p * W + k];
        dst[p * V] = w;
    }
}

template <typename T, int RECON>
__global__ void reconstruct_gauge_kernel(double* __restrict__ aos, const typename LinkLayout<T, RECON>::LVec* __restrict__ g,
                                         long long V) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 4 * V) return;
    int mu = (int)(i / V);
    long long s = i - (long long)mu * V;
    cx<T> U[3][3];
    load_link<T, RECON>(g, V, mu, s, U);
    double* dst = aos + i * 18;
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++) { dst[2 * (3 * a + b)] = (double)U[a][b].re; dst[2 * (3 * a + b) + 1] = (double)U[a][b].im; }
}

template <typename T, int RECON>
int set_gauge_t(nd_ctx* ctx, const void* d_aos, int src_prec, double* d_stats) {
    using LVec = typename LinkLayout<T, RECON>::LVec;
    const int threads = 128;
    const unsigned blocks = (unsigned)((4 * ctx->V + threads - 1) / threads);
    if (src_prec == 64)
        compress_gauge_kernel<T, RECON, double><<<blocks, threads, 0, ctx->stream>>>((LVec*)ctx->gauge, (const double*)d_aos, ctx->V, d_stats);
    else
        compress_gauge_kernel<T, RECON, float><<<blocks, threads, 0, ctx->stream>>>((LVec*)ctx->gauge, (const float*)d_aos, ctx->V, d_stats);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

template <typename T, int RECON>
int get_gauge_t(nd_ctx* ctx, double* d_aos) {
    using LVec = typename LinkLayout<T, RECON>::LVec;
    const int threads = 128;
    const unsigned blocks = (unsigned)((4 * ctx->V + threads - 1) / threads);
    reconstruct_gauge_kernel<T, RECON><<<blocks, threads, 0, ctx->stream>>>(d_aos, (const LVec*)ctx->gauge, ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

}  // namespace

#define ND_DISPATCH_TR(ctx, FN, ...)                                            \
    ((ctx)->prec == 32 ? ((ctx)->recon == 18 ? FN<float, 18>(__VA_ARGS__)       \
                          : (ctx)->recon == 12 ? FN<float, 12>(__VA_ARGS__)     \
                                               : FN<float, 8>(__VA_ARGS__))     \
                       : ((ctx)->recon == 18 ? FN<double, 18>(__VA_ARGS__)      \
                          : (ctx)->recon == 12 ? FN<double, 12>(__VA_ARGS__)    \
                                               : FN<double, 8>(__VA_ARGS__)))

extern "C" int nd_set_gauge(nd_ctx* ctx, const void* links_aos, int src_prec, int on_device) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!links_aos || (src_prec != 32 && src_prec != 64)) return nd_fail(ctx, ND_ERR_BAD_ARG, "set_gauge: bad argument");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    ctx->gauge_set = false;
    const size_t in_bytes = (size_t)ctx->V * 4 * 18 * (src_prec / 8);
    void* d_tmp = nullptr;
    const void* d_src = links_aos;
    if (!on_device) {
        ND_CUDA(ctx, cudaMalloc(&d_tmp, in_bytes));
        cudaError_t e = cudaMemcpyAsync(d_tmp, links_aos, in_bytes, cudaMemcpyHostToDevice, ctx->stream);
        if (e != cudaSuccess) { cudaFree(d_tmp); return nd_cuda_check(ctx, e, "set_gauge H2D"); }
        d_src = d_tmp;
    }
    double init[3] = {0.0, 0.0, 1.0e300};
    double* d_stats = ctx->d_result;
    int rc = nd_cuda_check(ctx, cudaMemcpyAsync(d_stats, init, sizeof(init), cudaMemcpyHostToDevice, ctx->stream), "stats init");
    if (rc == ND_OK) rc = ND_DISPATCH_TR(ctx, set_gauge_t, ctx, d_src, src_prec, d_stats);
    if (rc == ND_OK) rc = ndi_read_result(ctx, d_stats, ctx->gstats, 3);
    if (d_tmp) cudaFree(d_tmp);
    if (rc != ND_OK) return rc;
    const double tol = (src_prec == 32) ? 2e-5 : 1e-10;
    if (ctx->gstats[0] > tol || ctx->gstats[1] > tol)
        return nd_fail(ctx, ND_ERR_NOT_SU3, "set_gauge: links are not SU(3): max|U^dag U-1| = %.3e, max|det-1| = %.3e",
                       ctx->gstats[0], ctx->gstats[1]);
    if (ctx->recon == 8) {
        const double thr = (ctx->prec == 32) ? 1e-6 : 1e-10;
        if (ctx->gstats[2] < thr)
            return nd_fail(ctx, ND_ERR_RECON8_SINGULAR, "set_gauge: 8-parameter form singular: min(|a2|^2+|a3|^2) = %.3e < %.1e",
                           ctx->gstats[2], thr);
    }
    ctx->gauge_set = true;
    return ND_OK;
}

extern "C" int nd_get_gauge(nd_ctx* ctx, void* links_aos_c128, int on_device) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!links_aos_c128) return nd_fail(ctx, ND_ERR_BAD_ARG, "get_gauge: null output");
    if (!ctx->gauge_set) return nd_fail(ctx, ND_ERR_BAD_STATE, "get_gauge: gauge field not set");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t bytes = (size_t)ctx->V * 4 * 18 * sizeof(double);
    double* d_out = (double*)links_aos_c128;
    void* d_tmp = nullptr;
    if (!on_device) {
        ND_CUDA(ctx, cudaMalloc(&d_tmp, bytes));
        d_out = (double*)d_tmp;
    }
    int rc = ND_DISPATCH_TR(ctx, get_gauge_t, ctx, d_out);
    if (rc == ND_OK && !on_device)
        rc = nd_cuda_check(ctx, cudaMemcpyAsync(links_aos_c128, d_out, bytes, cudaMemcpyDeviceToHost, ctx->stream), "get_gauge D2H");
    if (rc == ND_OK) rc = nd_cuda_check(ctx, cudaStreamSynchronize(ctx->stream), "get_gauge sync");
    if (d_tmp) cudaFree(d_tmp);
    return rc;
}

extern "C" int nd_gauge_stats(nd_ctx* ctx, double out[3]) {
    if (!ctx || !out) return ND_ERR_BAD_ARG;
    out[0] = ctx->gstats[0]; out[1] = ctx->gstats[1]; out[2] = ctx->gstats[2];
    return ND_OK;
}

namespace {
template <typename T>
int pack_t(nd_ctx* ctx, const void* d_aos, int aos_prec, void* soa) {
    using Vec = typename Prec<T>::Vec;
    const int threads = 256;
    const unsigned blocks = (unsigned)((ctx->V * Prec<T>::NV + threads - 1) / threads);
    if (aos_prec == 64) pack_spinor_kernel<T, double><<<blocks, threads, 0, ctx->stream>>>((Vec*)soa, (const double*)d_aos, ctx->V);
    else pack_spinor_kernel<T, float><<<blocks, threads, 0, ctx->stream>>>((Vec*)soa, (const float*)d_aos, ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
template <typename T>
int unpack_t(nd_ctx* ctx, const void* soa, void* d_aos, int aos_prec) {
    using Vec = typename Prec<T>::Vec;
    const int threads = 256;
    const unsigned blocks = (unsigned)((ctx->V * Prec<T>::NV + threads - 1) / threads);
    if (aos_prec == 64) unpack_spinor_kernel<T, double><<<blocks, threads, 0, ctx->stream>>>((double*)d_aos, (const Vec*)soa, ctx->V);
    else unpack_spinor_kernel<T, float><<<blocks, threads, 0, ctx->stream>>>((float*)d_aos, (const Vec*)soa, ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
}  // namespace

extern "C" int nd_pack_spinor(nd_ctx* ctx, const void* aos, int aos_prec, int aos_on_device, void* soa) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!aos || !soa || (aos_prec != 32 && aos_prec != 64)) return nd_fail(ctx, ND_ERR_BAD_ARG, "pack_spinor: bad argument");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t bytes = (size_t)ctx->V * 24 * (aos_prec / 8);
    void* d_tmp = nullptr;
    const void* d_src = aos;
    if (!aos_on_device) {
        ND_CUDA(ctx, cudaMallocAsync(&d_tmp, bytes, ctx->stream));
        cudaError_t e = cudaMemcpyAsync(d_tmp, aos, bytes, cudaMemcpyHostToDevice, ctx->stream);
        if (e != cudaSuccess) { cudaFreeAsync(d_tmp, ctx->stream); return nd_cuda_check(ctx, e, "pack_spinor H2D"); }
        d_src = d_tmp;
    }
    int rc = (ctx->prec == 32) ? pack_t<float>(ctx, d_src, aos_prec, soa) : pack_t<double>(ctx, d_src, aos_prec, soa);
    if (d_tmp) cudaFreeAsync(d_tmp, ctx->stream);
    return rc;
}

extern "C" int nd_unpack_spinor(nd_ctx* ctx, const void* soa, void* aos, int aos_prec, int aos_on_device) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!aos || !soa || (aos_prec != 32 && aos_prec != 64)) return nd_fail(ctx, ND_ERR_BAD_ARG, "unpack_spinor: bad argument");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t bytes = (size_t)ctx->V * 24 * (aos_prec / 8);
    void* d_tmp = nullptr;
    void* d_dst = aos;
    if (!aos_on_device) {
        ND_CUDA(ctx, cudaMallocAsync(&d_tmp, bytes, ctx->stream));
        d_dst = d_tmp;
    }
    int rc = (ctx->prec == 32) ? unpack_t<float>(ctx, soa, d_dst, aos_prec) : unpack_t<double>(ctx, soa, d_dst, aos_prec);
    if (rc == ND_OK && !aos_on_device) {
        rc = nd_cuda_check(ctx, cudaMemcpyAsync(aos, d_dst, bytes, cudaMemcpyDeviceToHost, ctx->stream), "unpack_spinor D2H");
        if (rc == ND_OK) rc = nd_cuda_check(ctx, cudaStreamSynchronize(ctx->stream), "unpack_spinor sync");
    }
    if (d_tmp) cudaFreeAsync(d_tmp, ctx->stream);
    return rc;
}

extern "C" int nd_convert_spinor(nd_ctx* ctx, void* dst, int dst_prec, const void* src, int src_prec) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!dst || !src || dst == src || (dst_prec != 32 && dst_prec != 64) || (src_prec != 32 && src_prec != 64))
        return nd_fail(ctx, ND_ERR_BAD_ARG, "convert_spinor: bad argument");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    if (dst_prec == src_prec) {
        ND_CUDA(ctx, cudaMemcpyAsync(dst, src, (size_t)24 * ctx->V * (src_prec / 8), cudaMemcpyDeviceToDevice, ctx->stream));
        return ND_OK;
    }
    const int threads = 128;
    const unsigned blocks = (unsigned)((ctx->V + threads - 1) / threads);
    if (dst_prec == 32) convert_spinor_kernel<float, double><<<blocks, threads, 0, ctx->stream>>>((float4*)dst, (const double2*)src, ctx->V);
    else convert_spinor_kernel<double, float><<<blocks, threads, 0, ctx->stream>>>((double2*)dst, (const float4*)src, ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
