// layout.cu - canonical AoS <-> device plane-SoA reordering of spinors, and SU(3) link checking, compression to
// 18 / 12 / 8 reals and reordering (section 2.1, eq. 2.3; 8-parameter form DESIGN.md R8).
//
// All four kernels are pure streaming work and are written so that BOTH sides move in whole 128-byte lines: a CTA takes a
// chunk of consecutive sites, moves the chunk's AoS bytes (contiguous in memory) with coalesced 16-byte accesses through a
// padded shared-memory tile, and every thread touches the plane-SoA side as one 128-bit word per (plane, site) with
// consecutive lanes on consecutive sites.  The shared tile's row stride is padded so that the transposed accesses are free
// of bank conflicts (stride 28 floats / 26 doubles for the 24 reals of a spinor, 19 reals for the 18 of a link).
#include "nd_internal.cuh"
#include "nd_su3.cuh"

namespace {

constexpr int LAYOUT_THREADS = 256;
constexpr int SPINOR_CHUNK = 128;   // sites per CTA
constexpr int LINK_CHUNK = 256;     // links (one mu) per CTA

template <typename Tin> struct Pad24 { static constexpr int stride = sizeof(Tin) == 4 ? 28 : 26; };
template <typename Tin> struct Vec16;
template <> struct Vec16<float> { using type = float4; static constexpr int R = 4; };
template <> struct Vec16<double> { using type = double2; static constexpr int R = 2; };

// contiguous reals [n_rows][ROW] (global, 16-byte aligned start) <-> padded smem rows [n_rows][STRIDE]; ROW % R == 0
template <typename Tin, int ROW, int STRIDE, bool TO_SMEM>
__device__ __forceinline__ void move_rows(Tin* sm, Tin* g, long long n_rows) {
    using V16 = typename Vec16<Tin>::type;
    constexpr int R = Vec16<Tin>::R;
    const int total = (int)n_rows * ROW;
    // 16-byte pieces where the chunk starts on a 16-byte boundary (always, except odd volumes), scalars for the rest
    const int pieces = (((size_t)g & 15) == 0) ? total / R : 0;
    V16* gv = reinterpret_cast<V16*>(g);
    for (int i = threadIdx.x; i < pieces; i += blockDim.x) {
        const int e = i * R;
        if (TO_SMEM) {
            const V16 v = gv[i];
            const Tin* vr = reinterpret_cast<const Tin*>(&v);
#pragma unroll
            for (int j = 0; j < R; j++) sm[((e + j) / ROW) * STRIDE + (e + j) % ROW] = vr[j];   // a piece may straddle two rows
        } else {
            V16 v;
            Tin* vr = reinterpret_cast<Tin*>(&v);
#pragma unroll
            for (int j = 0; j < R; j++) vr[j] = sm[((e + j) / ROW) * STRIDE + (e + j) % ROW];
            gv[i] = v;
        }
    }
    for (int e = pieces * R + threadIdx.x; e < total; e += blockDim.x) {
        if (TO_SMEM) sm[(e / ROW) * STRIDE + e % ROW] = g[e];
        else g[e] = sm[(e / ROW) * STRIDE + e % ROW];
    }
}

// NB bytes between shared memory and registers as 16-byte (or one 8-byte) accesses: with the padded row strides a
// quarter-warp's 128-bit accesses fall on distinct banks, which scalar accesses at the same stride would not
template <int NB> __device__ __forceinline__ void copy_bytes(void* dst, const void* src) {
    if (NB == 8) *reinterpret_cast<uint2*>(dst) = *reinterpret_cast<const uint2*>(src);
    else {
#pragma unroll
        for (int i = 0; i < NB / 16; i++) reinterpret_cast<uint4*>(dst)[i] = reinterpret_cast<const uint4*>(src)[i];
    }
}

// ------------------------------------------------------------------------------------------------- spinors
// AoS reals [s][24] (Tin) -> word (p, s) of the device layout (T)
template <typename T, typename Tin>
__global__ void __launch_bounds__(LAYOUT_THREADS) pack_spinor_kernel(typename Prec<T>::Vec* __restrict__ soa, const Tin* __restrict__ aos,
                                                                     long long V) {
    constexpr int NV = Prec<T>::NV, W = 24 / NV, ST = Pad24<Tin>::stride;
    __shared__ __align__(16) Tin tile[SPINOR_CHUNK * ST];
    const long long s0 = (long long)blockIdx.x * SPINOR_CHUNK;
    const long long ns = (V - s0 < SPINOR_CHUNK) ? V - s0 : SPINOR_CHUNK;
    move_rows<Tin, 24, ST, true>(tile, const_cast<Tin*>(aos) + s0 * 24, ns);
    __syncthreads();
    for (int i = threadIdx.x; i < SPINOR_CHUNK * NV; i += blockDim.x) {
        const int p = i / SPINOR_CHUNK, s = i % SPINOR_CHUNK;
        if (s >= ns) continue;
        __align__(16) Tin r[W];
        copy_bytes<W * (int)sizeof(Tin)>(r, tile + s * ST + p * W);
        typename Prec<T>::Vec w;
        T* wr = reinterpret_cast<T*>(&w);
#pragma unroll
        for (int k = 0; k < W; k++) wr[k] = (T)r[k];
        soa[(long long)p * V + s0 + s] = w;
    }
}

template <typename T, typename Tout>
__global__ void __launch_bounds__(LAYOUT_THREADS) unpack_spinor_kernel(Tout* __restrict__ aos, const typename Prec<T>::Vec* __restrict__ soa,
                                                                       long long V) {
    constexpr int NV = Prec<T>::NV, W = 24 / NV, ST = Pad24<Tout>::stride;
    __shared__ __align__(16) Tout tile[SPINOR_CHUNK * ST];
    const long long s0 = (long long)blockIdx.x * SPINOR_CHUNK;
    const long long ns = (V - s0 < SPINOR_CHUNK) ? V - s0 : SPINOR_CHUNK;
    for (int i = threadIdx.x; i < SPINOR_CHUNK * NV; i += blockDim.x) {
        const int p = i / SPINOR_CHUNK, s = i % SPINOR_CHUNK;
        if (s >= ns) continue;
        const typename Prec<T>::Vec w = soa[(long long)p * V + s0 + s];
        const T* wr = reinterpret_cast<const T*>(&w);
        __align__(16) Tout r[W];
#pragma unroll
        for (int k = 0; k < W; k++) r[k] = (Tout)wr[k];
        copy_bytes<W * (int)sizeof(Tout)>(tile + s * ST + p * W, r);
    }
    __syncthreads();
    move_rows<Tout, 24, ST, false>(tile, aos + s0 * 24, ns);
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
// the statistics are non-negative doubles: their bit patterns order like the values.  A NaN must not be lost on the way
// (fmax/fmin drop NaN operands), so every candidate is first mapped NaN -> +inf for the maxima and NaN -> 0 for the minimum.
template <typename C> __device__ __forceinline__ C nan_to(C x, C v) { return (x == x) ? x : v; }
__device__ __forceinline__ void atomic_max_nonneg(double* addr, double v) {
    atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}
__device__ __forceinline__ void atomic_min_nonneg(double* addr, double v) {
    atomicMin(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

// CTA = LINK_CHUNK consecutive links of one direction mu (grid.y = mu).
// stats[0] = max |U^dag U - 1|, stats[1] = max |det U - 1|, stats[2] = min N, stats[3] = max |reconstruct(stored) - U| entry
template <typename T, int RECON, typename Tin>
__global__ void __launch_bounds__(LAYOUT_THREADS) compress_gauge_kernel(typename LinkLayout<T, RECON>::LVec* __restrict__ g,
                                                                        const Tin* __restrict__ aos, long long V, double* stats) {
    using LL = LinkLayout<T, RECON>;
    using LVec = typename LL::LVec;
    constexpr int W = sizeof(LVec) / sizeof(T);
    constexpr int ST = 19;
    __shared__ __align__(16) Tin tile[LINK_CHUNK * ST];
    const int mu = blockIdx.y;
    const long long s0 = (long long)blockIdx.x * LINK_CHUNK;
    const long long ns = (V - s0 < LINK_CHUNK) ? V - s0 : LINK_CHUNK;
    move_rows<Tin, 18, ST, true>(tile, const_cast<Tin*>(aos) + ((long long)mu * V + s0) * 18, ns);
    __syncthreads();
    const int t = threadIdx.x;
    const bool valid = t < ns;
    const int tr = valid ? t : 0;   // keep the whole warp alive for the shuffles below; the store is predicated
    // checks in the precision of the links as given (C): fp32 input is judged against 2e-5, fp32 arithmetic resolves 1e-7
    using C = Tin;
    cx<C> U[3][3];
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++) U[a][b] = {tile[tr * ST + 2 * (3 * a + b)], tile[tr * ST + 2 * (3 * a + b) + 1]};
    C dev_c = C(0);
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++) {
            cx<C> acc = {a == b ? C(-1) : C(0), C(0)};
#pragma unroll
            for (int k = 0; k < 3; k++) cfma_cj(acc, U[k][a], U[k][b]);
            dev_c = fmax(dev_c, fmax(nan_to(fabs(acc.re), C(INFINITY)), nan_to(fabs(acc.im), C(INFINITY))));
        }
    cx<C> det = U[0][0] * (U[1][1] * U[2][2] - U[1][2] * U[2][1]) - U[0][1] * (U[1][0] * U[2][2] - U[1][2] * U[2][0]) +
                     U[0][2] * (U[1][0] * U[2][1] - U[1][1] * U[2][0]);
    C ddev_c = fmax(nan_to(fabs(det.re - C(1)), C(INFINITY)), nan_to(fabs(det.im), C(INFINITY)));
    C N_c = nan_to(U[0][1].re * U[0][1].re + U[0][1].im * U[0][1].im + U[0][2].re * U[0][2].re + U[0][2].im * U[0][2].im, C(0));
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
        r[6] = (T)tan(0.25 * atan2((double)U[0][0].im, (double)U[0][0].re));
        r[7] = (T)tan(0.25 * atan2((double)U[2][0].im, (double)U[2][0].re));
    }
    LVec words[LL::NL];
#pragma unroll
    for (int p = 0; p < LL::NL; p++) {
        T* wr = reinterpret_cast<T*>(&words[p]);
#pragma unroll
        for (int k = 0; k < W; k++) wr[k] = r[p * W + k];
    }
    // what the stencil will see: rebuild the link from the stored words with the stencil's own routine and compare
    C rerr_c = C(0);
    {
        cx<T> R[3][3];
        reconstruct_link<T, RECON>(words, R);
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++)
                rerr_c = fmax(rerr_c, fmax(nan_to(fabs((C)R[a][b].re - U[a][b].re), C(INFINITY)),
                                       nan_to(fabs((C)R[a][b].im - U[a][b].im), C(INFINITY))));
    }
    // warp-level reduce before the atomics (statistics in fp64 from here on)
    double dev = dev_c, ddev = ddev_c, rerr = rerr_c, N = N_c;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dev = fmax(dev, __shfl_xor_sync(0xffffffffu, dev, o));
        ddev = fmax(ddev, __shfl_xor_sync(0xffffffffu, ddev, o));
        rerr = fmax(rerr, __shfl_xor_sync(0xffffffffu, rerr, o));
        N = fmin(N, __shfl_xor_sync(0xffffffffu, N, o));
    }
    // ... one CTA-level reduction through shared memory, and an atomic only where the CTA improves on the value already there
    // (tens of thousands of CTAs hammering four addresses with atomics were the kernel's bottleneck)
    __shared__ double cta_stats[LAYOUT_THREADS / 32][4];
    if ((threadIdx.x & 31) == 0) {
        double* r = cta_stats[threadIdx.x >> 5];
        r[0] = dev; r[1] = ddev; r[2] = N; r[3] = rerr;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < LAYOUT_THREADS / 32; w++) {
            dev = fmax(dev, cta_stats[w][0]);
            ddev = fmax(ddev, cta_stats[w][1]);
            N = fmin(N, cta_stats[w][2]);
            rerr = fmax(rerr, cta_stats[w][3]);
        }
        const volatile double* cur = stats;
        if (dev > cur[0]) atomic_max_nonneg(stats + 0, dev);
        if (ddev > cur[1]) atomic_max_nonneg(stats + 1, ddev);
        if (N < cur[2]) atomic_min_nonneg(stats + 2, N);
        if (rerr > cur[3]) atomic_max_nonneg(stats + 3, rerr);
    }
    if (!valid) return;
    LVec* dst = g + (long long)mu * LL::NL * V + s0 + t;
#pragma unroll
    for (int p = 0; p < LL::NL; p++) dst[p * V] = words[p];
}

template <typename T, int RECON>
__global__ void __launch_bounds__(LAYOUT_THREADS) reconstruct_gauge_kernel(double* __restrict__ aos,
                                                                           const typename LinkLayout<T, RECON>::LVec* __restrict__ g, long long V) {
    constexpr int ST = 19;
    __shared__ __align__(16) double tile[LINK_CHUNK * ST];
    const int mu = blockIdx.y;
    const long long s0 = (long long)blockIdx.x * LINK_CHUNK;
    const long long ns = (V - s0 < LINK_CHUNK) ? V - s0 : LINK_CHUNK;
    const int t = threadIdx.x;
    if (t < ns) {
        cx<T> U[3][3];
        load_link<T, RECON>(g, V, mu, s0 + t, U);
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) { tile[t * ST + 2 * (3 * a + b)] = (double)U[a][b].re; tile[t * ST + 2 * (3 * a + b) + 1] = (double)U[a][b].im; }
    }
    __syncthreads();
    move_rows<double, 18, ST, false>(tile, aos + ((long long)mu * V + s0) * 18, ns);
}

template <typename T, int RECON>
int set_gauge_t(nd_ctx* ctx, const void* d_aos, int src_prec, double* d_stats) {
    using LVec = typename LinkLayout<T, RECON>::LVec;
    const dim3 grid((unsigned)((ctx->V + LINK_CHUNK - 1) / LINK_CHUNK), 4, 1);
    if (src_prec == 64)
        compress_gauge_kernel<T, RECON, double><<<grid, LAYOUT_THREADS, 0, ctx->stream>>>((LVec*)ctx->gauge, (const double*)d_aos, ctx->V, d_stats);
    else
        compress_gauge_kernel<T, RECON, float><<<grid, LAYOUT_THREADS, 0, ctx->stream>>>((LVec*)ctx->gauge, (const float*)d_aos, ctx->V, d_stats);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

template <typename T, int RECON>
int get_gauge_t(nd_ctx* ctx, double* d_aos) {
    using LVec = typename LinkLayout<T, RECON>::LVec;
    const dim3 grid((unsigned)((ctx->V + LINK_CHUNK - 1) / LINK_CHUNK), 4, 1);
    reconstruct_gauge_kernel<T, RECON><<<grid, LAYOUT_THREADS, 0, ctx->stream>>>(d_aos, (const LVec*)ctx->gauge, ctx->V);
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
    ndi_drop_graphs(ctx);
    const size_t in_bytes = (size_t)ctx->V * 4 * 18 * (src_prec / 8);
    void* d_tmp = nullptr;
    const void* d_src = links_aos;
    if (!on_device) {
        ND_CUDA(ctx, cudaMalloc(&d_tmp, in_bytes));
        cudaError_t e = cudaMemcpyAsync(d_tmp, links_aos, in_bytes, cudaMemcpyHostToDevice, ctx->stream);
        if (e != cudaSuccess) { cudaFree(d_tmp); return nd_cuda_check(ctx, e, "set_gauge H2D"); }
        d_src = d_tmp;
    } else if (((size_t)links_aos & 15) != 0) {
        return nd_fail(ctx, ND_ERR_BAD_ARG, "set_gauge: device links must be 16-byte aligned");
    }
    double* d_stats = ctx->d_result;
    ctx->h_result[0] = 0.0; ctx->h_result[1] = 0.0; ctx->h_result[2] = 1.0e300; ctx->h_result[3] = 0.0;
    int rc = nd_cuda_check(ctx, cudaMemcpyAsync(d_stats, ctx->h_result, 4 * sizeof(double), cudaMemcpyHostToDevice, ctx->stream), "stats init");
    if (rc == ND_OK) rc = nd_cuda_check(ctx, cudaStreamSynchronize(ctx->stream), "stats init");   // h_result is reused below
    if (rc == ND_OK) rc = ND_DISPATCH_TR(ctx, set_gauge_t, ctx, d_src, src_prec, d_stats);
    if (rc == ND_OK) rc = ndi_read_result(ctx, d_stats, ctx->gstats, 4);
    if (d_tmp) cudaFree(d_tmp);
    if (rc != ND_OK) return rc;
    // written so that a NaN statistic (a NaN link) FAILS the test
    const double tol = (src_prec == 32) ? 2e-5 : 1e-10;
    if (!(ctx->gstats[0] <= tol) || !(ctx->gstats[1] <= tol))
        return nd_fail(ctx, ND_ERR_NOT_SU3, "set_gauge: links are not SU(3): max|U^dag U-1| = %.3e, max|det-1| = %.3e",
                       ctx->gstats[0], ctx->gstats[1]);
    if (ctx->recon == 8) {
        // singular as N -> 0 (R8): refuse fields where the 8-parameter form is undefined, and fields whose links
        // come back from the stored parameters with more than rtol error (rounding is amplified by ~1/N)
        const double thr = (ctx->prec == 32) ? 1e-6 : 1e-10;
        const double rtol = (ctx->prec == 32) ? 2e-3 : 1e-8;
        if (!(ctx->gstats[2] >= thr) || !(ctx->gstats[3] <= rtol))
            return nd_fail(ctx, ND_ERR_RECON8_SINGULAR,
                           "set_gauge: 8-parameter form ill-conditioned: min(|a2|^2+|a3|^2) = %.3e (need >= %.1e), "
                           "max reconstruction error = %.3e (need <= %.1e)", ctx->gstats[2], thr, ctx->gstats[3], rtol);
    } else if (!(ctx->gstats[3] <= ((ctx->prec == 32) ? 1e-5 : 1e-12))) {
        return nd_fail(ctx, ND_ERR_NOT_SU3, "set_gauge: stored links do not reproduce the input: max error %.3e", ctx->gstats[3]);
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
    } else if (((size_t)links_aos_c128 & 15) != 0) {
        return nd_fail(ctx, ND_ERR_BAD_ARG, "get_gauge: device output must be 16-byte aligned");
    }
    int rc = ND_DISPATCH_TR(ctx, get_gauge_t, ctx, d_out);
    if (rc == ND_OK && !on_device)
        rc = nd_cuda_check(ctx, cudaMemcpyAsync(links_aos_c128, d_out, bytes, cudaMemcpyDeviceToHost, ctx->stream), "get_gauge D2H");
    if (rc == ND_OK) rc = nd_cuda_check(ctx, cudaStreamSynchronize(ctx->stream), "get_gauge sync");
    if (d_tmp) cudaFree(d_tmp);
    return rc;
}

extern "C" int nd_gauge_stats(nd_ctx* ctx, double out[4]) {
    if (!ctx || !out) return ND_ERR_BAD_ARG;
    for (int i = 0; i < 4; i++) out[i] = ctx->gstats[i];
    return ND_OK;
}

namespace {
template <typename T>
int pack_t(nd_ctx* ctx, const void* d_aos, int aos_prec, void* soa) {
    using Vec = typename Prec<T>::Vec;
    const unsigned blocks = (unsigned)((ctx->V + SPINOR_CHUNK - 1) / SPINOR_CHUNK);
    if (aos_prec == 64) pack_spinor_kernel<T, double><<<blocks, LAYOUT_THREADS, 0, ctx->stream>>>((Vec*)soa, (const double*)d_aos, ctx->V);
    else pack_spinor_kernel<T, float><<<blocks, LAYOUT_THREADS, 0, ctx->stream>>>((Vec*)soa, (const float*)d_aos, ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
template <typename T>
int unpack_t(nd_ctx* ctx, const void* soa, void* d_aos, int aos_prec) {
    using Vec = typename Prec<T>::Vec;
    const unsigned blocks = (unsigned)((ctx->V + SPINOR_CHUNK - 1) / SPINOR_CHUNK);
    if (aos_prec == 64) unpack_spinor_kernel<T, double><<<blocks, LAYOUT_THREADS, 0, ctx->stream>>>((double*)d_aos, (const Vec*)soa, ctx->V);
    else unpack_spinor_kernel<T, float><<<blocks, LAYOUT_THREADS, 0, ctx->stream>>>((float*)d_aos, (const Vec*)soa, ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
}  // namespace

extern "C" int nd_pack_spinor(nd_ctx* ctx, const void* aos, int aos_prec, int aos_on_device, void* soa) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!aos || !soa || (aos_prec != 32 && aos_prec != 64)) return nd_fail(ctx, ND_ERR_BAD_ARG, "pack_spinor: bad argument");
    if (aos_on_device && ((size_t)aos & 15) != 0) return nd_fail(ctx, ND_ERR_BAD_ARG, "pack_spinor: device AoS must be 16-byte aligned");
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
    if (aos_on_device && ((size_t)aos & 15) != 0) return nd_fail(ctx, ND_ERR_BAD_ARG, "unpack_spinor: device AoS must be 16-byte aligned");
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
