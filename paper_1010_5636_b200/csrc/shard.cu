// shard.cu - domain decomposition of the lattice along x0 (time) over several GPUs, one process per GPU (
// PAPER.md:L52 "no communication necessary if we assign each lattice site ... a single thread", L146 "increase the lattice volume").
//
// Rank r of R owns the time-slices [r T/R, (r+1) T/R) as a LOCAL lattice of dims (T/R, L1, L2, L3): a context of that size whose
// time direction is OPEN.  Of the stencil's eight hops only the two time hops of the two boundary slices leave the rank, and
// what they need is a half-spinor (12 reals per site, the projected spinor of eq. 2.1's (1 -+ gamma_0)) - the links never travel:
//     to the NEXT rank  (its backward hop at its first slice):  w(x) = U_0(x, last)^dagger (1 + gamma_0) phi(x, last)
//     to the PREVIOUS rank (its forward hop at its last slice):  h(x) = (1 - gamma_0) phi(x, first)   (it multiplies by its own U_0)
// each times bc_time where the face crosses the global seam T-1 <-> 0.  One stencil application is then
//     halo_pack (faces of `in`)  ->  exchange start  ->  the ordinary stencil kernel on the local lattice with the wrapped time
//     hops switched off (phase 0; it overlaps the transfer)  ->  exchange wait  ->  halo_apply: the two boundary slices receive
//     their missing hop, scaled like the kernel's own output (gamma5, -1/2, the fused epilogue's s0).
// The transfers themselves are the caller's (callbacks: NCCL send/recv over NVLink from torch.distributed in dist.py, device
// copies in the single-GPU emulation of the tests); reductions (block dot, residues) are summed over ranks by the all-reduce
// callback before anything consumes them, so every rank takes identical decisions.
#include "nd_dirac.cuh"

namespace {

template <typename T> struct HaloWords { static constexpr int NW = sizeof(T) == 4 ? 3 : 6; };

__device__ __forceinline__ void half_store(float4* dst, long long n, long long i, const cx<float> (&h)[2][3]) {
    dst[0 * n + i] = make_float4(h[0][0].re, h[0][0].im, h[0][1].re, h[0][1].im);
    dst[1 * n + i] = make_float4(h[0][2].re, h[0][2].im, h[1][0].re, h[1][0].im);
    dst[2 * n + i] = make_float4(h[1][1].re, h[1][1].im, h[1][2].re, h[1][2].im);
}
__device__ __forceinline__ void half_load(const float4* src, long long n, long long i, cx<float> (&h)[2][3]) {
    const float4 a = src[0 * n + i], b = src[1 * n + i], c = src[2 * n + i];
    h[0][0] = {a.x, a.y}; h[0][1] = {a.z, a.w}; h[0][2] = {b.x, b.y};
    h[1][0] = {b.z, b.w}; h[1][1] = {c.x, c.y}; h[1][2] = {c.z, c.w};
}
__device__ __forceinline__ void half_store(double2* dst, long long n, long long i, const cx<double> (&h)[2][3]) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int c = 0; c < 3; c++) dst[(3 * s + c) * n + i] = make_double2(h[s][c].re, h[s][c].im);
}
__device__ __forceinline__ void half_load(const double2* src, long long n, long long i, cx<double> (&h)[2][3]) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const double2 v = src[(3 * s + c) * n + i];
            h[s][c] = {v.x, v.y};
        }
}

// faces of `in`: blockIdx.y = 0: to_next (from the last slice), 1: to_prev (from the first slice); thread = site of the slice
template <typename T, int RECON>
__global__ void halo_pack_kernel(typename Prec<T>::Vec* __restrict__ to_next, typename Prec<T>::Vec* __restrict__ to_prev,
                                 const typename Prec<T>::Vec* __restrict__ in, const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge,
                                 long long V, long long S0, int L0, T phase_next, T phase_prev) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S0) return;
    cx<T> psi[12], h[2][3];
    if (blockIdx.y == 0) {
        const long long s = (long long)(L0 - 1) * S0 + i;
        cx<T> U[3][3], g[2][3];
        load_spinor<T>(in, V, s, psi);
        load_link<T, RECON>(gauge, V, 0, s, U);
        project<T, 0, +1>(psi, phase_next, h);
        mul_Udag(U, h, g);
        half_store(to_next, S0, i, g);
    } else {
        load_spinor<T>(in, V, i, psi);
        project<T, 0, -1>(psi, phase_prev, h);
        half_store(to_prev, S0, i, h);
    }
}

// out(x) += s0 * gamma5 (-1/2) [the time hop that came from the neighbour rank]; blockIdx.y = 0: first slice (backward hop,
// complete in from_prev), 1: last slice (forward hop: own link times the projected spinor in from_next)
template <typename T, int RECON>
__global__ void halo_apply_kernel(typename Prec<T>::Vec* out, const typename Prec<T>::Vec* __restrict__ from_prev,
                                  const typename Prec<T>::Vec* __restrict__ from_next,
                                  const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, long long V, long long S0, int L0, T s0) {
    constexpr int NV = Prec<T>::NV;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S0) return;
    cx<T> acc[12], g[2][3];
#pragma unroll
    for (int k = 0; k < 12; k++) acc[k] = {T(0), T(0)};
    long long s;
    if (blockIdx.y == 0) {
        s = i;
        half_load(from_prev, S0, i, g);
        accumulate<T, 0, +1>(g, acc);
    } else {
        s = (long long)(L0 - 1) * S0 + i;
        cx<T> U[3][3], h[2][3];
        half_load(from_next, S0, i, h);
        load_link<T, RECON>(gauge, V, 0, s, U);
        mul_U(U, h, g);
        accumulate<T, 0, -1>(g, acc);
    }
    typename Prec<T>::Vec w[NV];
#pragma unroll
    for (int p = 0; p < NV; p++) w[p] = out[p * V + s];
    cx<T> o[12];
    words_to_cx(w, o);
#pragma unroll
    for (int k = 0; k < 12; k++) {
        const T f = s0 * ((k < 6) ? T(-0.5) : T(0.5));   // gamma5 [ -1/2 ... ], then the fused epilogue's factor
        o[k] = {fma(f, acc[k].re, o[k].re), fma(f, acc[k].im, o[k].im)};
    }
    cx_to_words(o, w);
#pragma unroll
    for (int p = 0; p < NV; p++) out[p * V + s] = w[p];
}

template <typename T, int RECON>
int halo_pack_t(nd_ctx* ctx, const void* in) {
    using Vec = typename Prec<T>::Vec;
    using LVec = typename LinkLayout<T, RECON>::LVec;
    const long long S0 = ctx->V / ctx->dims[0];
    const dim3 grid((unsigned)((S0 + 127) / 128), 2, 1);
    const T pn = (ctx->shard_rank == ctx->shard_n - 1) ? T(ctx->bc) : T(1);
    const T pp = (ctx->shard_rank == 0) ? T(ctx->bc) : T(1);
    // destinations: the own send buffers (the caller's callbacks move them), or - peer-to-peer mode - the neighbours' receive
    // windows themselves: the stores of this kernel ARE the transfer (over NVLink when the windows are peer-mapped)
    Vec* to_next = (Vec*)ctx->halo[0];
    Vec* to_prev = (Vec*)ctx->halo[1];
    if (ctx->peer_own) {
        const size_t hb = nd_halo_bytes(ctx);
        to_next = (Vec*)((char*)ctx->peer_next + (size_t)(2 * ctx->halo_parity + 0) * hb);   // the next rank's from_prev face
        to_prev = (Vec*)((char*)ctx->peer_prev + (size_t)(2 * ctx->halo_parity + 1) * hb);   // the previous rank's from_next face
    }
    halo_pack_kernel<T, RECON><<<grid, 128, 0, ctx->stream>>>(to_next, to_prev, (const Vec*)in, (const LVec*)ctx->gauge,
                                                                ctx->V, S0, ctx->dims[0], pn, pp);
    ND_LAUNCHED(ctx);
    return ND_OK;
}
template <typename T, int RECON>
int halo_apply_t(nd_ctx* ctx, void* out, double s0) {
    using Vec = typename Prec<T>::Vec;
    using LVec = typename LinkLayout<T, RECON>::LVec;
    const long long S0 = ctx->V / ctx->dims[0];
    const dim3 grid((unsigned)((S0 + 127) / 128), 2, 1);
    const Vec* from_prev = (const Vec*)ctx->halo[2];
    const Vec* from_next = (const Vec*)ctx->halo[3];
    if (ctx->peer_own) {
        const size_t hb = nd_halo_bytes(ctx);
        from_prev = (const Vec*)((const char*)ctx->peer_own + (size_t)(2 * ctx->halo_parity + 0) * hb);
        from_next = (const Vec*)((const char*)ctx->peer_own + (size_t)(2 * ctx->halo_parity + 1) * hb);
    }
    halo_apply_kernel<T, RECON><<<grid, 128, 0, ctx->stream>>>((Vec*)out, from_prev, from_next, (const LVec*)ctx->gauge, ctx->V, S0,
                                                                 ctx->dims[0], T(s0));
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

int ndi_halo_pack(nd_ctx* ctx, const void* in) { return ND_DISPATCH_TR(ctx, halo_pack_t, ctx, in); }
int ndi_halo_apply(nd_ctx* ctx, void* out, double s0) { return ND_DISPATCH_TR(ctx, halo_apply_t, ctx, out, s0); }

// sum over ranks of n doubles in device memory, before anything consumes them (no-op without sharding)
int ndi_allreduce(nd_ctx* ctx, double* d_buf, int n) {
    if (ctx->shard_n <= 1 || !ctx->allreduce) return ND_OK;
    const int rc = ctx->allreduce(ctx->comm_user, d_buf, n);
    return rc == 0 ? ND_OK : nd_fail(ctx, ND_ERR_CUDA, "sharding: the all-reduce callback failed (%d)", rc);
}

extern "C" int nd_shard_layout(int T, int nranks, int rank, int* t_begin, int* t_local, int* crosses_seam_prev, int* crosses_seam_next) {
    if (T < 2 || nranks < 1 || rank < 0 || rank >= nranks || T % nranks != 0 || T / nranks < 2) return ND_ERR_BAD_ARG;
    if (t_begin) *t_begin = rank * (T / nranks);
    if (t_local) *t_local = T / nranks;
    if (crosses_seam_prev) *crosses_seam_prev = (rank == 0);
    if (crosses_seam_next) *crosses_seam_next = (rank == nranks - 1);
    return ND_OK;
}

extern "C" size_t nd_halo_bytes(const nd_ctx* ctx) { return ctx ? (size_t)(ctx->V / ctx->dims[0]) * 12 * (ctx->prec / 8) : 0; }

extern "C" int nd_set_sharding(nd_ctx* ctx, int rank, int nranks, nd_exchange_start_fn start, nd_exchange_wait_fn wait,
                               nd_allreduce_fn allreduce, void* user) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (nranks < 1 || rank < 0 || rank >= nranks) return nd_fail(ctx, ND_ERR_BAD_ARG, "set_sharding: bad rank %d of %d", rank, nranks);
    if (nranks > 1 && (!wait || !allreduce)) return nd_fail(ctx, ND_ERR_BAD_ARG, "set_sharding: callbacks missing");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    ndi_drop_graphs(ctx);
    for (int i = 0; i < 4; i++) {
        if (ctx->halo[i]) cudaFree(ctx->halo[i]);
        ctx->halo[i] = nullptr;
    }
    ctx->shard_rank = rank;
    ctx->shard_n = nranks;
    ctx->exchange_start = start;
    ctx->exchange_wait = wait;
    ctx->allreduce = allreduce;
    ctx->comm_user = user;
    ctx->peer_own = ctx->peer_next = ctx->peer_prev = nullptr;
    ctx->halo_parity = 0;
    if (nranks > 1)
        for (int i = 0; i < 4; i++) ND_CUDA(ctx, cudaMalloc(&ctx->halo[i], nd_halo_bytes(ctx)));
    return ND_OK;
}

extern "C" int nd_set_halo_peers(nd_ctx* ctx, void* recv_own, void* recv_of_next, void* recv_of_prev) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (ctx->shard_n <= 1) return nd_fail(ctx, ND_ERR_BAD_STATE, "set_halo_peers: the context is not sharded (nd_set_sharding first)");
    const bool all = recv_own && recv_of_next && recv_of_prev, none = !recv_own && !recv_of_next && !recv_of_prev;
    if (!all && !none) return nd_fail(ctx, ND_ERR_BAD_ARG, "set_halo_peers: give all three windows or none");
    if (none && !ctx->exchange_start) return nd_fail(ctx, ND_ERR_BAD_STATE, "set_halo_peers: no exchange-start callback to fall back to");
    if (all && ((((size_t)recv_own | (size_t)recv_of_next | (size_t)recv_of_prev) & 15) != 0 || (nd_halo_bytes(ctx) & 15) != 0))
        return nd_fail(ctx, ND_ERR_BAD_ARG, "set_halo_peers: windows must be 16-byte aligned");
    ctx->peer_own = recv_own;
    ctx->peer_next = recv_of_next;
    ctx->peer_prev = recv_of_prev;
    ctx->halo_parity = 0;
    return ND_OK;
}

// The two halves of a sharded stencil application, also exported for callers that drive the exchange themselves.
extern "C" int nd_halo_buffers(nd_ctx* ctx, void** send_next, void** send_prev, void** recv_prev, void** recv_next) {
    if (!ctx || ctx->shard_n <= 1) return ND_ERR_BAD_STATE;
    if (send_next) *send_next = ctx->halo[0];
    if (send_prev) *send_prev = ctx->halo[1];
    if (recv_prev) *recv_prev = ctx->halo[2];
    if (recv_next) *recv_next = ctx->halo[3];
    return ND_OK;
}
