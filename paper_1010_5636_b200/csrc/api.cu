// api.cu - context life cycle and error reporting of the C-ABI library (include/nd_b200.h).
#include <cstdarg>
#include <cstdlib>
#include <cstring>
#include <new>

#include "nd_internal.cuh"

int nd_fail(nd_ctx* ctx, int code, const char* fmt, ...) {
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

int nd_cuda_check(nd_ctx* ctx, cudaError_t e, const char* what) {
    if (e == cudaSuccess) return ND_OK;
    return nd_fail(ctx, ND_ERR_CUDA, "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
}

extern "C" int nd_create(nd_ctx** out, const int dims[4], int prec, int recon, int bc_time, int device, void* stream) {
    if (!out) return ND_ERR_BAD_ARG;
    *out = nullptr;
    if (!dims) return ND_ERR_BAD_ARG;
    for (int i = 0; i < 4; i++)
        if (dims[i] < 2) return ND_ERR_BAD_ARG;
    if ((prec != 32 && prec != 64) || (recon != 18 && recon != 12 && recon != 8) || (bc_time != 1 && bc_time != -1))
        return ND_ERR_BAD_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return ND_ERR_CUDA;   // no CPU fallback
    if (cudaSetDevice(device) != cudaSuccess) return ND_ERR_CUDA;
    nd_ctx* ctx = new (std::nothrow) nd_ctx();
    if (!ctx) return ND_ERR_NOMEM;
    for (int i = 0; i < 4; i++) ctx->dims[i] = dims[i];
    ctx->V = (long long)dims[0] * dims[1] * dims[2] * dims[3];
    ctx->prec = prec;
    ctx->recon = recon;
    ctx->bc = bc_time;
    ctx->device = device;
    ctx->stream = (cudaStream_t)stream;
    ctx->gauge = nullptr;
    ctx->gauge_set = false;
    ctx->gstats[0] = ctx->gstats[1] = ctx->gstats[2] = ctx->gstats[3] = 0.0;
    ctx->d_partial = ctx->d_result = ctx->h_result = ctx->d_coef = ctx->d_nu = nullptr;
    ctx->n = 0;
    ctx->eps = ctx->qnorm = ctx->m_sign = 0.0;
    ctx->poly_set = false;
    ctx->l = 0;
    ctx->u = nullptr;
    ctx->launches = 0;
    ctx->capturing = false;
    {
        // stencil CTA tile (x1, x2, x3) of 128 sites: x3 extent = the largest power of two <= 32 dividing L3, then x2 and
        // x1 are doubled in turn while they divide the lattice (32^3: 2 x 2 x 32); lattices without a tile of >= 64 sites
        // use the linear mapping.
        int lb[3] = {0, 0, 0}, threads = 1;
        auto grow = [&](int i) {
            if (threads * 2 > 128 || (2 << lb[i]) > (i == 2 ? 32 : 128) || dims[i + 1] % (2 << lb[i]) != 0) return false;
            lb[i]++;
            threads *= 2;
            return true;
        };
        while (grow(2)) {}
        for (bool g = true; g;) {
            g = grow(1);
            g = grow(0) || g;
        }
        for (int i = 0; i < 3; i++) ctx->tile_lb[i] = lb[i];
        ctx->tile_threads = (threads >= 64) ? threads : 0;
    }
    ctx->hop_max_sites = 16384;   // below this volume there are fewer sites than lanes: hop-parallel stencil (wilson.cu)
    ctx->num_sms = 148;
    cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, device);
    ctx->err[0] = 0;
    for (int i = 0; i < 8; i++) ctx->tile_ctas_per_sm[i] = 0;
    for (int i = 0; i < ND_TMAP_SLOTS; i++) ctx->tmaps[i].base = nullptr;
    ctx->tmap_next = 0;
    ctx->tile_ok = ndi_tile_supported(ctx);
    ctx->stencil_variant = ND_STENCIL_AUTO;
    ctx->dot_configured = false;
    ctx->shard_rank = 0;
    ctx->shard_n = 1;
    ctx->in_shard_call = false;
    for (int i = 0; i < 4; i++) ctx->halo[i] = nullptr;
    ctx->peer_own = ctx->peer_next = ctx->peer_prev = nullptr;
    ctx->halo_parity = 0;
    ctx->exchange_start = nullptr;
    ctx->exchange_wait = nullptr;
    ctx->allreduce = nullptr;
    ctx->comm_user = nullptr;
    // fp32 recon 18 is stored as 9 float2, everything else in 128-bit words: bytes = 4 * recon * V * prec/8
    ctx->gauge_bytes = (size_t)4 * recon * ctx->V * (prec / 8);
    cudaError_t e = cudaMalloc(&ctx->gauge, ctx->gauge_bytes);
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_partial, (size_t)ND_RESULT_DOUBLES * ND_MAX_RED_BLOCKS * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_result, ND_RESULT_DOUBLES * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_coef, 2 * ND_MAX_BLOCK_L * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_nu, ND_MAX_BLOCK_L * sizeof(double));
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->h_result, ND_RESULT_DOUBLES * sizeof(double));
    if (e != cudaSuccess) {
        nd_destroy(ctx);
        return (e == cudaErrorMemoryAllocation) ? ND_ERR_NOMEM : ND_ERR_CUDA;
    }
    *out = ctx;
    return ND_OK;
}

int ndi_drop_graphs(nd_ctx* ctx) {
    for (auto& g : ctx->graphs)
        if (g.exec) cudaGraphExecDestroy(g.exec);
    ctx->graphs.clear();
    return ND_OK;
}

extern "C" int nd_destroy(nd_ctx* ctx) {
    if (!ctx) return ND_ERR_BAD_ARG;
    cudaSetDevice(ctx->device);
    ndi_drop_graphs(ctx);
    if (ctx->gauge) cudaFree(ctx->gauge);
    if (ctx->d_partial) cudaFree(ctx->d_partial);
    if (ctx->d_result) cudaFree(ctx->d_result);
    if (ctx->d_coef) cudaFree(ctx->d_coef);
    if (ctx->d_nu) cudaFree(ctx->d_nu);
    if (ctx->h_result) cudaFreeHost(ctx->h_result);
    for (int i = 0; i < 4; i++)
        if (ctx->halo[i]) cudaFree(ctx->halo[i]);
    delete ctx;
    return ND_OK;
}

extern "C" const char* nd_last_error(const nd_ctx* ctx) { return ctx ? ctx->err : "null context"; }

extern "C" int nd_set_stream(nd_ctx* ctx, void* stream) {
    if (!ctx) return ND_ERR_BAD_ARG;
    ctx->stream = (cudaStream_t)stream;
    ndi_drop_graphs(ctx);
    return ND_OK;
}

extern "C" int nd_set_stencil_variant(nd_ctx* ctx, int variant) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (variant != ND_STENCIL_AUTO && variant != ND_STENCIL_SITE && variant != ND_STENCIL_TILE && variant != ND_STENCIL_TILE_TMA &&
        variant != ND_STENCIL_TILE4)
        return nd_fail(ctx, ND_ERR_BAD_ARG, "set_stencil_variant: unknown variant %d", variant);
    if ((variant == ND_STENCIL_TILE || variant == ND_STENCIL_TILE_TMA || variant == ND_STENCIL_TILE4) && !ctx->tile_ok)
        return nd_fail(ctx, ND_ERR_BAD_ARG, "set_stencil_variant: the tiled kernel needs x3 extent 32 or 16, even x1 / x2 extents >= 4 (x3 extent 16: x2 extent divisible by 4; fp64: recon 12 / 8) and >= 8 slices of 128 sites per SM");
    if (variant == ND_STENCIL_TILE4 && (ctx->prec != 32 || ctx->dims[3] != 32))
        return nd_fail(ctx, ND_ERR_BAD_ARG, "set_stencil_variant: the four-slot tiled kernel exists in fp32 for x3 extent 32 only");
    if (variant == ND_STENCIL_TILE_TMA && ctx->dims[3] != 32)
        return nd_fail(ctx, ND_ERR_BAD_ARG, "set_stencil_variant: the tensor-map tiled kernel exists for x3 extent 32 only");
    ctx->stencil_variant = variant;
    ndi_drop_graphs(ctx);
    return ND_OK;
}

extern "C" int nd_get_stencil_variant(const nd_ctx* ctx) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (ctx->stencil_variant != ND_STENCIL_AUTO) return ctx->stencil_variant;
    return ctx->tile_ok ? ND_STENCIL_TILE : ND_STENCIL_SITE;
}

extern "C" int nd_get_stencil_variant_for(const nd_ctx* ctx, int fused_epilogue, int nrhs) {
    if (!ctx || nrhs < 1) return ND_ERR_BAD_ARG;
    return ndi_select_stencil(ctx, fused_epilogue != 0, nrhs);
}

extern "C" long long nd_volume(const nd_ctx* ctx) { return ctx ? ctx->V : 0; }
extern "C" size_t nd_spinor_bytes(const nd_ctx* ctx) { return ctx ? (size_t)24 * ctx->V * (ctx->prec / 8) : 0; }
extern "C" size_t nd_gauge_bytes(const nd_ctx* ctx) { return ctx ? ctx->gauge_bytes : 0; }
extern "C" long long nd_launch_count(const nd_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int nd_apply_Q(nd_ctx* ctx, void* out, const void* in, double m) {
    if (!ctx) return ND_ERR_BAD_ARG;
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    return ndi_apply_Q(ctx, out, in, m, false, 1.0, 0.0, nullptr, 0.0, nullptr, 0.0, nullptr);
}

extern "C" int nd_apply_Q2(nd_ctx* ctx, void* out, const void* in, void* tmp, double m) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!tmp || tmp == in || tmp == out) return nd_fail(ctx, ND_ERR_BAD_ARG, "apply_Q2: tmp null or aliased");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    int rc = ndi_apply_Q(ctx, tmp, in, m, false, 1.0, 0.0, nullptr, 0.0, nullptr, 0.0, nullptr);
    if (rc != ND_OK) return rc;
    return ndi_apply_Q(ctx, out, tmp, m, false, 1.0, 0.0, nullptr, 0.0, nullptr, 0.0, nullptr);
}

extern "C" int nd_apply_Q_axpbycz(nd_ctx* ctx, void* out, const void* in, double m, double s0, double s1, const void* v1,
                                  double s2, const void* v2, double s3, const void* v3) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if ((s1 != 0.0 && !v1) || (s2 != 0.0 && !v2) || (s3 != 0.0 && !v3)) return nd_fail(ctx, ND_ERR_BAD_ARG, "apply_Q_axpbycz: null vector with non-zero scalar");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    return ndi_apply_Q(ctx, out, in, m, true, s0, s1, v1, s2, v2, s3, v3);
}
