// sign.cu - Chebyshev approximation of sign(Q) by a fused Clenshaw recurrence, the projected sign function and the
// Neuberger-Dirac operator (section 2.2-2.3: eq. 2.4-2.6, 2.7, 2.11; L56-73, L81-84, L110-113).
//
//   sign(Q) ~ X P_n(X^2),  X = Q/qnorm,  P_n(y) = sum_{k=0}^n c_k T_k(z),  z = (2y-1-eps)/(1-eps)      (2.5; R7)
//   Z = alpha Q^2 + beta,  alpha = 2/((1-eps) qnorm^2),  beta = -(1+eps)/(1-eps)
//   b_n = c_n eta;  b_k = c_k eta + 2 Z b_{k+1} - b_{k+2}  (k = n-1..1);  P eta = c_0 eta + Z b_1 - b_2    (R9)
//   chi = Q P eta / qnorm;   sign eta ~ sum_k sign(nu_k) u_k <u_k,eta> + chi - sum_k u_k <u_k,chi>           (2.11)
//   D_N eta = prefactor (eta + gamma5 sign eta)                                                             (2.4)
//
// Every Clenshaw step is two stencil launches; the vector update is the epilogue of the second one
// (nd_apply_Q_axpbycz), so the recurrence vectors are read/written exactly once per step: 2n+1 stencil launches per
// sign application and nothing else - no axpy kernels, and no copy for b_n = c_n eta either (its factor rides in the scalars of
// the first two steps).  No host synchronisation anywhere: the projection coefficients stay on
// the device, so the whole application can be replayed as one CUDA graph.
#include <algorithm>
#include <cmath>

#include "nd_internal.cuh"

namespace {

// coef_jk = sign(nu_k) <u_k,eta_j> - <u_k,chi_j> for nb right-hand sides
// (dots = [<u,eta_0> (2l) | ... | <u,eta_{nb-1}> | <u,chi_0> (2l) | ... | <u,chi_{nb-1}>], coef[(j*l + k)*2])
__global__ void lowmode_coef_kernel(double* __restrict__ coef, const double* __restrict__ dots, const double* __restrict__ nu, int l, int nb) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= l * nb) return;
    const int k = i % l;
    const double sg = (nu[k] > 0.0) ? 1.0 : ((nu[k] < 0.0) ? -1.0 : 0.0);
    coef[2 * i] = sg * dots[2 * i] - dots[2 * (l * nb + i)];
    coef[2 * i + 1] = sg * dots[2 * i + 1] - dots[2 * (l * nb + i) + 1];
}

// kind 0: out = sign(Q) in ; kind 1: out = pa in + pb gamma5 sign(Q) in ; for nb right-hand sides stored back to back
// (out, eta: nb spinors; work: 3 nb spinors): every launch of the sequence handles all of them (stencils: blockIdx.y = rhs)
int enqueue_sign(nd_ctx* ctx, int nb, void* out, const void* eta, void* work, int kind, double pa, double pb) {
    const size_t sb = nd_spinor_bytes(ctx) * (size_t)nb;
    char* bA = (char*)work;
    char* bB = bA + sb;
    char* tmp = bB + sb;
    const int n = ctx->n;
    const double* c = ctx->cheb.data();
    const double m = ctx->m_sign;
    const double alpha = 2.0 / ((1.0 - ctx->eps) * ctx->qnorm * ctx->qnorm);
    const double beta = -(1.0 + ctx->eps) / (1.0 - ctx->eps);
    int rc;
    if (n == 0) {
        rc = ndi_apply_Q_batch(ctx, nb, out, eta, m, true, c[0] / ctx->qnorm, 0, nullptr, 0, nullptr, 0, nullptr);
        if (rc != ND_OK) return rc;
    } else {
        // b_n = c_n eta is never materialised (nor b_{n+1} = 0): the first step reads eta itself and carries c_n in its scalars,
        //   b_{n-1} = f alpha c_n Q Q eta + (f beta c_n + c_{n-1}) eta,
        // and the second step's "- b_n" becomes part of its eta term, (c_{n-2} - c_n) eta.  2n + 1 launches, no copy kernel.
        for (int k = n - 1; k >= 0; k--) {
            // tmp = Q b_{k+1};   b_k = f*(alpha Q tmp + beta b_{k+1}) - b_{k+2} + c_k eta,  f = 2 (k >= 1) or 1 (k = 0)
            const bool first = (k == n - 1), second = (k == n - 2);
            rc = ndi_apply_Q_batch(ctx, nb, tmp, first ? eta : bA, m, false, 1, 0, nullptr, 0, nullptr, 0, nullptr);
            if (rc != ND_OK) return rc;
            const double f = (k >= 1) ? 2.0 : 1.0;
            if (first)
                rc = ndi_apply_Q_batch(ctx, nb, bB, tmp, m, true, f * alpha * c[n], 0, nullptr, 0, nullptr, f * beta * c[n] + c[k], eta);
            else
                rc = ndi_apply_Q_batch(ctx, nb, bB, tmp, m, true, f * alpha, f * beta, bA, second ? 0.0 : -1.0, bB, second ? c[k] - c[n] : c[k], eta);
            if (rc != ND_OK) return rc;
            char* t = bA; bA = bB; bB = t;
        }
        // bA = P eta ;  chi = Q P eta / qnorm
        rc = ndi_apply_Q_batch(ctx, nb, out, bA, m, true, 1.0 / ctx->qnorm, 0, nullptr, 0, nullptr, 0, nullptr);
        if (rc != ND_OK) return rc;
    }
    const int l = ctx->l;
    if (l > 0) {
        // one pass over the modes for <u_k,eta_j> and <u_k,chi_j> of all right-hand sides
        const size_t s1 = nd_spinor_bytes(ctx);
        const void* cols[2 * ND_MAX_RHS];
        for (int j = 0; j < nb; j++) {
            cols[j] = (const char*)eta + (size_t)j * s1;
            cols[nb + j] = (const char*)out + (size_t)j * s1;
        }
        rc = ndi_block_dot_cols_dev(ctx, l, ctx->u, 2 * nb, cols, ctx->d_result);
        if (rc != ND_OK) return rc;
        lowmode_coef_kernel<<<(l * nb + 63) / 64, 64, 0, ctx->stream>>>(ctx->d_coef, ctx->d_result, ctx->d_nu, l, nb);
        ND_LAUNCHED(ctx);
    }
    if (l > 0 || kind == 1) {
        rc = (nb == 1) ? ndi_block_axpy_dev(ctx, l, ctx->d_coef, ctx->u, out, kind, eta, pa, pb)
                       : ndi_block_axpy_batch_dev(ctx, l, nb, ctx->d_coef, ctx->u, out, kind, eta, pa, pb);
        if (rc != ND_OK) return rc;
    }
    return ND_OK;
}

int apply_sign_impl(nd_ctx* ctx, int nb, void* out, const void* in, void* work, int kind, double pa, double pb, int use_graph) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!out || !in || !work || out == in) return nd_fail(ctx, ND_ERR_BAD_ARG, "apply_sign/DN: null or aliased argument");
    if (nb < 1 || nb > ND_MAX_RHS || 4 * nb * (ctx->l > 0 ? ctx->l : 1) > ND_RESULT_DOUBLES || 2 * nb * ctx->l > 2 * ND_MAX_BLOCK_L)
        return nd_fail(ctx, ND_ERR_BAD_ARG, "apply_sign/DN: 1 <= nrhs <= %d and nrhs * l <= %d", ND_MAX_RHS, ND_MAX_BLOCK_L);
    if (!ctx->gauge_set) return nd_fail(ctx, ND_ERR_BAD_STATE, "apply_sign/DN: gauge field not set");
    if (!ctx->poly_set) return nd_fail(ctx, ND_ERR_BAD_STATE, "apply_sign/DN: polynomial not set (nd_set_sign_poly)");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    if (!use_graph || ctx->stream == nullptr || ctx->shard_n > 1) return enqueue_sign(ctx, nb, out, in, work, kind, pa, pb);
    for (auto& g : ctx->graphs)
        if (g.out == out && g.in == in && g.work == work && g.kind == kind && g.pa == pa && g.pb == pb && g.nrhs == nb) {
            ND_CUDA(ctx, cudaGraphLaunch(g.exec, ctx->stream));
            ctx->launches += g.nodes;
            return ND_OK;
        }
    const long long before = ctx->launches;
    ND_CUDA(ctx, cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal));
    int rc = enqueue_sign(ctx, nb, out, in, work, kind, pa, pb);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(ctx->stream, &graph);
    const long long nodes = ctx->launches - before;
    ctx->launches = before;
    if (rc != ND_OK) {
        if (graph) cudaGraphDestroy(graph);
        return rc;
    }
    ND_CUDA(ctx, e);
    nd_graph_entry g;
    g.out = out; g.in = in; g.work = work; g.kind = kind; g.pa = pa; g.pb = pb; g.exec = nullptr; g.nodes = nodes; g.nrhs = nb;
    e = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    ND_CUDA(ctx, e);
    if (ctx->graphs.size() >= 16) ndi_drop_graphs(ctx);
    ctx->graphs.push_back(g);
    ND_CUDA(ctx, cudaGraphLaunch(g.exec, ctx->stream));
    ctx->launches += nodes;
    return ND_OK;
}

}  // namespace

int ndi_apply_DNm(nd_ctx* ctx, void* out, const void* in, double pa, double pb, void* work, int use_graph) {
    return apply_sign_impl(ctx, 1, out, in, work, 1, pa, pb, use_graph);
}

// --------------------------------------------------------------------------------------------------- C ABI
extern "C" int nd_cheb_coeffs(int n, double eps, double* c, double* delta) {
    if (n < 0 || !(eps > 0.0 && eps < 1.0) || !c) return ND_ERR_BAD_ARG;
    typedef long double ld;
    const ld pi = acosl(-1.0L);
    std::vector<ld> f(n + 1), th(n + 1);
    for (int j = 0; j <= n; j++) {
        th[j] = pi * ((ld)j + 0.5L) / (ld)(n + 1);
        const ld z = cosl(th[j]);
        const ld y = ((1.0L - (ld)eps) * z + 1.0L + (ld)eps) / 2.0L;
        f[j] = 1.0L / sqrtl(y);
    }
    for (int k = 0; k <= n; k++) {
        ld s = 0.0L;
        for (int j = 0; j <= n; j++) s += f[j] * cosl((ld)k * th[j]);
        s *= 2.0L / (ld)(n + 1);
        if (k == 0) s *= 0.5L;   // full c_0: P = sum_{k=0}^n c_k T_k as eq. 2.5 is printed
        c[k] = (double)s;
    }
    if (delta) {
        // delta = max |1 - sqrt(y) P(y)| on a geometric and a linear grid of [eps, 1] (eq. 2.6)
        const int npts = 200001;
        double worst = 0.0;
        const double lr = log(1.0 / eps);
        for (int pass = 0; pass < 2; pass++)
            for (int i = 0; i < npts; i++) {
                const double t = (double)i / (double)(npts - 1);
                const double y = pass == 0 ? eps * exp(lr * t) : eps + (1.0 - eps) * t;
                const double z = (2.0 * y - 1.0 - eps) / (1.0 - eps);
                double b1 = 0.0, b2 = 0.0;
                for (int k = n; k >= 1; k--) {
                    const double b0 = c[k] + 2.0 * z * b1 - b2;
                    b2 = b1;
                    b1 = b0;
                }
                const double P = c[0] + z * b1 - b2;
                const double d = fabs(1.0 - sqrt(y) * P);
                if (d > worst) worst = d;
            }
        *delta = worst;
    }
    return ND_OK;
}

// Min-max coefficients (eq. 2.6, "minmax polynomials"): the polynomial of degree n minimising
// delta = max_{eps<=y<=1} |1 - sqrt(y) P(y)|, by the Remez exchange for the weighted problem w (f - P), f = y^{-1/2}, w = y^{1/2}:
// solve  sum_k c_k T_k(z_i) + (-1)^i E / w(y_i) = f(y_i)  on a reference of n+2 points (long double elimination), move the
// reference to the alternating extrema of the error on a fine grid, repeat until max|e| <= (1 + 1e-3) |E|.  Conventions as
// nd_cheb_coeffs (z = (2y-1-eps)/(1-eps), full c_0).  Host utility, no GPU.
extern "C" int nd_minmax_coeffs(int n, double eps, double* c, double* delta, double* levelled) {
    if (n < 0 || n > 4096 || !(eps > 0.0 && eps < 1.0) || !c) return ND_ERR_BAD_ARG;
    typedef long double ld;
    const ld pi = acosl(-1.0L);
    const int m = n + 2;
    std::vector<ld> z(m), sol(m), M((size_t)m * (m + 1));
    for (int i = 0; i < m; i++) z[i] = -cosl(pi * (ld)i / (ld)(m - 1));
    const int ng = 64 * m + 2;
    std::vector<double> zg(ng), eg(ng);
    zg[0] = -1.0;
    zg[ng - 1] = 1.0;
    for (int i = 1; i < ng - 1; i++) zg[i] = -cos(M_PI * ((double)i - 0.5) / (double)(ng - 2));
    auto error_at = [&](double zz) {
        double b1 = 0.0, b2 = 0.0;
        for (int k = n; k >= 1; k--) {
            const double b0 = c[k] + 2.0 * zz * b1 - b2;
            b2 = b1;
            b1 = b0;
        }
        const double y = 0.5 * ((1.0 - eps) * zz + 1.0 + eps);
        return 1.0 - sqrt(y) * (c[0] + zz * b1 - b2);
    };
    ld E = 0.0L;
    double emax = 0.0;
    for (int it = 0; it < 80; it++) {
        for (int i = 0; i < m; i++) {
            const ld y = 0.5L * ((1.0L - (ld)eps) * z[i] + 1.0L + (ld)eps);
            const ld th = acosl(z[i] > 1.0L ? 1.0L : (z[i] < -1.0L ? -1.0L : z[i]));
            for (int k = 0; k <= n; k++) M[(size_t)i * (m + 1) + k] = cosl((ld)k * th);
            M[(size_t)i * (m + 1) + n + 1] = ((i & 1) ? -1.0L : 1.0L) / sqrtl(y);
            M[(size_t)i * (m + 1) + m] = 1.0L / sqrtl(y);
        }
        for (int k = 0; k < m; k++) {   // elimination with partial pivoting
            int p = k;
            for (int i = k + 1; i < m; i++)
                if (fabsl(M[(size_t)i * (m + 1) + k]) > fabsl(M[(size_t)p * (m + 1) + k])) p = i;
            if (M[(size_t)p * (m + 1) + k] == 0.0L) return ND_ERR_NO_CONVERGENCE;
            if (p != k)
                for (int j = 0; j <= m; j++) std::swap(M[(size_t)k * (m + 1) + j], M[(size_t)p * (m + 1) + j]);
            for (int i = k + 1; i < m; i++) {
                const ld f = M[(size_t)i * (m + 1) + k] / M[(size_t)k * (m + 1) + k];
                if (f == 0.0L) continue;
                for (int j = k; j <= m; j++) M[(size_t)i * (m + 1) + j] -= f * M[(size_t)k * (m + 1) + j];
            }
        }
        for (int k = m - 1; k >= 0; k--) {
            ld t = M[(size_t)k * (m + 1) + m];
            for (int j = k + 1; j < m; j++) t -= M[(size_t)k * (m + 1) + j] * sol[j];
            sol[k] = t / M[(size_t)k * (m + 1) + k];
        }
        for (int k = 0; k <= n; k++) c[k] = (double)sol[k];
        E = sol[n + 1];
        emax = 0.0;
        for (int i = 0; i < ng; i++) {
            eg[i] = error_at(zg[i]);
            emax = std::max(emax, fabs(eg[i]));
        }
        if (emax <= (1.0 + 1e-3) * (double)fabsl(E)) break;
        // the alternating extrema: the largest |e| of every stretch of constant sign; surplus ones are dropped at the ends
        std::vector<int> ext;
        int best = 0;
        for (int i = 1; i <= ng; i++) {
            if (i == ng || (eg[i] >= 0.0) != (eg[best] >= 0.0)) {
                ext.push_back(best);
                best = i;
            } else if (fabs(eg[i]) > fabs(eg[best])) {
                best = i;
            }
        }
        size_t lo = 0, hi = ext.size();
        while (hi - lo > (size_t)m) {
            if (fabs(eg[ext[lo]]) < fabs(eg[ext[hi - 1]])) lo++;
            else hi--;
        }
        if (hi - lo < (size_t)m) break;   // degree beyond what the grid / fp64 evaluation resolves: keep the last iterate
        for (int i = 0; i < m; i++) z[i] = (ld)zg[ext[lo + i]];
    }
    if (levelled) *levelled = (double)fabsl(E);
    if (delta) {
        // the same measurement as nd_cheb_coeffs: geometric and linear grid of [eps, 1]
        double worst = emax;
        const int npts = 100001;
        const double lr = log(1.0 / eps);
        for (int pass = 0; pass < 2; pass++)
            for (int i = 0; i < npts; i++) {
                const double t = (double)i / (double)(npts - 1);
                const double y = pass == 0 ? eps * exp(lr * t) : eps + (1.0 - eps) * t;
                worst = std::max(worst, fabs(error_at((2.0 * y - 1.0 - eps) / (1.0 - eps))));
            }
        *delta = worst;
    }
    return ND_OK;
}

extern "C" int nd_set_sign_poly(nd_ctx* ctx, int n, const double* c, double eps, double qnorm, double m) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (n < 0 || !c || !(eps > 0.0 && eps < 1.0) || !(qnorm > 0.0)) return nd_fail(ctx, ND_ERR_BAD_ARG, "set_sign_poly: bad argument");
    ctx->cheb.assign(c, c + n + 1);
    ctx->n = n;
    ctx->eps = eps;
    ctx->qnorm = qnorm;
    ctx->m_sign = m;
    ctx->poly_set = true;
    ndi_drop_graphs(ctx);
    return ND_OK;
}

extern "C" int nd_set_lowmodes(nd_ctx* ctx, int l, const void* u_soa, const double* nu) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (l < 0 || l > ND_MAX_BLOCK_L || (l > 0 && (!u_soa || !nu))) return nd_fail(ctx, ND_ERR_BAD_ARG, "set_lowmodes: bad argument (0 <= l <= %d)", ND_MAX_BLOCK_L);
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    ndi_drop_graphs(ctx);
    ctx->l = l;
    ctx->u = l ? u_soa : nullptr;
    ctx->nu.assign(nu, nu + l);
    if (l) {
        ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        for (int i = 0; i < l; i++) ctx->h_result[i] = nu[i];
        ND_CUDA(ctx, cudaMemcpyAsync(ctx->d_nu, ctx->h_result, (size_t)l * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    }
    return ND_OK;
}

extern "C" int nd_apply_sign(nd_ctx* ctx, void* out, const void* in, void* work, int use_graph) {
    return apply_sign_impl(ctx, 1, out, in, work, 0, 0.0, 0.0, use_graph);
}
extern "C" int nd_apply_DN(nd_ctx* ctx, void* out, const void* in, double prefactor, void* work, int use_graph) {
    return apply_sign_impl(ctx, 1, out, in, work, 1, prefactor, prefactor, use_graph);
}
extern "C" int nd_apply_sign_multi(nd_ctx* ctx, int nrhs, void* out, const void* in, void* work, int use_graph) {
    return apply_sign_impl(ctx, nrhs, out, in, work, 0, 0.0, 0.0, use_graph);
}
extern "C" int nd_apply_DN_multi(nd_ctx* ctx, int nrhs, void* out, const void* in, double prefactor, void* work, int use_graph) {
    return apply_sign_impl(ctx, nrhs, out, in, work, 1, prefactor, prefactor, use_graph);
}
