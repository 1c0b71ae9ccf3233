// lowmodes.cu - the l lowest eigenpairs of Q^2 and the Rayleigh-Ritz step of Q in their span (PAPER.md:L79-88,
// section 2.3, eq. 2.7-2.8).
//
// PAPER.md:L79 says only that the low modes are found "by minimizing the Ritz functional of Q^2" (ref. [13]); no steps
// are given.  DESIGN.md reading R13: any method delivering ||Q^2 x - theta x|| <= tol with orthonormal x.  Built here:
// Chebyshev-filtered block subspace iteration, which minimises the block Ritz functional tr(X^dagger Q^2 X) over
// orthonormal blocks X and is made of exactly the kernels D_N uses (plain stencil, stencil with the fused three-term
// epilogue, block dot, grouped Gram / rotation kernels):
//
//   X = k = l + lextra Gaussian vectors, orthonormalised
//   repeat:  X_j <- T_d((Q^2 - c)/e) X_j       [c-e, c+e] = [cut, qnorm^2] is damped, everything below cut amplified
//            orthonormalise X  (Gram matrix, Hermitian eigendecomposition on the host, X <- X W Lambda^{-1/2}; repeated
//                               when the Gram matrix is ill-conditioned)
//            Rayleigh-Ritz of Q^2 in span X: H = X^dagger (Q^2 X), H = W Theta W^dagger, X <- X W
//            residuals r_j = ||Q^2 x_j - theta_j x_j|| for j < l (computed explicitly), cut <- theta_{k-1};
//            leading columns with r_j <= tol/2 are locked (not filtered again)
//   until max_j r_j <= tol
//   Rayleigh-Ritz of Q in the span of the l lowest x_j: M = X^dagger Q X -> (nu_k, u_k), rho_k = ||(Q - nu_k) u_k||   (2.7, 2.8)
//
// Everything of size V runs on the GPU; the k x k Hermitian eigenproblems (k <= 256) run on the host in fp64 with a
// cyclic Jacobi method (nd_heev, no LAPACK dependency).
#include <algorithm>
#include <cmath>
#include <complex>

#include "nd_internal.cuh"

typedef std::complex<double> zc;

// ------------------------------------------------------------------------------- host Hermitian eigen-solver
// Cyclic Jacobi for a k x k Hermitian matrix a (row-major complex, (re, im) pairs): a = Z diag(w) Z^dagger, w ascending,
// eigenvector j in COLUMN j of z (row-major).  Only the Hermitian part of a is used.
extern "C" int nd_heev(int k, const double* a_in, double* w, double* z_out) {
    if (k < 1 || !a_in || !w || !z_out) return ND_ERR_BAD_ARG;
    std::vector<zc> A((size_t)k * k), Z((size_t)k * k, zc(0.0, 0.0));
    for (int i = 0; i < k; i++)
        for (int j = 0; j < k; j++) {
            const zc x(a_in[2 * ((size_t)i * k + j)], a_in[2 * ((size_t)i * k + j) + 1]);
            const zc y(a_in[2 * ((size_t)j * k + i)], a_in[2 * ((size_t)j * k + i) + 1]);
            A[(size_t)i * k + j] = 0.5 * (x + std::conj(y));
        }
    for (int i = 0; i < k; i++) Z[(size_t)i * k + i] = 1.0;
    double scale = 0.0;
    for (auto& x : A) scale = std::max(scale, std::abs(x));
    if (scale == 0.0) scale = 1.0;
    for (int sweep = 0; sweep < 60; sweep++) {
        double off = 0.0;
        for (int p = 0; p < k; p++)
            for (int q = p + 1; q < k; q++) off += std::norm(A[(size_t)p * k + q]);
        if (std::sqrt(off) <= 1e-14 * scale * std::sqrt((double)k)) break;   // off-diagonal Frobenius norm at rounding level
        for (int p = 0; p < k; p++)
            for (int q = p + 1; q < k; q++) {
                const zc apq = A[(size_t)p * k + q];
                const double b = std::abs(apq);
                if (b <= 1e-300) continue;
                const double app = A[(size_t)p * k + p].real(), aqq = A[(size_t)q * k + q].real();
                if (b <= 1e-18 * (std::fabs(app) + std::fabs(aqq)) && sweep > 3) {
                    A[(size_t)p * k + q] = A[(size_t)q * k + p] = 0.0;
                    continue;
                }
                const zc ph = apq / b;   // e^{i phi}
                const double tau = (aqq - app) / (2.0 * b);
                const double t = (tau >= 0.0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
                const double c = 1.0 / std::sqrt(1.0 + t * t), s = t * c;
                const zc sp = s * ph;   // s e^{i phi}
                // A <- A J,  J = [[c, s e^{i phi}], [-s e^{-i phi}, c]] on columns (p, q); Z <- Z J.  Written in real
                // arithmetic: std::complex products go through the NaN-recovering library routine and run 10x slower.
                const double sr = sp.real(), si = sp.imag();   // s e^{i phi} = sr + i si, s e^{-i phi} = sr - i si
                auto rot_cols = [&](zc& ap, zc& aq) {
                    const double pr = ap.real(), pi = ap.imag(), qr = aq.real(), qi = aq.imag();
                    ap = zc(c * pr - (sr * qr + si * qi), c * pi - (sr * qi - si * qr));
                    aq = zc((sr * pr - si * pi) + c * qr, (sr * pi + si * pr) + c * qi);
                };
                for (int i = 0; i < k; i++) {
                    rot_cols(A[(size_t)i * k + p], A[(size_t)i * k + q]);
                    rot_cols(Z[(size_t)i * k + p], Z[(size_t)i * k + q]);
                }
                // A <- J^dagger A on rows (p, q): row_p <- c row_p - s e^{i phi} row_q, row_q <- s e^{-i phi} row_p + c row_q
                zc* rp = &A[(size_t)p * k];
                zc* rq = &A[(size_t)q * k];
                for (int j = 0; j < k; j++) {
                    const double pr = rp[j].real(), pi = rp[j].imag(), qr = rq[j].real(), qi = rq[j].imag();
                    rp[j] = zc(c * pr - (sr * qr - si * qi), c * pi - (sr * qi + si * qr));
                    rq[j] = zc((sr * pr + si * pi) + c * qr, (sr * pi - si * pr) + c * qi);
                }
                A[(size_t)p * k + q] = A[(size_t)q * k + p] = 0.0;
                A[(size_t)p * k + p] = A[(size_t)p * k + p].real();
                A[(size_t)q * k + q] = A[(size_t)q * k + q].real();
            }
    }
    std::vector<int> order(k);
    for (int i = 0; i < k; i++) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int x, int y) { return A[(size_t)x * k + x].real() < A[(size_t)y * k + y].real(); });
    for (int j = 0; j < k; j++) {
        w[j] = A[(size_t)order[j] * k + order[j]].real();
        for (int i = 0; i < k; i++) {
            z_out[2 * ((size_t)i * k + j)] = Z[(size_t)i * k + order[j]].real();
            z_out[2 * ((size_t)i * k + j) + 1] = Z[(size_t)i * k + order[j]].imag();
        }
    }
    return ND_OK;
}

extern "C" int nd_projector_error(int l, const double* nu, const double* rho, int nrest, const double* rest,
                                  double kappa[2], double bound[2], double* d) {
    if (l < 1 || !nu || !rho || nrest < 0 || (nrest > 0 && !rest) || !kappa || !bound) return ND_ERR_BAD_ARG;
    double k2[2] = {0.0, 0.0};
    for (int k = 0; k < l; k++) {
        if (nu[k] == 0.0) return ND_ERR_BAD_ARG;   // the sign of nu_k must be unambiguous
        double dk = INFINITY;
        for (int j = 0; j < nrest; j++) dk = std::min(dk, std::fabs(rest[j] - nu[k]));
        for (int j = 0; j < l; j++)
            if ((nu[j] > 0.0) != (nu[k] > 0.0)) dk = std::min(dk, std::fabs(nu[j] - nu[k]));
        if (d) d[k] = dk;
        const double q = rho[k] / dk;
        k2[nu[k] > 0.0 ? 0 : 1] += q * q;
    }
    for (int i = 0; i < 2; i++) {
        kappa[i] = std::sqrt(k2[i]);
        const double x = 2.0 * kappa[i] * (1.0 + 2.0 * kappa[i]);
        bound[i] = (x < 1.0) ? kappa[i] * (1.0 + 2.0 * kappa[i]) / (1.0 - x) : INFINITY;
    }
    return ND_OK;
}

namespace {

struct Solver {
    nd_ctx* ctx;
    size_t sb;
    int k;
    double m;
    char *X, *Y, *s0, *s1, *s2;
    double* d_mat;   // 2 k^2 doubles on the device
    std::vector<double> h_mat;
    long long stencils;

    char* x(int j) { return X + (size_t)j * sb; }
    char* y(int j) { return Y + (size_t)j * sb; }

    int Q(void* out, const void* in) {
        stencils++;
        return ndi_apply_Q(ctx, out, in, m, false, 1, 0, nullptr, 0, nullptr, 0, nullptr);
    }
    int Qepi(void* out, const void* in, double a0, double a1, const void* v1, double a2, const void* v2) {
        stencils++;
        return ndi_apply_Q(ctx, out, in, m, true, a0, a1, v1, a2, v2, 0, nullptr);
    }
    // G[i][j] = <A_i, B_j>, i < na, j < nb  -> h_mat row-major (na x nb complex)
    int gram(char* A, int na, char* B, int nb) {
        int rc = ndi_block_gram_dev(ctx, na, A, nb, B, d_mat);   // d_mat[(j*na + i)*2 + c] = <A_i, B_j>
        if (rc != ND_OK) return rc;
        std::vector<double> tmp((size_t)2 * na * nb);
        ND_CUDA(ctx, cudaMemcpyAsync(tmp.data(), d_mat, tmp.size() * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        h_mat.resize((size_t)2 * na * nb);
        for (int j = 0; j < nb; j++)
            for (int i = 0; i < na; i++) {
                h_mat[2 * ((size_t)i * nb + j)] = tmp[(size_t)2 * na * j + 2 * i];
                h_mat[2 * ((size_t)i * nb + j) + 1] = tmp[(size_t)2 * na * j + 2 * i + 1];
            }
        return ND_OK;
    }
    // dst_j = sum_i src_i C[i][j], i < ns, j < nd   (C row-major complex on the host)
    int rotate(char* dst, int nd, char* src, int ns, const std::vector<zc>& C) {
        std::vector<double> col((size_t)2 * ns * nd);
        for (int j = 0; j < nd; j++)
            for (int i = 0; i < ns; i++) {
                col[(size_t)2 * ns * j + 2 * i] = C[(size_t)i * nd + j].real();
                col[(size_t)2 * ns * j + 2 * i + 1] = C[(size_t)i * nd + j].imag();
            }
        ND_CUDA(ctx, cudaMemcpyAsync(d_mat, col.data(), col.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));   // `col` is pageable and dies with this frame
        return ndi_block_rotate_dev(ctx, ns, d_mat, src, nd, dst);
    }
    // X <- X W Lambda^{-1/2} with X^dagger X = W Lambda W^dagger (result back in X)
    int orthonormalise(int reps) {
        std::vector<double> w(k), z((size_t)2 * k * k);
        for (int r = 0; r < reps; r++) {
            int rc = gram(X, k, X, k);
            if (rc != ND_OK) return rc;
            rc = nd_heev(k, h_mat.data(), w.data(), z.data());
            if (rc != ND_OK) return rc;
            std::vector<zc> C((size_t)k * k);
            for (int j = 0; j < k; j++) {
                if (!(w[j] > 0.0) || !std::isfinite(w[j])) return nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "lowmodes: block lost rank (Gram eigenvalue %g)", w[j]);
                const double f = 1.0 / std::sqrt(w[j]);
                for (int i = 0; i < k; i++) C[(size_t)i * k + j] = f * zc(z[2 * ((size_t)i * k + j)], z[2 * ((size_t)i * k + j) + 1]);
            }
            rc = rotate(Y, k, X, k, C);
            if (rc != ND_OK) return rc;
            std::swap(X, Y);
            // the loss of orthogonality of X W Lambda^{-1/2} is ~ rounding * cond(Gram): a second pass only when needed
            if (w[k - 1] / w[0] < (ctx->prec == 32 ? 30.0 : 1.0e6)) break;
        }
        return ND_OK;
    }
    // X_j <- T_d((Q^2 - c)/e) X_j, d even; t_{i+1} = (2/e)(Q^2 - c) t_i - t_{i-1}, the update folded into the 2nd stencil
    // columns j < first are locked (their residual met the tolerance): they stay in the block for the orthonormalisation
    // and the Rayleigh-Ritz step but are not filtered again
    int filter(int d, double lo, double hi, int first) {
        const double c = 0.5 * (hi + lo), e = 0.5 * (hi - lo);
        for (int j = first; j < k; j++) {
            char* P = x(j);   // t_{i-1}
            char* R = s0;     // t_i
            int rc = Q(s1, P);
            if (rc != ND_OK) return rc;
            rc = Qepi(R, s1, 1.0 / e, -c / e, P, 0.0, nullptr);   // t_1
            if (rc != ND_OK) return rc;
            for (int i = 1; i < d; i++) {
                rc = Q(s1, R);
                if (rc != ND_OK) return rc;
                rc = Qepi(P, s1, 2.0 / e, -2.0 * c / e, R, -1.0, P);   // t_{i+1} over t_{i-1}
                if (rc != ND_OK) return rc;
                std::swap(P, R);
            }
            // d even: t_d sits in x(j) again
        }
        return ND_OK;
    }
    int norm(const void* v, double* out) {
        int rc = ndi_block_dot_dev(ctx, 1, v, v, ctx->d_result);
        if (rc != ND_OK) return rc;
        double t[2];
        rc = ndi_read_result(ctx, ctx->d_result, t, 2);
        *out = std::sqrt(std::max(t[0], 0.0));
        return rc;
    }
};

}  // namespace

extern "C" int nd_lowmodes_compute(nd_ctx* ctx, int l, int lextra, int degree, double m, double tol, int maxit,
                                   unsigned long long seed, void* u_out, double* nu, double* resid, double* theta_rest,
                                   void* work, long long* stats) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (l < 1 || lextra < 0 || l + lextra > ND_MAX_BLOCK_L || degree < 2 || maxit < 1 || !(tol > 0.0) || !u_out || !nu ||
        !resid || !work)
        return nd_fail(ctx, ND_ERR_BAD_ARG, "lowmodes_compute: bad argument (1 <= l, l + lextra <= %d, degree >= 2)", ND_MAX_BLOCK_L);
    if (!ctx->gauge_set) return nd_fail(ctx, ND_ERR_BAD_STATE, "lowmodes_compute: gauge field not set");
    if (12 * ctx->V < l + lextra) return nd_fail(ctx, ND_ERR_BAD_ARG, "lowmodes_compute: block larger than the space");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    Solver S;
    S.ctx = ctx;
    S.sb = nd_spinor_bytes(ctx);
    S.k = l + lextra;
    S.m = m;
    S.stencils = 0;
    const int k = S.k;
    S.X = (char*)work;
    S.Y = S.X + (size_t)k * S.sb;
    S.s0 = S.Y + (size_t)k * S.sb;
    S.s1 = S.s0 + S.sb;
    S.s2 = S.s1 + S.sb;
    S.d_mat = nullptr;
    ND_CUDA(ctx, cudaMalloc((void**)&S.d_mat, (size_t)2 * k * k * sizeof(double)));
    const int d = degree + (degree & 1);
    const double hi = (std::fabs(4.0 + m) + 4.0) * (std::fabs(4.0 + m) + 4.0);   // ||Q||^2 <= (|4+m|+4)^2 (R6)
    int rc = ND_OK, it = 0;
    bool converged = false;
    std::vector<double> theta(k), z((size_t)2 * k * k), rq(l, 0.0);
    auto finish = [&](int code) {
        cudaFree(S.d_mat);
        if (stats) { stats[0] = it; stats[1] = S.stencils; }
        return code;
    };
    for (int j = 0; j < k; j++) {
        rc = nd_gaussian(ctx, S.x(j), seed + (unsigned long long)j);
        if (rc != ND_OK) return finish(rc);
    }
    rc = S.orthonormalise(2);
    if (rc != ND_OK) return finish(rc);
    double cut = -1.0;   // unknown before the first Rayleigh-Ritz step
    int nlock = 0;
    for (it = 0; it <= maxit; it++) {
        if (it > 0) {
            rc = S.filter(d, cut, hi, nlock);
            if (rc != ND_OK) return finish(rc);
            rc = S.orthonormalise(2);
            if (rc != ND_OK) return finish(rc);
        }
        // Rayleigh-Ritz of Q^2: Y = Q^2 X, H = X^dagger Y
        for (int j = 0; j < k; j++) {
            rc = S.Q(S.s1, S.x(j));
            if (rc == ND_OK) rc = S.Q(S.y(j), S.s1);
            if (rc != ND_OK) return finish(rc);
        }
        rc = S.gram(S.X, k, S.Y, k);
        if (rc == ND_OK) rc = nd_heev(k, S.h_mat.data(), theta.data(), z.data());
        if (rc != ND_OK) return finish(rc);
        std::vector<zc> W((size_t)k * k);
        for (size_t i = 0; i < W.size(); i++) W[i] = zc(z[2 * i], z[2 * i + 1]);
        rc = S.rotate(S.Y, k, S.X, k, W);
        if (rc != ND_OK) return finish(rc);
        std::swap(S.X, S.Y);
        // explicit residuals of the l lowest Ritz pairs
        double worst = 0.0;
        for (int j = 0; j < l; j++) {
            rc = S.Q(S.s1, S.x(j));
            if (rc == ND_OK) rc = S.Qepi(S.s0, S.s1, 1.0, -theta[j], S.x(j), 0.0, nullptr);
            if (rc == ND_OK) rc = S.norm(S.s0, &rq[j]);
            if (rc != ND_OK) return finish(rc);
            worst = std::max(worst, rq[j]);
        }
        if (worst <= tol) { converged = true; break; }
        nlock = 0;
        while (nlock < l && rq[nlock] <= 0.5 * tol) nlock++;   // leading Ritz pairs already well inside the tolerance
        // damp everything above the block's largest Ritz value next time (keep the interval non-degenerate)
        cut = std::min(theta[k - 1], 0.5 * hi);
        if (lextra == 0) cut = std::min(theta[k - 1] * 1.05 + 1e-3, 0.5 * hi);
    }
    if (it > maxit) it = maxit;
    if (theta_rest)
        for (int j = l; j < k; j++) theta_rest[j - l] = theta[j];
    // Rayleigh-Ritz of Q in the span of the l lowest vectors (eq. 2.7): Y_j = Q X_j, M = X^dagger Y
    for (int j = 0; j < l; j++) {
        rc = S.Q(S.y(j), S.x(j));
        if (rc != ND_OK) return finish(rc);
    }
    rc = S.gram(S.X, l, S.Y, l);
    std::vector<double> nuv(l), zq((size_t)2 * l * l);
    if (rc == ND_OK) rc = nd_heev(l, S.h_mat.data(), nuv.data(), zq.data());
    if (rc != ND_OK) return finish(rc);
    std::vector<int> order(l);
    for (int i = 0; i < l; i++) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int a, int b) { return nuv[a] * nuv[a] < nuv[b] * nuv[b]; });
    std::vector<zc> Wq((size_t)l * l);
    for (int j = 0; j < l; j++) {
        nu[j] = nuv[order[j]];
        for (int i = 0; i < l; i++) Wq[(size_t)i * l + j] = zc(zq[2 * ((size_t)i * l + order[j])], zq[2 * ((size_t)i * l + order[j]) + 1]);
    }
    rc = S.rotate((char*)u_out, l, S.X, l, Wq);
    if (rc != ND_OK) return finish(rc);
    for (int j = 0; j < l; j++) {
        char* uj = (char*)u_out + (size_t)j * S.sb;
        rc = S.Qepi(S.s0, uj, 1.0, -nu[j], uj, 0.0, nullptr);   // (Q - nu_j) u_j   (eq. 2.8)
        if (rc == ND_OK) rc = S.norm(S.s0, &resid[j]);
        if (rc != ND_OK) return finish(rc);
    }
    ND_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (!converged) {
        double worst = 0.0;
        for (int j = 0; j < l; j++) worst = std::max(worst, rq[j]);
        nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "lowmodes_compute: max residual of Q^2 %.3e > tol %.3e after %d iterations", worst, tol, it);
        return finish(ND_ERR_NO_CONVERGENCE);
    }
    return finish(ND_OK);
}
