// lowmodes.cu - the low modes of Q and the error control of their projectors (section 2.3, eq. 2.7-2.10).
//
// PAPER.md:L79 says only that the low modes are found "by minimizing the Ritz functional of Q^2" (ref. [13]); no steps
// are given.  DESIGN.md reading R13: any method that delivers small residues; R17: the dynamic choice of l (L110).
// Built here: Chebyshev-filtered block subspace iteration, which minimises the block Ritz functional
// tr(X^dagger Q^2 X) over orthonormal blocks X and is made of exactly the kernels D_N uses (plain stencil, stencil with
// the fused three-term epilogue, grouped Gram / rotation kernels), with the Rayleigh-Ritz step of Q (eq. 2.7) done in
// the WHOLE block so that +nu / -nu partners are never separated by the cut:
//
//   X = k = l_max + lguard Gaussian vectors, orthonormalised
//   repeat:  X_j <- p_d(Q^2) X_j, p_d = the degree-d Chebyshev polynomial that is small on [cut, qnorm^2] and normalised
//                                 to 1 at the lowest Ritz value (scaled three-term recurrence: no overflow in fp32);
//                                 columns whose residue is already far below what the tolerance needs are locked
//            orthonormalise X    (equilibrated Gram matrix, Hermitian eigendecomposition on the host,
//                                 X <- X D^{-1/2} W Lambda^{-1/2}; repeated while the Gram matrix is ill-conditioned)
//            Y = Q X;  H = Y^dagger Y (-> largest Ritz value of Q^2 in the block = next cut);
//            M = X^dagger Y = W diag(nu) W^dagger: Rayleigh-Ritz of Q in the block (2.7); pairs ordered by
//            a_j = ||Q u_j|| = sqrt(nu_j^2 + rho_j^2) (= |nu_j| once converged);  X <- X W
//            Y = Q X;  rho_j = ||Y_j - nu_j X_j||  for every j                                        (2.8)
//            cut l' in [l_min, l_max] at the largest gap of a_j (R17); d_k, kappa_+-, bound           (2.9, 2.10)
//   until the stop rule holds:  rule 0: max_{k < l'} rho_k <= tol      rule 1: max(bound_+, bound_-) <= tol   (L110)
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
    bool done = false;
    for (int sweep = 0; sweep < 60 && !done; sweep++) {
        double off = 0.0;
        for (int p = 0; p < k; p++)
            for (int q = p + 1; q < k; q++) off += std::norm(A[(size_t)p * k + q]);
        if (std::sqrt(off) <= 1e-14 * scale * std::sqrt((double)k)) { done = true; break; }   // off-diagonal Frobenius norm at rounding level
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
    if (!done) {
        // the sweep limit was hit: accept only if the last sweep did bring the off-diagonal part down to rounding level
        double off = 0.0;
        for (int p = 0; p < k; p++)
            for (int q = p + 1; q < k; q++) off += std::norm(A[(size_t)p * k + q]);
        if (!(std::sqrt(off) <= 1e-12 * scale * std::sqrt((double)k))) return ND_ERR_NO_CONVERGENCE;
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

extern "C" int nd_choose_l(int k, const double* abs_nu, int l_min, int l_max, int* l, double* gap) {
    if (!abs_nu || !l || l_min < 1 || l_max < l_min || l_max >= k) return ND_ERR_BAD_ARG;
    for (int i = 1; i < k; i++)
        if (!(abs_nu[i] >= abs_nu[i - 1]) || !(abs_nu[i - 1] >= 0.0)) return ND_ERR_BAD_ARG;   // ascending moduli (NaN fails)
    int best = l_min;
    double best_gap = -1.0;
    for (int c = l_min; c <= l_max; c++) {
        const double g = abs_nu[c] - abs_nu[c - 1];
        if (g > best_gap) { best = c; best_gap = g; }
    }
    *l = best;
    if (gap) *gap = best_gap;
    return ND_OK;
}

namespace {

struct Solver {
    nd_ctx* ctx;
    size_t sb;
    int k;
    double m;
    char *X, *Y, *Z, *s0, *s1;
    double* d_mat;   // 2 k^2 doubles on the device
    std::vector<double> h_mat;
    long long stencils;

    char* x(int j) { return X + (size_t)j * sb; }
    char* y(int j) { return Y + (size_t)j * sb; }

    // Q and the fused-epilogue Q on n columns stored back to back, one launch for all of them (small lattices: the columns fill the machine)
    int Qb(int n, void* out, const void* in) {
        stencils += n;
        return ndi_apply_Q_batch(ctx, n, out, in, m, false, 1, 0, nullptr, 0, nullptr, 0, nullptr);
    }
    int Qepib(int n, void* out, const void* in, double a0, double a1, const void* v1, double a2, const void* v2) {
        stencils += n;
        return ndi_apply_Q_batch(ctx, n, out, in, m, true, a0, a1, v1, a2, v2, 0, nullptr);
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
    // X <- X D^{-1/2} W Lambda^{-1/2} with D = diag(G), D^{-1/2} G D^{-1/2} = W Lambda W^dagger, G = X^dagger X.
    // The column scaling takes the grading of the filtered block (column norms differ by orders of magnitude) out of the
    // eigenproblem; passes are repeated while the equilibrated Gram matrix is ill-conditioned (the loss of orthogonality
    // of one pass is ~ rounding * cond), and the result is refused if it does not get well-conditioned.
    int orthonormalise() {
        std::vector<double> w(k), z((size_t)2 * k * k), dscale(k);
        const double cond_ok = (ctx->prec == 32) ? 30.0 : 1.0e6;
        for (int pass = 0; pass < 5; pass++) {
            int rc = gram(X, k, X, k);
            if (rc != ND_OK) return rc;
            for (int j = 0; j < k; j++) {
                const double g = h_mat[2 * ((size_t)j * k + j)];
                if (!(g > 0.0) || !std::isfinite(g)) return nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "lowmodes: block column %d has norm^2 %g", j, g);
                dscale[j] = 1.0 / std::sqrt(g);
            }
            for (int i = 0; i < k; i++)
                for (int j = 0; j < k; j++) {
                    h_mat[2 * ((size_t)i * k + j)] *= dscale[i] * dscale[j];
                    h_mat[2 * ((size_t)i * k + j) + 1] *= dscale[i] * dscale[j];
                }
            rc = nd_heev(k, h_mat.data(), w.data(), z.data());
            if (rc != ND_OK) return nd_fail(ctx, rc, "lowmodes: Jacobi eigen-solver did not converge on the Gram matrix");
            if (!(w[0] > 0.0) || !std::isfinite(w[0])) return nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "lowmodes: block lost rank (Gram eigenvalue %g)", w[0]);
            const double cond = w[k - 1] / w[0];
            if (pass > 0 && cond < 1.0 + (ctx->prec == 32 ? 1e-4 : 1e-12)) return ND_OK;   // already orthonormal to rounding
            std::vector<zc> C((size_t)k * k);
            for (int j = 0; j < k; j++) {
                const double f = 1.0 / std::sqrt(w[j]);
                for (int i = 0; i < k; i++) C[(size_t)i * k + j] = dscale[i] * f * zc(z[2 * ((size_t)i * k + j)], z[2 * ((size_t)i * k + j) + 1]);
            }
            rc = rotate(Z, k, X, k, C);
            if (rc != ND_OK) return rc;
            std::swap(X, Z);
            if (cond < cond_ok) return ND_OK;
        }
        return nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "lowmodes: the block does not orthonormalise (Gram matrix stays ill-conditioned)");
    }
    // X_j <- p_d(Q^2) X_j for j >= first: scaled Chebyshev recurrence on [lo, hi] (damped), normalised to 1 at `low`
    //   sigma_1 = e/(low - c);  t_1 = (sigma_1/e)(Q^2 - c) t_0
    //   sigma_{i+1} = 1/(2/sigma_1 - sigma_i);  t_{i+1} = (2 sigma_{i+1}/e)(Q^2 - c) t_i - sigma_i sigma_{i+1} t_{i-1}
    // each step = one plain stencil + one stencil with the update in its epilogue (the Clenshaw step's kernel); d even
    int filter(int d, double low, double lo, double hi, int first) {
        const double c = 0.5 * (hi + lo), e = 0.5 * (hi - lo);
        const double sigma1 = e / (low - c);
        const int n = k - first;              // the same polynomial for every column: all of them in each launch
        if (n <= 0) return ND_OK;
        char* P = x(first);                   // t_{i-1}
        char* R = Z + (size_t)first * sb;     // t_i     (Z and Y are free between two Rayleigh-Ritz steps)
        char* tmp = y(first);
        int rc = Qb(n, tmp, P);
        if (rc != ND_OK) return rc;
        rc = Qepib(n, R, tmp, sigma1 / e, -c * sigma1 / e, P, 0.0, nullptr);   // t_1
        if (rc != ND_OK) return rc;
        double sigma = sigma1;
        for (int i = 1; i < d; i++) {
            const double sn = 1.0 / (2.0 / sigma1 - sigma);
            rc = Qb(n, tmp, R);
            if (rc != ND_OK) return rc;
            rc = Qepib(n, P, tmp, 2.0 * sn / e, -2.0 * sn * c / e, R, -sigma * sn, P);   // t_{i+1} over t_{i-1}
            if (rc != ND_OK) return rc;
            std::swap(P, R);
            sigma = sn;
        }
        // d even: t_d sits in X again
        return ND_OK;
    }
};

}  // namespace

extern "C" size_t nd_lowmodes_work_spinors(int l_max, int lguard) { return (size_t)3 * (l_max + lguard) + 2; }

extern "C" int nd_lowmodes_compute(nd_ctx* ctx, int l_min, int l_max, int lguard, int degree, double m, int stop_rule, double tol,
                                   int maxit, unsigned long long seed, void* u_out, double* nu, double* resid, int* l_chosen,
                                   double kappa[2], double bound[2], void* work, long long* stats) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (l_min < 1 || l_max < l_min || lguard < 1 || l_max + lguard > ND_MAX_BLOCK_L || degree < 2 || maxit < 1 || !(tol > 0.0) ||
        (stop_rule != 0 && stop_rule != 1) || !u_out || !nu || !resid || !l_chosen || !work)
        return nd_fail(ctx, ND_ERR_BAD_ARG, "lowmodes_compute: bad argument (1 <= l_min <= l_max, lguard >= 1, l_max + lguard <= %d, degree >= 2)",
                       ND_MAX_BLOCK_L);
    if (!ctx->gauge_set) return nd_fail(ctx, ND_ERR_BAD_STATE, "lowmodes_compute: gauge field not set");
    if (12 * ctx->V < l_max + lguard) return nd_fail(ctx, ND_ERR_BAD_ARG, "lowmodes_compute: block larger than the space");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    Solver S;
    S.ctx = ctx;
    S.sb = nd_spinor_bytes(ctx);
    S.k = l_max + lguard;
    S.m = m;
    S.stencils = 0;
    const int k = S.k;
    S.X = (char*)work;
    S.Y = S.X + (size_t)k * S.sb;
    S.Z = S.Y + (size_t)k * S.sb;
    S.s0 = S.Z + (size_t)k * S.sb;
    S.s1 = S.s0 + S.sb;
    S.d_mat = nullptr;
    ND_CUDA(ctx, cudaMalloc((void**)&S.d_mat, (size_t)2 * k * k * sizeof(double)));
    const int d = degree + (degree & 1);
    const double hi = (std::fabs(4.0 + m) + 4.0) * (std::fabs(4.0 + m) + 4.0);   // ||Q||^2 <= (|4+m|+4)^2 (R6)
    int rc = ND_OK, it = 0, lp = l_min;
    bool converged = false;
    std::vector<double> theta(k), z((size_t)2 * k * k), nuv(k), rho(k, 0.0), dk(k, 0.0), amod(k), tau(k), Hm;
    double kap[2] = {INFINITY, INFINITY}, bnd[2] = {INFINITY, INFINITY};
    auto finish = [&](int code) {
        cudaFree(S.d_mat);
        if (stats) { stats[0] = it; stats[1] = S.stencils; }
        return code;
    };
    for (int j = 0; j < k; j++) {
        rc = nd_gaussian(ctx, S.x(j), seed + (unsigned long long)j);
        if (rc != ND_OK) return finish(rc);
    }
    rc = S.orthonormalise();
    if (rc != ND_OK) return finish(rc);
    double cut = -1.0, low = 0.0;   // unknown before the first Rayleigh-Ritz step
    int nlock = 0;
    for (it = 0; it <= maxit; it++) {
        if (it > 0) {
            rc = S.filter(d, low, cut, hi, nlock);
            if (rc == ND_OK) rc = S.orthonormalise();
            if (rc != ND_OK) return finish(rc);
        }
        // Y = Q X;  H = Y^dagger Y = X^dagger Q^2 X: its extreme eigenvalues are the extreme Ritz values of Q^2 in the block
        rc = S.Qb(k, S.Y, S.X);
        if (rc == ND_OK) rc = S.gram(S.Y, k, S.Y, k);
        if (rc != ND_OK) return finish(rc);
        Hm.assign(S.h_mat.begin(), S.h_mat.end());
        rc = nd_heev(k, Hm.data(), theta.data(), z.data());
        // Rayleigh-Ritz of Q in the whole block (eq. 2.7): M = X^dagger Q X = W diag(nu) W^dagger
        if (rc == ND_OK) rc = S.gram(S.X, k, S.Y, k);
        if (rc == ND_OK) rc = nd_heev(k, S.h_mat.data(), nuv.data(), z.data());
        if (rc != ND_OK) return finish(rc == ND_ERR_NO_CONVERGENCE ? nd_fail(ctx, rc, "lowmodes: Jacobi eigen-solver did not converge") : rc);
        // Order the Ritz pairs by the Rayleigh quotient of Q^2, a_j^2 = ||Q u_j||^2 = w_j^dagger H w_j (= nu_j^2 + rho_j^2):
        // for a converged pair a_j = |nu_j|, while a spurious small Ritz value of the indefinite Q (a vector mixing +nu and
        // -nu modes whose partner combination is not in the block yet) has a large residue and goes to the end (R17).
        for (int j = 0; j < k; j++) {
            double t = 0.0;
            for (int a = 0; a < k; a++) {
                zc acc(0.0, 0.0);
                for (int b = 0; b < k; b++)
                    acc += zc(Hm[2 * ((size_t)a * k + b)], Hm[2 * ((size_t)a * k + b) + 1]) * zc(z[2 * ((size_t)b * k + j)], z[2 * ((size_t)b * k + j) + 1]);
                t += (std::conj(zc(z[2 * ((size_t)a * k + j)], z[2 * ((size_t)a * k + j) + 1])) * acc).real();
            }
            tau[j] = t;
        }
        std::vector<int> order(k);
        for (int i = 0; i < k; i++) order[i] = i;
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return tau[a] < tau[b]; });
        std::vector<zc> W((size_t)k * k);
        for (int j = 0; j < k; j++) {
            nu[j] = nuv[order[j]];
            for (int i = 0; i < k; i++) W[(size_t)i * k + j] = zc(z[2 * ((size_t)i * k + order[j])], z[2 * ((size_t)i * k + order[j]) + 1]);
        }
        rc = S.rotate(S.Z, k, S.X, k, W);
        if (rc != ND_OK) return finish(rc);
        std::swap(S.X, S.Z);
        // residues rho_j = ||(Q - nu_j) u_j|| of the whole block (eq. 2.8), Q u_j recomputed on the rotated vectors
        rc = S.Qb(k, S.Y, S.X);
        if (rc == ND_OK) rc = ndi_block_resid(ctx, k, S.X, S.Y, nu, rho.data());
        if (rc != ND_OK) return finish(rc);
        for (int j = 0; j < k; j++) {
            resid[j] = rho[j];
            amod[j] = std::sqrt(nu[j] * nu[j] + rho[j] * rho[j]);
        }
        // the measured residues replace the small-matrix estimate; keep the list ascending for the gap rule (changes
        // nothing for converged pairs, clamps the noise of unconverged guard pairs)
        for (int j = 1; j < k; j++) amod[j] = std::max(amod[j], amod[j - 1]);
        // error control: the cut, d_k from the guard moduli (both signs) and the opposite-sign values
        rc = nd_choose_l(k, amod.data(), l_min, l_max, &lp, nullptr);
        if (rc != ND_OK) return finish(nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "lowmodes: Ritz values not finite"));
        bool signs_ok = true;
        for (int j = 0; j < lp; j++) signs_ok = signs_ok && nu[j] != 0.0;
        if (signs_ok) {
            std::vector<double> rest((size_t)2 * (k - lp));
            for (int j = lp; j < k; j++) { rest[2 * (j - lp)] = amod[j]; rest[2 * (j - lp) + 1] = -amod[j]; }
            nd_projector_error(lp, nu, rho.data(), (int)rest.size(), rest.data(), kap, bnd, dk.data());
        } else {
            kap[0] = kap[1] = bnd[0] = bnd[1] = INFINITY;
        }
        double worst = 0.0;
        for (int j = 0; j < lp; j++) worst = std::max(worst, rho[j]);
        converged = (stop_rule == 0) ? (worst <= tol) : (std::max(bnd[0], bnd[1]) <= tol);
        if (converged || it == maxit) break;
        // lock the leading columns whose residue is already far below what the stop rule needs from them
        nlock = 0;
        while (nlock < lp) {
            const double need = (stop_rule == 0) ? 0.5 * tol : 0.25 * tol * dk[nlock] / std::sqrt((double)l_max);
            if (!(rho[nlock] <= need)) break;
            nlock++;
        }
        // damp everything above the block's largest Ritz value of Q^2 next time, normalise at its lowest one
        cut = std::min(theta[k - 1], 0.5 * hi);
        low = std::max(0.0, std::min(theta[0], 0.5 * cut));
    }
    *l_chosen = lp;
    if (kappa) { kappa[0] = kap[0]; kappa[1] = kap[1]; }
    if (bound) { bound[0] = bnd[0]; bound[1] = bnd[1]; }
    rc = nd_cuda_check(ctx, cudaMemcpyAsync(u_out, S.X, (size_t)l_max * S.sb, cudaMemcpyDeviceToDevice, ctx->stream), "lowmodes copy-out");
    if (rc == ND_OK) rc = nd_cuda_check(ctx, cudaStreamSynchronize(ctx->stream), "lowmodes sync");
    if (rc != ND_OK) return finish(rc);
    if (!converged) {
        nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "lowmodes_compute: after %d iterations l' = %d, max residue %.3e, kappa = (%.3e, %.3e), stop rule %d not met (tol %.3e)",
                it, lp, *std::max_element(rho.begin(), rho.begin() + lp), kap[0], kap[1], stop_rule, tol);
        return finish(ND_ERR_NO_CONVERGENCE);
    }
    return finish(ND_OK);
}

// ------------------------------------------------------------------------ index by zero-mode counting
// PAPER.md:L146 ("the calculation of the index of our Neuberger-Dirac operator via zero-mode counting").  D_N obeys the
// Ginsparg-Wilson relation, so D_N^dagger D_N commutes with gamma5 and its zero modes have a definite chirality.  On the
// sector gamma5 = sigma,
//     D_N^dagger D_N / (2 c^2) = B_sigma = P_sigma (1 + gamma5 sign(Q)) P_sigma,   P_sigma = (1 + sigma gamma5)/2,
// with spectrum in [0, 2].  For each sigma the lowest nvec eigenvalues of B_sigma are found by the block machinery above:
//   X = nvec Gaussian vectors projected to the sector, orthonormalised
//   repeat:  X_j <- p_d(B_sigma) X_j   (scaled Chebyshev recurrence, small on [cut, 2], 1 at the lowest Ritz value; one sign-
//                                       function application = 2n+1 stencils per degree, nd_apply_DNm's launch sequence)
//            orthonormalise;  Y = B_sigma X;  H = X^dagger Y = W diag(theta) W^dagger;  X <- X W, Y <- Y W;
//            r_j = ||Y_j - theta_j X_j||: an eigenvalue of B_sigma lies within r_j of theta_j
//   until every pair is decided: zero mode (theta_j + r_j <= zero_tol) or not (theta_j - r_j > zero_tol), the lowest pair
//   that is not has r_j <= 0.1 theta_j (the block has converged onto the low end of the spectrum), and at least one pair is
//   not a zero mode (else the block may be smaller than the kernel: ND_ERR_BAD_ARG, enlarge nvec).
// n_sigma = number of zero modes of chirality sigma, index = n_+ - n_-.
namespace {

struct SectorOp {
    Solver* S;
    int sigma;
    char* sw;          // 3 work spinors of the sign function
    long long signs;   // sign-function applications
    // out = P_sigma (pa in + pb gamma5 sign(Q) in) + pc out
    int apply(void* out, const void* in, double pa, double pb, double pc, char* tmp) {
        signs++;
        int rc = ndi_apply_DNm(S->ctx, tmp, in, pa, pb, sw, 0);
        if (rc != ND_OK) return rc;
        return ndi_chiral_combine(S->ctx, sigma, out, tmp, pc);
    }
    // X_j <- p_d(B) X_j on [lo, hi] damped, normalised to 1 at `low` (the recurrence of Solver::filter with B for Q^2)
    int filter(int d, double low, double lo, double hi) {
        const double c = 0.5 * (hi + lo), e = 0.5 * (hi - lo);
        const double sigma1 = e / (low - c);
        for (int j = 0; j < S->k; j++) {
            char* P = S->x(j);
            char* R = S->s0;
            // t_1 = (sigma_1/e)(B - c) t_0
            int rc = apply(R, P, (1.0 - c) * sigma1 / e, sigma1 / e, 0.0, S->s1);
            if (rc != ND_OK) return rc;
            double sg = sigma1;
            for (int i = 1; i < d; i++) {
                const double sn = 1.0 / (2.0 / sigma1 - sg);
                // t_{i+1} = (2 sn/e)(B - c) t_i - sg sn t_{i-1}, written over t_{i-1}
                rc = apply(P, R, (1.0 - c) * 2.0 * sn / e, 2.0 * sn / e, -sg * sn, S->s1);
                if (rc != ND_OK) return rc;
                std::swap(P, R);
                sg = sn;
            }
            // d even: t_d sits in x(j) again
        }
        return ND_OK;
    }
};

}  // namespace

extern "C" size_t nd_index_work_spinors(int nvec) { return (size_t)3 * nvec + 5; }

extern "C" int nd_index_count(nd_ctx* ctx, int nvec, int degree, double zero_tol, int maxit, unsigned long long seed, int counts[2],
                              double* evals, double* resid, void* work, long long* stats) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (nvec < 2 || nvec > ND_MAX_BLOCK_L || degree < 2 || maxit < 1 || !(zero_tol > 0.0 && zero_tol < 1.0) || !counts || !evals ||
        !resid || !work)
        return nd_fail(ctx, ND_ERR_BAD_ARG, "index_count: bad argument (2 <= nvec <= %d, degree >= 2, 0 < zero_tol < 1)", ND_MAX_BLOCK_L);
    if (!ctx->gauge_set || !ctx->poly_set) return nd_fail(ctx, ND_ERR_BAD_STATE, "index_count: gauge field / sign polynomial not set");
    if (6 * ctx->V < nvec) return nd_fail(ctx, ND_ERR_BAD_ARG, "index_count: block larger than a chirality sector");
    ND_CUDA(ctx, cudaSetDevice(ctx->device));
    Solver S;
    S.ctx = ctx;
    S.sb = nd_spinor_bytes(ctx);
    S.k = nvec;
    S.m = ctx->m_sign;
    S.stencils = 0;
    const int k = nvec;
    char* base = (char*)work;
    S.s0 = base + (size_t)3 * k * S.sb;
    S.s1 = S.s0 + S.sb;
    S.d_mat = nullptr;
    ND_CUDA(ctx, cudaMalloc((void**)&S.d_mat, (size_t)2 * k * k * sizeof(double)));
    SectorOp B;
    B.S = &S;
    B.sw = S.s1 + S.sb;
    B.signs = 0;
    const int d = degree + (degree & 1);
    long long its = 0;
    auto finish = [&](int code) {
        cudaFree(S.d_mat);
        if (stats) { stats[0] = its; stats[1] = B.signs; }
        return code;
    };
    std::vector<double> theta(k), z((size_t)2 * k * k), rho(k);
    for (int sec = 0; sec < 2; sec++) {
        B.sigma = (sec == 0) ? +1 : -1;
        S.X = base;
        S.Y = base + (size_t)k * S.sb;
        S.Z = base + (size_t)2 * k * S.sb;
        int rc = ND_OK;
        for (int j = 0; j < k && rc == ND_OK; j++) {
            rc = nd_gaussian(ctx, S.s0, seed + (unsigned long long)(sec * k + j));
            if (rc == ND_OK) rc = ndi_chiral_combine(ctx, B.sigma, S.x(j), S.s0, 0.0);
        }
        if (rc == ND_OK) rc = S.orthonormalise();
        if (rc != ND_OK) return finish(rc);
        double cut = 2.0, low = 0.0;
        bool decided = false;
        int nzero = 0;
        for (int it = 0; it <= maxit; it++) {
            if (it > 0) {
                rc = B.filter(d, low, cut, 2.0);
                if (rc == ND_OK) rc = S.orthonormalise();
                if (rc != ND_OK) return finish(rc);
                its++;
            }
            for (int j = 0; j < k && rc == ND_OK; j++) rc = B.apply(S.y(j), S.x(j), 1.0, 1.0, 0.0, S.s1);
            if (rc == ND_OK) rc = S.gram(S.X, k, S.Y, k);
            if (rc == ND_OK) rc = nd_heev(k, S.h_mat.data(), theta.data(), z.data());
            if (rc != ND_OK) return finish(rc == ND_ERR_NO_CONVERGENCE ? nd_fail(ctx, rc, "index_count: Jacobi eigen-solver did not converge") : rc);
            std::vector<zc> W((size_t)k * k);
            for (size_t i = 0; i < (size_t)k * k; i++) W[i] = zc(z[2 * i], z[2 * i + 1]);
            rc = S.rotate(S.Z, k, S.X, k, W);
            if (rc != ND_OK) return finish(rc);
            std::swap(S.X, S.Z);
            rc = S.rotate(S.Z, k, S.Y, k, W);
            if (rc != ND_OK) return finish(rc);
            std::swap(S.Y, S.Z);
            rc = ndi_block_resid(ctx, k, S.X, S.Y, theta.data(), rho.data());
            if (rc != ND_OK) return finish(rc);
            nzero = 0;
            int nrest = 0;
            for (int j = 0; j < k; j++) {
                evals[sec * k + j] = theta[j];
                resid[sec * k + j] = rho[j];
                if (theta[j] + rho[j] <= zero_tol) nzero++;
                else if (theta[j] - rho[j] > zero_tol) nrest++;
            }
            // every pair decided, and the block has settled on the LOW end of the spectrum: the lowest non-zero pair is located
            // to 10 % (a block of unconverged vectors has theta ~ 1 and residues ~ 0.3: "no zero modes" only by accident)
            decided = (nzero + nrest == k) && nzero < k && rho[nzero] <= 0.1 * theta[nzero];
            if (nzero == k) decided = true;   // reported below
            if (decided || it == maxit) break;
            // damp everything above the block's largest Ritz value next time; keep the damped interval off the lowest values
            cut = std::max(theta[k - 1], 4.0 * zero_tol);
            low = std::max(0.0, std::min(theta[0], 0.5 * cut));
            if (!(cut < 1.9)) cut = 1.9;
        }
        counts[sec] = nzero;
        if (!decided) {
            nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "index_count: sector %+d undecided after %d iterations (lowest Ritz value %.3e, residue %.3e, zero_tol %.3e)",
                    B.sigma, maxit, theta[0], rho[0], zero_tol);
            return finish(ND_ERR_NO_CONVERGENCE);
        }
        if (nzero == k) {
            nd_fail(ctx, ND_ERR_BAD_ARG, "index_count: all %d vectors of sector %+d are zero modes: the block may be smaller than the kernel, enlarge nvec", k,
                    B.sigma);
            return finish(ND_ERR_BAD_ARG);
        }
    }
    return finish(ND_OK);
}
