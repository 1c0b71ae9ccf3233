// solver.cu - the massive Neuberger-Dirac operator and its inversion (eq. 2.12).
//
// PAPER.md names D_N^m only through the bound (2.12), whose factor (2/a)(1 + s - a m/2) fixes it (R16) as
//     D_N^m = (1 - abar m / 2) D_N + m,   abar = a/(1+s),   D_N = (1/abar)(1 + gamma5 sign(Q))
//           = (1/abar + m/2) + (1/abar - m/2) gamma5 sign(Q)
// (the convention of the paper's ref. [10]); 1/abar is the caller's `prefactor` (R5).  One application costs
// exactly one sign-function application: the two scalars go into the D_N epilogue of the last projection kernel.
//
// nd_solve_DNm solves D_N^m x = b by conjugate gradients on the normal equations (the standard use of the operator,
// PAPER.md:L146 "inversion"), with D_N^m^dagger = gamma5 D_N^m gamma5.  Every vector operation is a kernel of blas.cu;
// per iteration two operator applications and two host reads of a reduction (the step lengths).
#include <cmath>

#include "nd_internal.cuh"

extern "C" int nd_apply_DNm(nd_ctx* ctx, void* out, const void* in, double prefactor, double mq, void* work, int use_graph) {
    if (!ctx) return ND_ERR_BAD_ARG;
    return ndi_apply_DNm(ctx, out, in, prefactor + 0.5 * mq, prefactor - 0.5 * mq, work, use_graph);
}

extern "C" int nd_solve_DNm(nd_ctx* ctx, void* x, const void* b, double prefactor, double mq, double tol, int maxit, void* work,
                            double* relres, int* iters) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (!x || !b || !work || x == b || !(tol > 0.0) || maxit < 1)
        return nd_fail(ctx, ND_ERR_BAD_ARG, "solve_DNm: null / aliased argument, tol <= 0 or maxit < 1");
    const size_t sb = nd_spinor_bytes(ctx);
    char* w = (char*)work;
    void *r = w, *p = w + sb, *t = w + 2 * sb, *q = w + 3 * sb, *g = w + 4 * sb, *sw = w + 5 * sb;   // + 3 for the sign
    const double pa = prefactor + 0.5 * mq, pb = prefactor - 0.5 * mq;
    const double one[2] = {1.0, 0.0};
    int rc;
    // out = D^dagger in = gamma5 D gamma5 in   (through g; out != in)
    auto Ddag = [&](void* out, const void* in) -> int {
        int e = nd_gamma5(ctx, g, in);
        if (e == ND_OK) e = ndi_apply_DNm(ctx, out, g, pa, pb, sw, 1);
        if (e == ND_OK) e = nd_gamma5(ctx, out, out);
        return e;
    };
    double bb = 0.0, rr = 0.0;
    rc = nd_norm2(ctx, b, &bb);
    if (rc != ND_OK) return rc;
    ND_CUDA(ctx, cudaMemsetAsync(x, 0, sb, ctx->stream));
    if (iters) *iters = 0;
    if (bb == 0.0) {
        if (relres) *relres = 0.0;
        return ND_OK;
    }
    rc = Ddag(r, b);                 // x = 0: the residual of the normal equations is D^dagger b
    if (rc == ND_OK) rc = nd_copy(ctx, p, r);
    if (rc == ND_OK) rc = nd_norm2(ctx, r, &rr);
    if (rc != ND_OK) return rc;
    const double stop = tol * tol * rr;
    int it = 0;
    bool ok = rr <= 0.0;
    while (!ok && it < maxit) {
        rc = ndi_apply_DNm(ctx, t, p, pa, pb, sw, 1);          // t = D p
        if (rc == ND_OK) rc = Ddag(q, t);                      // q = D^dagger D p
        double tt = 0.0;
        if (rc == ND_OK) rc = nd_norm2(ctx, t, &tt);           // <p, A p> = |D p|^2
        if (rc != ND_OK) return rc;
        if (!(tt > 0.0)) return nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "solve_DNm: breakdown (|D p| = 0)");
        const double alpha = rr / tt;
        const double pal[2] = {alpha, 0.0}, mal[2] = {-alpha, 0.0};
        rc = nd_axpy(ctx, pal, p, x);
        if (rc == ND_OK) rc = nd_axpy(ctx, mal, q, r);
        double rn = 0.0;
        if (rc == ND_OK) rc = nd_norm2(ctx, r, &rn);
        if (rc != ND_OK) return rc;
        it++;
        if (rn <= stop) { rr = rn; ok = true; break; }
        const double beta[2] = {rn / rr, 0.0};
        rc = nd_scale(ctx, beta, p);                           // p = r + beta p
        if (rc == ND_OK) rc = nd_axpy(ctx, one, r, p);
        if (rc != ND_OK) return rc;
        rr = rn;
    }
    if (iters) *iters = it;
    // true residual |b - D x| / |b|
    rc = ndi_apply_DNm(ctx, t, x, pa, pb, sw, 1);
    const double m1[2] = {-1.0, 0.0};
    if (rc == ND_OK) rc = nd_scale(ctx, m1, t);
    if (rc == ND_OK) rc = nd_axpy(ctx, one, b, t);
    double res = 0.0;
    if (rc == ND_OK) rc = nd_norm2(ctx, t, &res);
    if (rc != ND_OK) return rc;
    if (relres) *relres = std::sqrt(res / bb);
    if (!ok) return nd_fail(ctx, ND_ERR_NO_CONVERGENCE, "solve_DNm: %d iterations, |D^dagger r|/|D^dagger b| = %.3e > tol %.3e", it, std::sqrt(rr / (stop / (tol * tol))), tol);
    return ND_OK;
}

// Mixed precision ("fp32-inner / fp64-outer"): iterative refinement.  The fp64 context owns x, b and
// the residual r = b - D x, recomputed in fp64 once per outer step; the correction D e = r is solved in the fp32 context
// (same lattice, gauge field and polynomial) to a loose tolerance and added in fp64.
extern "C" int nd_solve_DNm_mixed(nd_ctx* ctx64, nd_ctx* ctx32, void* x, const void* b, double prefactor, double mq, double tol,
                                  double inner_tol, int max_outer, int max_inner, void* work64, void* work32, double* relres,
                                  int* stats) {
    if (!ctx64 || !ctx32) return ND_ERR_BAD_ARG;
    if (ctx64->prec != 64 || ctx32->prec != 32 || ctx64->V != ctx32->V || ctx64->device != ctx32->device)
        return nd_fail(ctx64, ND_ERR_BAD_ARG, "solve_DNm_mixed: needs an fp64 and an fp32 context of the same lattice and device");
    for (int i = 0; i < 4; i++)
        if (ctx64->dims[i] != ctx32->dims[i]) return nd_fail(ctx64, ND_ERR_BAD_ARG, "solve_DNm_mixed: lattices differ");
    if (!x || !b || x == b || !work64 || !work32 || !(tol > 0.0) || !(inner_tol > 0.0) || max_outer < 1 || max_inner < 1)
        return nd_fail(ctx64, ND_ERR_BAD_ARG, "solve_DNm_mixed: bad argument");
    const size_t sb64 = nd_spinor_bytes(ctx64), sb32 = nd_spinor_bytes(ctx32);
    char* w64 = (char*)work64;
    char* w32 = (char*)work32;
    void *r = w64, *t = w64 + sb64, *e64 = w64 + 2 * sb64, *sw = w64 + 3 * sb64;   // 6 fp64 spinors
    void *r32 = w32, *e32 = w32 + sb32, *iw = w32 + 2 * sb32;                      // 2 + 8 fp32 spinors
    const double pa = prefactor + 0.5 * mq, pb = prefactor - 0.5 * mq;
    const double one[2] = {1.0, 0.0}, m1[2] = {-1.0, 0.0};
    int outer = 0, inner_total = 0, rc;
    double bb = 0.0, rr = 0.0;
    rc = nd_norm2(ctx64, b, &bb);
    if (rc != ND_OK) return rc;
    ND_CUDA(ctx64, cudaMemsetAsync(x, 0, sb64, ctx64->stream));
    rc = nd_copy(ctx64, r, b);
    if (rc != ND_OK) return rc;
    rr = bb;
    bool ok = bb == 0.0;
    while (!ok && outer < max_outer) {
        rc = nd_convert_spinor(ctx64, r32, 32, r, 64);
        if (rc != ND_OK) return rc;
        ND_CUDA(ctx64, cudaStreamSynchronize(ctx64->stream));        // the fp32 context may run on another stream
        int it = 0;
        double ires = 0.0;
        rc = nd_solve_DNm(ctx32, e32, r32, prefactor, mq, inner_tol, max_inner, iw, &ires, &it);   // synchronises
        if (rc != ND_OK && rc != ND_ERR_NO_CONVERGENCE) return nd_fail(ctx64, rc, "solve_DNm_mixed: inner solve: %s", nd_last_error(ctx32));
        inner_total += it;
        rc = nd_convert_spinor(ctx64, e64, 64, e32, 32);
        if (rc == ND_OK) rc = nd_axpy(ctx64, one, e64, x);
        if (rc == ND_OK) rc = ndi_apply_DNm(ctx64, t, x, pa, pb, sw, 1);   // r = b - D x in fp64
        if (rc == ND_OK) rc = nd_copy(ctx64, r, b);
        if (rc == ND_OK) rc = nd_axpy(ctx64, m1, t, r);
        if (rc == ND_OK) rc = nd_norm2(ctx64, r, &rr);
        if (rc != ND_OK) return rc;
        outer++;
        ok = rr <= tol * tol * bb;
    }
    if (relres) *relres = bb > 0.0 ? std::sqrt(rr / bb) : 0.0;
    if (stats) { stats[0] = outer; stats[1] = inner_total; }
    if (!ok) return nd_fail(ctx64, ND_ERR_NO_CONVERGENCE, "solve_DNm_mixed: |b - D x|/|b| = %.3e > tol %.3e after %d outer steps", std::sqrt(rr / bb), tol, outer);
    return ND_OK;
}
