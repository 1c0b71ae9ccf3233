// lowmodes.cu - the l lowest eigenpairs of Q^2 and the Rayleigh-Ritz step of Q in their span.
#include "nd_internal.cuh"

extern "C" int nd_lowmodes_compute(nd_ctx* ctx, int l, int lextra, int degree, double m, double tol, int maxit,
                                   unsigned long long seed, void* u_out, double* nu, double* resid, void* work,
                                   long long* stats) {
    if (!ctx) return ND_ERR_BAD_ARG;
    return nd_fail(ctx, ND_ERR_BAD_STATE, "lowmodes_compute: under construction");
}
