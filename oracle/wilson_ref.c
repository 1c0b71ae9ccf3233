/* Oracle (TEST INFRASTRUCTURE, not product code): plain-C restatement of eq. 2.1-2.2 of arXiv:1010.5636
 * (PAPER.md:L35-42), used where the numpy oracle (oracle/wilson.py) is too slow: full-size parity
 * samples, the D_N recipe at 16^3x32, eigsh on Q^2, and the timed `cpu_baseline` of bench.py.
 *
 *   D_W phi(x) = (4+m) phi(x) - 1/2 sum_{mu=0}^{3} [ U_mu(x) (1-gamma_mu) phi(x+mu^)
 *                                                   + U_mu(x-mu^)^dagger (1+gamma_mu) phi(x-mu^) ],  Q = gamma5 D_W
 *
 * Written as the definition: a loop over sites, full 4x4 gamma matrices, full 3x3 complex links, no
 * spin-projection shortcut, no compression, no blocking, no intrinsics.  It shares nothing with the CUDA
 * path (own file, no common header).  It is itself pinned against oracle/wilson.py and the same
 * invariants (tests/test_oracle_c.py).
 *
 * Layout (C order, complex128 = double _Complex):
 *   psi[x0][x1][x2][x3][spin 4][colour 3]         U[mu 4][x0][x1][x2][x3][row 3][col 3]
 * bc_time = +1 / -1: sign carried by hops across the x0 = T-1 <-> 0 seam (reading R1).
 */
#include <complex.h>
#include <stddef.h>

typedef double _Complex cplx;

static cplx GAM[4][4][4];
static double G5[4];
static int gam_ready = 0;

/* Chiral basis, reading R2: gamma_0 = [[0,-1],[-1,0]], gamma_k = [[0,-i sigma_k],[i sigma_k,0]],
 * gamma_5 = gamma_0 gamma_1 gamma_2 gamma_3 = diag(1,1,-1,-1). */
static void init_gamma(void)
{
    const cplx sig[3][2][2] = {{{0, 1}, {1, 0}}, {{0, -I}, {I, 0}}, {{1, 0}, {0, -1}}};
    for (int mu = 0; mu < 4; mu++)
        for (int s = 0; s < 4; s++)
            for (int t = 0; t < 4; t++) GAM[mu][s][t] = 0;
    for (int i = 0; i < 2; i++) {
        GAM[0][i][2 + i] = -1;
        GAM[0][2 + i][i] = -1;
    }
    for (int k = 0; k < 3; k++)
        for (int i = 0; i < 2; i++)
            for (int j = 0; j < 2; j++) {
                GAM[k + 1][i][2 + j] = -I * sig[k][i][j];
                GAM[k + 1][2 + i][j] = I * sig[k][i][j];
            }
    G5[0] = G5[1] = 1.0;
    G5[2] = G5[3] = -1.0;
    gam_ready = 1;
}

static size_t site_index(const int *d, int x0, int x1, int x2, int x3)
{
    return (((size_t)x0 * d[1] + x1) * d[2] + x2) * d[3] + x3;
}

/* out = Q psi.  out must not alias psi. */
void wd_apply_Q(const cplx *psi, const cplx *U, cplx *out, const int *dims, double m, int bc_time)
{
    if (!gam_ready) init_gamma();
    const size_t V = (size_t)dims[0] * dims[1] * dims[2] * dims[3];
    const long n0 = dims[0];
#pragma omp parallel for schedule(static)
    for (long x0 = 0; x0 < n0; x0++)
        for (int x1 = 0; x1 < dims[1]; x1++)
            for (int x2 = 0; x2 < dims[2]; x2++)
                for (int x3 = 0; x3 < dims[3]; x3++) {
                    const int x[4] = {(int)x0, x1, x2, x3};
                    const size_t ix = site_index(dims, x[0], x[1], x[2], x[3]);
                    cplx acc[4][3];
                    for (int s = 0; s < 4; s++)
                        for (int a = 0; a < 3; a++) acc[s][a] = (4.0 + m) * psi[ix * 12 + s * 3 + a];
                    for (int mu = 0; mu < 4; mu++) {
                        int xf[4] = {x[0], x[1], x[2], x[3]}, xb[4] = {x[0], x[1], x[2], x[3]};
                        double pf = 1.0, pb = 1.0;
                        xf[mu] = x[mu] + 1;
                        if (xf[mu] == dims[mu]) {
                            xf[mu] = 0;
                            if (mu == 0) pf = bc_time;
                        }
                        xb[mu] = x[mu] - 1;
                        if (xb[mu] < 0) {
                            xb[mu] = dims[mu] - 1;
                            if (mu == 0) pb = bc_time;
                        }
                        const size_t iF = site_index(dims, xf[0], xf[1], xf[2], xf[3]);
                        const size_t iB = site_index(dims, xb[0], xb[1], xb[2], xb[3]);
                        const cplx *Uf = U + ((size_t)mu * V + ix) * 9; /* U_mu(x)      */
                        const cplx *Ub = U + ((size_t)mu * V + iB) * 9; /* U_mu(x-mu^)  */
                        cplx cf[4][3], cb[4][3];                        /* colour-multiplied neighbours */
                        for (int s = 0; s < 4; s++)
                            for (int a = 0; a < 3; a++) {
                                cplx f = 0, b = 0;
                                for (int c = 0; c < 3; c++) {
                                    f += Uf[a * 3 + c] * psi[iF * 12 + s * 3 + c];
                                    b += conj(Ub[c * 3 + a]) * psi[iB * 12 + s * 3 + c];
                                }
                                cf[s][a] = f;
                                cb[s][a] = b;
                            }
                        for (int s = 0; s < 4; s++)
                            for (int a = 0; a < 3; a++) {
                                cplx f = cf[s][a], b = cb[s][a]; /* (1 -+ gamma_mu) in spin space */
                                for (int t = 0; t < 4; t++) {
                                    f -= GAM[mu][s][t] * cf[t][a];
                                    b += GAM[mu][s][t] * cb[t][a];
                                }
                                acc[s][a] -= 0.5 * (pf * f + pb * b);
                            }
                    }
                    for (int s = 0; s < 4; s++)
                        for (int a = 0; a < 3; a++) out[ix * 12 + s * 3 + a] = G5[s] * acc[s][a];
                }
}

int wd_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}
