/* nd_b200.h - C-ABI boundary of the B200-native Wilson-Dirac / Neuberger-Dirac hot path of
 * arXiv:1010.5636 ("Implementation of the Neuberger-Dirac operator on GPUs", PAPER.md).
 *
 * Every step behind these calls runs in hand-written CUDA kernels for sm_100a (csrc/ of the package).
 * There is no CPU fallback: without a CUDA device nd_create() fails with ND_ERR_CUDA.
 *
 * Conventions
 * -----------
 *  - Opaque context; EVERY call returns an int status (ND_OK = 0, negative = error).  No exceptions, no
 *    global state (one exception, stated there: the static scratch array of nd_dot_static).  nd_last_error(ctx) gives a
 *    human-readable message owned by the context.
 *  - Field memory is CALLER-OWNED DEVICE memory (e.g. torch tensors' data_ptr()).  A device spinor occupies
 *    nd_spinor_bytes(ctx) bytes and must be 16-byte aligned.  The context owns only: the compressed gauge
 *    field, reduction scratch, polynomial coefficients, a *pointer* to the caller's low-mode block.
 *  - Work is enqueued on the cudaStream_t given to nd_create (0 = legacy default stream).  Calls that return
 *    host scalars synchronise that stream; everything else is asynchronous.
 *  - "host AoS" = canonical site-major arrays, x3 fastest:
 *        spinor  psi[x0][x1][x2][x3][spin 4][colour 3]           complex (re, im interleaved)
 *        links   U[mu 4][x0][x1][x2][x3][row 3][col 3]           complex
 *    dims = (L0, L1, L2, L3) with L0 the time extent T (mu = 0 is time).
 *  - "device SoA" = the library's own layout: planes of 128-bit words,
 *        fp32: 6 planes of float4 [V]   (plane p = reals 4p..4p+3 of the 24 reals spin-major)
 *        fp64: 12 planes of double2 [V] (plane p = complex component p = spin*3 + colour)
 *    site index = ((x0*L1 + x1)*L2 + x2)*L3 + x3.  Convert with nd_pack_spinor / nd_unpack_spinor.
 *  - Complex scalars cross the boundary as double[2] = (re, im).  All reductions accumulate in fp64 in both
 *    precisions.
 *  - Stencil calls require out != in (and != tmp); violating it returns ND_ERR_BAD_ARG.
 */
#ifndef ND_B200_H
#define ND_B200_H

#include <stddef.h>

#if defined(__GNUC__)
#define ND_API __attribute__((visibility("default")))
#else
#define ND_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nd_ctx nd_ctx;

enum {
    ND_OK = 0,
    ND_ERR_BAD_ARG = -1,         /* null pointer, bad enum value, aliasing, size mismatch */
    ND_ERR_BAD_STATE = -2,       /* gauge field / polynomial / low modes not set yet */
    ND_ERR_NOT_SU3 = -3,         /* nd_set_gauge: a link violates U^dagger U = 1, det U = 1 beyond tolerance */
    ND_ERR_RECON8_SINGULAR = -4, /* nd_set_gauge with recon 8: |a2|^2+|a3|^2 below threshold (e.g. unit links) */
    ND_ERR_CUDA = -5,            /* CUDA runtime error (message in nd_last_error) */
    ND_ERR_NO_CONVERGENCE = -6,  /* nd_lowmodes_compute: maxit reached before tol */
    ND_ERR_NOMEM = -7
};

/* ---------------------------------------------------------------------------------------------- lifecycle
 * Geometry of the 4D lattice of eq. 2.1 and the storage choices of section 2.1
 * (PAPER.md:L44-50).
 *   dims     [in, host]  (L0=T, L1, L2, L3), each >= 2
 *   prec     32 or 64: arithmetic and storage type of spinors and links
 *   recon    18, 12 or 8: real parameters stored per SU(3) link (12: eq. 2.3; 8: PAPER.md:L46, R8)
 *   bc_time  +1 periodic / -1 antiperiodic in mu = 0 (space is periodic)
 *   device   CUDA device ordinal
 *   stream   cudaStream_t as void* (may be NULL)
 * On failure *ctx is NULL.  nd_destroy frees everything the context owns. */
ND_API int nd_create(nd_ctx** ctx, const int dims[4], int prec, int recon, int bc_time, int device, void* stream);
ND_API int nd_destroy(nd_ctx* ctx);
ND_API const char* nd_last_error(const nd_ctx* ctx);   /* never NULL; valid until the next call on ctx */
ND_API int nd_set_stream(nd_ctx* ctx, void* stream);
ND_API long long nd_volume(const nd_ctx* ctx);          /* number of sites V */
ND_API size_t nd_spinor_bytes(const nd_ctx* ctx);       /* bytes of one device SoA spinor = 24 * V * prec/8 */
ND_API size_t nd_gauge_bytes(const nd_ctx* ctx);        /* bytes of the compressed device gauge field */
/* Which kernel applies the stencil (csrc/wilson.cu, csrc/wilson_tile.cu).  ND_STENCIL_AUTO (default)
 * picks the fastest one measured for the context and call: the tiled marching kernel (neighbour exchange through shared memory,
 * cp.async prefetch of links, halos and the next spinor) on lattices it supports - x3 extent 32 or 16, even x1 / x2 extents >= 4
 * (x3 extent 16: x2 extent divisible by 4), at least 8 slices of 128 sites per SM, in fp64 recon 12 / 8 (recon 8: the plain
 * stencil only, with tensor-map loads on x3 extent 32) - and the site-per-thread kernel otherwise (hop-parallel below 16384 sites).  The other values force one kernel for every
 * call, for parity tests and for timing the variants against each other: ND_STENCIL_SITE; ND_STENCIL_TILE (the tiled kernel
 * above); ND_STENCIL_TILE_TMA (the same kernel with every prefetch issued as a TMA tensor-map box load instead of cp.async; x3
 * extent 32); ND_STENCIL_TILE4 (fp32, x3 extent 32: its predecessor with four link slots and the next spinor in registers).
 * ND_ERR_BAD_ARG if the context cannot run it.  Cached CUDA graphs are dropped.  nd_get_stencil_variant returns the variant in
 * effect for the plain stencil on lattices the tiled kernels take (never ND_STENCIL_AUTO); under ND_STENCIL_AUTO the choice also
 * depends on the call, and nd_get_stencil_variant_for answers for one call exactly - nd_apply_Q (fused_epilogue = 0) or
 * nd_apply_Q_axpbycz / the Clenshaw steps (fused_epilogue != 0) on nrhs right-hand sides - through the very function the dispatch
 * uses: ND_STENCIL_SITE covers the site-per-thread and, below 16384 sites x nrhs, the hop-parallel kernel. */
enum { ND_STENCIL_AUTO = 0, ND_STENCIL_SITE = 1, ND_STENCIL_TILE = 2, ND_STENCIL_TILE_TMA = 3, ND_STENCIL_TILE4 = 4 };
ND_API int nd_set_stencil_variant(nd_ctx* ctx, int variant);
ND_API int nd_get_stencil_variant(const nd_ctx* ctx);
ND_API int nd_get_stencil_variant_for(const nd_ctx* ctx, int fused_epilogue, int nrhs);
/* Number of kernels this context has launched since creation (bench.py's gpu_launches). */
ND_API long long nd_launch_count(const nd_ctx* ctx);

/* ------------------------------------------------------------------------------------------------- gauge
 * nd_set_gauge: take the canonical AoS links (src_prec 32: complex64, 64: complex128; on_device != 0: the
 * pointer is device memory, else host memory), check them (ND_ERR_NOT_SU3 / ND_ERR_RECON8_SINGULAR),
 * compress to `recon` reals and reorder to the device layout.  The input is not kept.
 * nd_get_gauge: reconstruct the full 3x3 links from the stored parameters into a canonical complex128 AoS
 * array (round-trip pin of eq. 2.3). */
ND_API int nd_set_gauge(nd_ctx* ctx, const void* links_aos, int src_prec, int on_device);
ND_API int nd_get_gauge(nd_ctx* ctx, void* links_aos_c128, int on_device);
/* Diagnostics of the last nd_set_gauge: out[0] = max |U^dagger U - 1| entry, out[1] = max |det U - 1|,
 * out[2] = min over links of N = |a2|^2 + |a3|^2 (conditioning of the 8-parameter form), out[3] = max entry of
 * |reconstruct(stored parameters) - U| (what the stencil will see; with recon 8 rounding is amplified by ~1/N and
 * nd_set_gauge returns ND_ERR_RECON8_SINGULAR above 2e-3 (fp32) / 1e-8 (fp64)).  A NaN anywhere in the links makes
 * out[0] = out[1] = +inf and nd_set_gauge fail with ND_ERR_NOT_SU3. */
ND_API int nd_gauge_stats(nd_ctx* ctx, double out[4]);

/* ------------------------------------------------------------------------------------------------ layout
 * Canonical AoS (prec 32: complex64 / 64: complex128; host or device) <-> device SoA in the context's
 * precision.  `soa` is always device memory of nd_spinor_bytes(ctx). */
ND_API int nd_pack_spinor(nd_ctx* ctx, const void* aos, int aos_prec, int aos_on_device, void* soa);
ND_API int nd_unpack_spinor(nd_ctx* ctx, const void* soa, void* aos, int aos_prec, int aos_on_device);
/* Device SoA spinor of precision src_prec -> device SoA spinor of precision dst_prec (32 / 64) on ctx's lattice and stream
 * (round to nearest when narrowing); the context's own precision does not matter.  dst != src. */
ND_API int nd_convert_spinor(nd_ctx* ctx, void* dst, int dst_prec, const void* src, int src_prec);

/* --------------------------------------------------------------------------------------------- operators
 * out = Q in,  Q = gamma5 D_W,
 *   D_W phi(x) = (4+m) phi(x) - 1/2 sum_{mu=0..3} [ U_mu(x)(1-gamma_mu) phi(x+mu^)
 *                                                 + U_mu(x-mu^)^dagger (1+gamma_mu) phi(x-mu^) ]
 * (eq. 2.1-2.2; chiral gamma basis, R2).  out, in: device SoA spinors.
 * nd_apply_Q2: out = Q (Q in) through the caller's temporary tmp. */
ND_API int nd_apply_Q(nd_ctx* ctx, void* out, const void* in, double m);
ND_API int nd_apply_Q2(nd_ctx* ctx, void* out, const void* in, void* tmp, double m);
/* out = s0 * Q(in) + s1*v1 + s2*v2 + s3*v3 with real scalars: the stencil with the vector recurrence folded
 * into its epilogue (the fused Clenshaw step of PAPER.md:L66).  v_i may be NULL when s_i == 0; out may
 * alias any v_i but not in. */
ND_API int nd_apply_Q_axpbycz(nd_ctx* ctx, void* out, const void* in, double m, double s0,
                       double s1, const void* v1, double s2, const void* v2, double s3, const void* v3);

/* ----------------------------------------------------------------------------- sign function / D_N set-up
 * nd_cheb_coeffs (host utility, no GPU): coefficients c[0..n] of P_n(y) = sum_k c_k T_k((2y-1-eps)/(1-eps))
 * approximating y^{-1/2} on [eps, 1] (eq. 2.5-2.6; Chebyshev interpolation, full c_0) and the
 * measured delta = max_{eps<=y<=1} |1 - sqrt(y) P(y)| (eq. 2.6). */
ND_API int nd_cheb_coeffs(int n, double eps, double* c, double* delta);
/* The same with the coefficients that MINIMISE delta of eq. 2.6 ("minmax polynomials"), by the Remez
 * exchange algorithm: delta is 1.6-1.9 times smaller than the interpolation polynomial's at equal degree.  *levelled (may be
 * NULL) = the levelled error |E| of the last reference: |E| <= the optimal delta <= *delta (de la Vallee-Poussin). */
ND_API int nd_minmax_coeffs(int n, double eps, double* c, double* delta, double* levelled);
/* Polynomial used by nd_apply_sign / nd_apply_DN: degree n, coefficients c[0..n] (host, copied), eps, the
 * norm bound qnorm >= ||Q|| (X = Q/qnorm) and the kernel mass m (= -(1+s), eq. 2.4). */
ND_API int nd_set_sign_poly(nd_ctx* ctx, int n, const double* c, double eps, double qnorm, double m);
/* Low-mode set of eq. 2.7: l orthonormal approximate eigenvectors u_k of Q (device SoA,
 * contiguous: vector k at byte offset k*nd_spinor_bytes) with Ritz values nu[k] (host).  The pointer is kept,
 * not copied; l = 0 clears it. */
ND_API int nd_set_lowmodes(nd_ctx* ctx, int l, const void* u_soa, const double* nu);

/* ------------------------------------------------------------------------------------------- sign / D_N
 * nd_apply_sign: out = sum_k sign(nu_k) u_k <u_k,in> + (1 - sum_k u_k u_k^dagger) X P_n(X^2) in   (eq. 2.11,
 * PAPER.md:L112; without low modes: eq. 2.5).  P_n(X^2) by the Clenshaw recurrence with each
 * step's vector update fused into the second stencil of Q^2: 2n+1 stencil launches.
 * nd_apply_DN: out = prefactor * (in + gamma5 sign(Q) in)   (eq. 2.4).
 * work = 3 caller-owned device spinors, contiguous (3*nd_spinor_bytes).  use_graph != 0 replays the launch
 * sequence as a CUDA graph cached on (out, in, work). */
ND_API int nd_apply_sign(nd_ctx* ctx, void* out, const void* in, void* work, int use_graph);
ND_API int nd_apply_DN(nd_ctx* ctx, void* out, const void* in, double prefactor, void* work, int use_graph);
/* The same operators on nrhs right-hand sides at once (1 <= nrhs <= 16, nrhs * l <= 256): in, out = nrhs device spinors stored
 * back to back, work = 3 * nrhs spinors.  Every launch of the sequence handles all right-hand sides (stencils: one grid row
 * per source, the links shared through L1 / L2; projection: the low modes are streamed once for all sources), so small
 * lattices - one source of 8^3x16 occupies a quarter of the machine - fill the GPU; per source the arithmetic is exactly that
 * of nd_apply_sign / nd_apply_DN. */
ND_API int nd_apply_sign_multi(nd_ctx* ctx, int nrhs, void* out, const void* in, void* work, int use_graph);
ND_API int nd_apply_DN_multi(nd_ctx* ctx, int nrhs, void* out, const void* in, double prefactor, void* work, int use_graph);

/* ------------------------------------------------------------------------------- massive operator and solver
 * nd_apply_DNm: the massive Neuberger-Dirac operator behind the bound (2.12) (R16)
 *     out = D_N^m in,   D_N^m = (1 - m/(2 prefactor)) D_N + m = (prefactor + m/2) in + (prefactor - m/2) gamma5 sign(Q) in
 * with prefactor = 1/abar as in nd_apply_DN; one sign-function application.  work: 3 device spinors.
 * nd_solve_DNm: x = (D_N^m)^{-1} b by conjugate gradients on the normal equations D^dagger D x = D^dagger b,
 * D^dagger = gamma5 D gamma5; x starts from 0; stops when |D^dagger(b - D x)| <= tol |D^dagger b| or after maxit
 * iterations (ND_ERR_NO_CONVERGENCE, x still the best iterate).  *relres = |b - D x| / |b| recomputed at the end,
 * *iters = CG iterations (2 operator applications each).  work: 8 device spinors.  Synchronises (host step lengths). */
ND_API int nd_apply_DNm(nd_ctx* ctx, void* out, const void* in, double prefactor, double mq, void* work, int use_graph);
ND_API int nd_solve_DNm(nd_ctx* ctx, void* x, const void* b, double prefactor, double mq, double tol, int maxit, void* work,
                        double* relres, int* iters);
/* Mixed precision ("fp32 inner Q applications with fp64 accumulation", BASELINE.json config 4): iterative
 * refinement x <- x + e, D e = r solved by nd_solve_DNm in the fp32 context ctx32 to inner_tol, r = b - D x recomputed in
 * the fp64 context ctx64 once per outer step, until |b - D x| <= tol |b|.  Both contexts must describe the same lattice on
 * the same device and have the same gauge field and polynomial set.  x, b: fp64 device spinors.
 * work64: 6 fp64 spinors, work32: 10 fp32 spinors.  stats (may be NULL): [0] outer steps (= fp64 operator applications),
 * [1] fp32 CG iterations in total. */
ND_API int nd_solve_DNm_mixed(nd_ctx* ctx64, nd_ctx* ctx32, void* x, const void* b, double prefactor, double mq, double tol,
                              double inner_tol, int max_outer, int max_inner, void* work64, void* work32, double* relres,
                              int* stats);

/* --------------------------------------------------------------------------------------------- low modes
 * nd_lowmodes_compute: the low modes of Q with their error control (section 2.3): minimise the block
 * Ritz functional of Q^2 (L79; method: Chebyshev-filtered subspace iteration, R13), Rayleigh-Ritz of Q (eq. 2.7,
 * L81) in the WHOLE block of k = l_max + lguard vectors, Ritz pairs sorted by |nu|, residues rho_j = ||(Q - nu_j) u_j||
 * (eq. 2.8) for every j < k, and the number of projected modes chosen dynamically (L110; R17): l' in
 * [l_min, l_max] at the largest gap |nu_{l'+1}| - |nu_{l'}|  (l_min == l_max fixes it).  d_k (L90) is estimated from the
 * guard values |nu_j|, j >= l', taken with both signs, and the projected values of the opposite sign; kappa_+- by eq. 2.9,
 * bound by eq. 2.10.  The iteration stops when (L110 "stopped when the desired level of precision is reached")
 *     stop_rule 0:  rho_k <= tol for all k < l'           stop_rule 1:  max(bound_+, bound_-) <= tol
 * or after maxit outer iterations (ND_ERR_NO_CONVERGENCE; all outputs are still filled with the last iterate).
 *   m        kernel mass;  degree: Chebyshev filter degree per outer iteration;  seed: start vectors (nd_gaussian)
 *   u_out    [out, device] l_max spinors; the first *l_chosen are the u_k of eq. 2.7, ascending in |nu|
 *   nu,resid [out, host]   k values each: the whole block's Ritz values of Q and residues, ascending in |nu|
 *                          (entries >= *l_chosen belong to the guard vectors)
 *   kappa, bound [out, host, may be NULL] (kappa_+, kappa_-) and the two bounds (2.10); +inf where undefined
 *   work     [device] nd_lowmodes_work_spinors(l_max, lguard) = 3k + 2 spinors
 *   stats    (may be NULL) [0] outer iterations, [1] stencil applications */
ND_API int nd_lowmodes_compute(nd_ctx* ctx, int l_min, int l_max, int lguard, int degree, double m, int stop_rule, double tol,
                               int maxit, unsigned long long seed, void* u_out, double* nu, double* resid, int* l_chosen,
                               double kappa[2], double bound[2], void* work, long long* stats);
ND_API size_t nd_lowmodes_work_spinors(int l_max, int lguard);
/* The gap rule alone (host utility, no GPU; R17): abs_nu[k] ascending moduli of the block's Ritz values;
 * *l = the cut in [l_min, l_max] (l_max < k) with the largest gap abs_nu[l] - abs_nu[l-1] (ties: smallest l), *gap = it. */
ND_API int nd_choose_l(int k, const double* abs_nu, int l_min, int l_max, int* l, double* gap);
/* Error control of the projectors (host utility, no GPU; eq. 2.8-2.10): from the Ritz values nu[l],
 * the residues rho[l] (eq. 2.8) and estimates rest[nrest] of the eigenvalues of Q outside the low-mode space, compute
 *   d_k      = distance of nu_k from {rest} and from the Ritz values of the opposite sign
 *   kappa[0] = kappa_+, kappa[1] = kappa_-,  kappa_+-^2 = sum_{+-nu_k > 0} rho_k^2 / d_k^2              (2.9)
 *   bound[i] = kappa (1 + 2 kappa) / (1 - 2 kappa (1 + 2 kappa))  >= || P_+- - (P_+-)_exact ||          (2.10)
 * bound[i] = +infinity when the denominator is not positive.  d (may be NULL) receives the l distances. */
ND_API int nd_projector_error(int l, const double* nu, const double* rho, int nrest, const double* rest, double kappa[2],
                              double bound[2], double* d);
/* Host utility (no GPU) used by nd_lowmodes_compute for the small dense problems of PAPER.md:L81: eigendecomposition
 * of a k x k Hermitian matrix a (row-major, complex as (re, im) pairs; only its Hermitian part is used) by the cyclic
 * Jacobi method: a = Z diag(w) Z^dagger, w[k] ascending, eigenvector j in COLUMN j of z (row-major, k*k complex). */
ND_API int nd_heev(int k, const double* a, double* w, double* z);

/* ------------------------------------------------------------------------------------------------- index
 * nd_index_count: the index of D_N by zero-mode counting (section 4).  D_N = c (1 + gamma5 sign(Q)) obeys the
 * Ginsparg-Wilson relation, so D_N^dagger D_N commutes with gamma5 and every zero mode has chirality +1 or -1;
 *     index = n_+ - n_-,   n_sigma = dim ker B_sigma,   B_sigma = P_sigma (1 + gamma5 sign(Q)) P_sigma = D_N^dagger D_N / (2 c^2)
 * on the sector gamma5 = sigma, P_sigma = (1 + sigma gamma5)/2, spectrum in [0, 2].  For each sigma the nvec lowest eigenvalues
 * of B_sigma are computed by Chebyshev-filtered block subspace iteration (filter degree `degree` per outer iteration, every
 * application of B_sigma = one sign-function application with the polynomial and low modes set in the context, 2n+1 stencils)
 * and a Rayleigh-Ritz step; a Ritz pair (theta_j, r_j = ||B x_j - theta_j x_j||) counts as a zero mode when
 * theta_j + r_j <= zero_tol and as a non-zero mode when theta_j - r_j > zero_tol; the iteration stops when every pair of the
 * block is decided and the lowest non-zero pair is located to 10 % (r_j <= 0.1 theta_j: the block sits on the low end).  zero_tol must sit between the sign function's error (delta, kappa_+-: the computed zero eigenvalues are
 * O(delta)) and the lowest non-zero eigenvalue of B_sigma.
 *   counts   [out, host]  (n_+, n_-)
 *   evals, resid [out, host]  2*nvec values each: theta_j and r_j of sector +1, then of sector -1, ascending in theta
 *   work     [device]  nd_index_work_spinors(nvec) = 3 nvec + 5 spinors
 *   stats    (may be NULL) [0] outer iterations (both sectors), [1] sign-function applications
 * Errors: ND_ERR_BAD_STATE without gauge field / polynomial; ND_ERR_NO_CONVERGENCE when a sector is undecided after maxit outer
 * iterations; ND_ERR_BAD_ARG when all nvec vectors of a sector come out as zero modes (nvec must exceed n_sigma). */
ND_API int nd_index_count(nd_ctx* ctx, int nvec, int degree, double zero_tol, int maxit, unsigned long long seed, int counts[2],
                          double* evals, double* resid, void* work, long long* stats);
ND_API size_t nd_index_work_spinors(int nvec);

/* ------------------------------------------------------------------------------------ domain decomposition
 * The lattice split along x0 (time) over nranks GPUs, one process per GPU: rank r owns
 * the slices [r T/nranks, (r+1) T/nranks) as a context created with the LOCAL dims (T/nranks, L1, L2, L3) and the GLOBAL
 * bc_time, its local links set by nd_set_gauge, then nd_set_sharding.  From then on every operator call of this header acts
 * on the rank's part of the global field and every reduction returns the GLOBAL value; all ranks must make the same calls in
 * the same order.  Per stencil application each rank sends two faces of projected half-spinors (nd_halo_bytes each; the face
 * for the next rank already multiplied by U_0^dagger, so links never travel; bc_time applied where a face crosses the global
 * seam) while the local stencil runs, and adds the two received hops to its boundary slices.  The transfers are the
 * caller's, through callbacks that work on DEVICE pointers owned by the context (valid until nd_destroy / the next
 * nd_set_sharding) and must be ordered with the context's stream:
 *   start(user, send_next, send_prev, recv_prev, recv_next, bytes): begin  send_next -> next rank's recv_prev,
 *                                                                          send_prev -> previous rank's recv_next
 *   wait(user):            the context's stream must not run past this point before both recv buffers are complete
 *   allreduce(user, d_buf, n): sum n doubles in device memory over the ranks, in place, ordered with the stream
 * (return 0 on success).  paper_1010_5636_b200/dist.py implements them with torch.distributed (NCCL send/recv over NVLink).
 * nranks == 1 removes the sharding.  CUDA graphs are not used while sharded.
 * nd_shard_layout (host helper, no GPU): first global slice and local extent of a rank, and whether its previous / next
 * face crosses the global seam; ND_ERR_BAD_ARG unless nranks divides T into parts of at least 2 slices. */
typedef int (*nd_exchange_start_fn)(void* user, const void* send_next, const void* send_prev, void* recv_prev, void* recv_next,
                                    size_t bytes);
typedef int (*nd_exchange_wait_fn)(void* user);
typedef int (*nd_allreduce_fn)(void* user, double* d_buf, int n);
ND_API int nd_shard_layout(int T, int nranks, int rank, int* t_begin, int* t_local, int* crosses_seam_prev, int* crosses_seam_next);
ND_API int nd_set_sharding(nd_ctx* ctx, int rank, int nranks, nd_exchange_start_fn start, nd_exchange_wait_fn wait,
                           nd_allreduce_fn allreduce, void* user);
ND_API size_t nd_halo_bytes(const nd_ctx* ctx);   /* bytes of one face: (V_local / T_local) * 12 reals */
/* Peer-to-peer mode of the face exchange: instead of packing into the context's send buffers and handing them to the `start`
 * callback, the pack kernel STORES the two faces directly into the neighbours' receive windows - the compute kernel's stores
 * are the transfer (over NVLink 5 / NVSwitch when the windows are peer-mapped device memory of the neighbouring GPUs, e.g. a
 * symmetric-memory allocation; paper_1010_5636_b200/dist.py: PeerComm).  A window is 4 * nd_halo_bytes(ctx) bytes of device
 * memory, caller-owned, laid out [parity 2][from_prev, from_next][nd_halo_bytes]: consecutive stencil applications alternate
 * between the two halves, so a rank may write the faces of application n+1 into a neighbour that is still consuming those of
 * application n.  recv_own = this rank's window, recv_of_next / recv_of_prev = the windows of the next / previous rank (the same
 * pointer twice when nranks = 2).  `start` is not called in this mode (it may be NULL in nd_set_sharding); `wait` must be a
 * barrier over the ranks ordered with the context's stream: when the stream passes it, every rank's pack kernel of this
 * application has completed and its stores are visible.  All three NULL: back to the callback transfers. */
ND_API int nd_set_halo_peers(nd_ctx* ctx, void* recv_own, void* recv_of_next, void* recv_of_prev);
ND_API int nd_halo_buffers(nd_ctx* ctx, void** send_next, void** send_prev, void** recv_prev, void** recv_next);

/* ------------------------------------------------------------------------------------------------ BLAS-1
 * Spinor-field vector operations (device SoA).  a = (re, im).
 *   nd_axpy:       y <- a x + y            nd_scale: x <- a x         nd_copy: y <- x
 *   nd_dot:        out = <x, y> = sum conj(x) y      (host result; synchronises)
 *   nd_norm2:      out = <x, x>
 *   nd_gamma5:     y <- gamma5 x  (y may alias x)
 *   nd_block_dot:  out[2k..2k+1] = <v_k, x>, k < l   (one pass over x and the block; host result)
 *   nd_block_axpy: y <- y + sum_k a[k] v_k           (a = l complex numbers on the host)
 *   nd_gaussian:   fill x with Re, Im ~ N(0,1) from a counter-based generator (Philox-4x32-10 + Box-Muller)
 *   nd_*_dev:      the same reductions with the result left in the caller's DEVICE memory (2l / 2 / 2 doubles, (re, im)
 *                  pairs; nd_norm2_dev: im = the rounding residue of the cancelling cross terms), and nd_block_axpy with its coefficients read from DEVICE memory (2l doubles):
 *                  enqueued on the context's stream without any synchronisation, so reductions and updates chain on the device */
ND_API int nd_axpy(nd_ctx* ctx, const double a[2], const void* x, void* y);
ND_API int nd_scale(nd_ctx* ctx, const double a[2], void* x);
ND_API int nd_copy(nd_ctx* ctx, void* y, const void* x);
ND_API int nd_dot(nd_ctx* ctx, const void* x, const void* y, double out[2]);
ND_API int nd_norm2(nd_ctx* ctx, const void* x, double* out);
ND_API int nd_gamma5(nd_ctx* ctx, void* y, const void* x);
ND_API int nd_block_dot(nd_ctx* ctx, int l, const void* v, const void* x, double* out2l);
ND_API int nd_block_axpy(nd_ctx* ctx, int l, const double* a2l, const void* v, void* y);
ND_API int nd_block_dot_dev(nd_ctx* ctx, int l, const void* v, const void* x, double* d_out2l);
ND_API int nd_dot_dev(nd_ctx* ctx, const void* x, const void* y, double* d_out2);
ND_API int nd_norm2_dev(nd_ctx* ctx, const void* x, double* d_out2);
ND_API int nd_block_axpy_dev(nd_ctx* ctx, int l, const double* d_a2l, const void* v, void* y);
ND_API int nd_gaussian(nd_ctx* ctx, void* x, unsigned long long seed);

/* ------------------------------------------------------------- inner product without any memory allocation
 * nd_dot_static: d_out2 = <x, y> = sum conj(x) y over two device SoA spinors of V sites (the BLAS-1 reduction of the
 * Clenshaw / low-mode steps), for callers that must not allocate device memory: a plug-in inside an
 * application whose own pool already holds the GPU's memory, code in a phase where cudaMalloc / cudaFree (which synchronise
 * the device) are off limits, a process with a fixed memory budget.  Every other reduction needs a context, and nd_create
 * calls cudaMalloc; this call needs no context and calls no cudaMalloc, cudaFree or any other allocating routine, ever.
 * Its partial sums go to an array that is part of the library image: ND_DOT_STATIC_SCRATCH_BYTES of device memory on every
 * GPU that loads the library's kernels, held until the process exits.
 *   x, y     [in, device]  SoA spinors of `prec` (32: 6 planes of float4[V], 64: 12 planes of double2[V]), 16-byte aligned
 *   V        sites, 1 <= V <= ND_DOT_STATIC_MAX_SITES (one partial sum per 256 sites must fit the array; 32^3 x 128 fits);
 *            anything else is refused with ND_ERR_BAD_ARG and a message naming the limit
 *   prec     32 or 64; products and sums are formed in fp64 in both cases
 *   device   CUDA device ordinal the pointers belong to (the caller's current device is restored before returning)
 *   stream   cudaStream_t as void* (may be NULL); the two kernels are enqueued there, nothing is synchronised
 *   d_out2   [out, device] 2 doubles (re, im), caller-owned, written by the second kernel
 *   errbuf   [out, host, may be NULL] receives a message of at most errbuf_len bytes when the call fails ("" on success)
 * Returns ND_OK, ND_ERR_BAD_ARG or ND_ERR_CUDA.  The result is bitwise reproducible and agrees with nd_dot_dev to rounding
 * (a different, equally fixed summation order).  On a sharded lattice it is the LOCAL sum - there is no context to reduce over.
 * The first call on each device looks up the array's device address (cudaGetSymbolAddress, cached afterwards): make that
 * first call outside any stream capture.  All calls on a device share the one array: a call overwrites the slots it later
 * reads, so nothing needs clearing between calls, but two calls that can overlap on the GPU (two streams, two host threads)
 * race on it - keep them on one stream or order them yourself. */
#define ND_DOT_STATIC_MAX_SITES 4194304
#define ND_DOT_STATIC_SCRATCH_BYTES 262144
ND_API int nd_dot_static(const void* x, const void* y, long long V, int prec, int device, void* stream, double* d_out2,
                         char* errbuf, size_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* ND_B200_H */
