// wilson.cu - the Wilson-Dirac stencil Q = gamma5 D_W (eq. 2.1-2.2) for sm_100a.
//
//   D_W phi(x) = (4+m) phi(x) - 1/2 sum_{mu=0..3} [ U_mu(x)(1-gamma_mu) phi(x+mu^) + U_mu(x-mu^)^dagger (1+gamma_mu) phi(x-mu^) ]
//
// One thread per output site, but: spin-projection to half-spinors BEFORE the SU(3) multiply,
// links reconstructed from 12 / 8 reals in registers, 128-bit coalesced loads from the
// plane-SoA layout, optional fused epilogue  out = s0*Q(in) + s1*v1 + s2*v2 + s3*v3  (the Clenshaw vector
// recurrence of PAPER.md:L66 folded into the stencil's store).
//
// Chiral basis (R2): gamma_mu = [[0, A_mu], [A_mu^dagger, 0]], A_0 = -1, A_k = -i sigma_k, gamma5 = diag(1,1,-1,-1).
//   (1-gamma_mu) psi = (h, -A^dagger h),  h  = psi_up - A psi_low
//   (1+gamma_mu) psi = (h',  A^dagger h'), h' = psi_up + A psi_low
#include "nd_dirac.cuh"

namespace {

struct Geom {
    int L0, L1, L2, L3;
    long long V;
    long long S1, S2;   // strides of x1, x0 in sites: S2 = L3 (x2 stride), S1 = L2*L3, S0 = L1*L2*L3
    long long S0;
    int bc;             // +1 / -1
    // CTA tile in (x1, x2, x3): 2^lb[i] sites along x_{i+1}, nt[i] tiles; nt[2] == 0: linear mapping
    int lb[3];
    int nt[3];
};

template <typename T, int RECON, int MU>
__device__ __forceinline__ void hop_pair(const typename Prec<T>::Vec* __restrict__ in,
                                         const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, const Geom& G,
                                         long long s, long long s_fwd, long long s_bwd, T ph_fwd, T ph_bwd, cx<T> (&acc)[12]) {
    cx<T> psi[12], U[3][3], h[2][3], g[2][3];
    // forward hop: U_mu(x) (1 - gamma_mu) phi(x + mu^)
    load_spinor<T>(in, G.V, s_fwd, psi);
    load_link<T, RECON>(gauge, G.V, MU, s, U);
    project<T, MU, -1>(psi, ph_fwd, h);
    mul_U(U, h, g);
    accumulate<T, MU, -1>(g, acc);
    // backward hop: U_mu(x - mu^)^dagger (1 + gamma_mu) phi(x - mu^)
    load_spinor<T>(in, G.V, s_bwd, psi);
    load_link<T, RECON>(gauge, G.V, MU, s_bwd, U);
    project<T, MU, +1>(psi, ph_bwd, h);
    mul_Udag(U, h, g);
    accumulate<T, MU, +1>(g, acc);
}

// 128 threads per CTA; resident CTAs per SM the register allocation is tuned for: 5 (fp32, 96 registers) / 3 (fp64, 168)
constexpr int Q_THREADS = 128;
template <typename T> constexpr int q_min_blocks() { return sizeof(T) == 4 ? 5 : 3; }

template <typename T, int RECON, bool EPI>
__global__ void __launch_bounds__(Q_THREADS, q_min_blocks<T>()) wilson_Q_kernel(typename Prec<T>::Vec* out,
                                                       const typename Prec<T>::Vec* __restrict__ in,
                                                       const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, Geom G,
                                                       T mass_term, T s0, T s1, const typename Prec<T>::Vec* v1, T s2,
                                                       const typename Prec<T>::Vec* v2, T s3,
                                                       const typename Prec<T>::Vec* v3, long long batch_stride) {
    {   // blockIdx.y = right-hand side of a batch (nd_apply_DN_multi): every field pointer moves on by one spinor
        const long long off = (long long)blockIdx.y * batch_stride;
        out += off; in += off;
        if (EPI) { if (v1) v1 += off; if (v2) v2 += off; if (v3) v3 += off; }
    }
    long long s;
    int x0, x1, x2, x3;
    if (G.nt[2] == 0) {
        s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (s >= G.V) return;
        x3 = (int)(s % G.L3);
        long long r = s / G.L3;
        x2 = (int)(r % G.L2);
        r /= G.L2;
        x1 = (int)(r % G.L1);
        x0 = (int)(r / G.L1);
    } else {
        // the CTA covers a (x1, x2, x3) block of one time-slice: its x1/x2/x3 neighbours are re-read through L1
        unsigned t = threadIdx.x, b = blockIdx.x;
        x3 = (int)(t & ((1u << G.lb[2]) - 1)); t >>= G.lb[2];
        x2 = (int)(t & ((1u << G.lb[1]) - 1)); t >>= G.lb[1];
        x1 = (int)t;
        x3 += (int)(b % G.nt[2]) << G.lb[2]; b /= G.nt[2];
        x2 += (int)(b % G.nt[1]) << G.lb[1]; b /= G.nt[1];
        x1 += (int)(b % G.nt[0]) << G.lb[0]; b /= G.nt[0];
        x0 = (int)b;
        s = (((long long)x0 * G.L1 + x1) * G.L2 + x2) * G.L3 + x3;
    }

    // The centre and the x1/x2/x3 hops come first: those are the lines neighbouring threads of the CTA share, and the
    // sooner after one another they are requested the more of them L1 still holds.  The time hops (no reuse inside the
    // CTA) come last.  The mass term enters through the accumulator: -1/2 acc = (4+m) phi - 1/2 sum(hops).
    cx<T> acc[12];
    {
        cx<T> phi[12];
        load_spinor<T>(in, G.V, s, phi);
        const T f = T(-2) * mass_term;
#pragma unroll
        for (int i = 0; i < 12; i++) acc[i] = {f * phi[i].re, f * phi[i].im};
    }
    {
        long long sf = (x1 == G.L1 - 1) ? s - (long long)(G.L1 - 1) * G.S1 : s + G.S1;
        long long sb = (x1 == 0) ? s + (long long)(G.L1 - 1) * G.S1 : s - G.S1;
        hop_pair<T, RECON, 1>(in, gauge, G, s, sf, sb, T(1), T(1), acc);
    }
    {
        long long sf = (x2 == G.L2 - 1) ? s - (long long)(G.L2 - 1) * G.S2 : s + G.S2;
        long long sb = (x2 == 0) ? s + (long long)(G.L2 - 1) * G.S2 : s - G.S2;
        hop_pair<T, RECON, 2>(in, gauge, G, s, sf, sb, T(1), T(1), acc);
    }
    {
        long long sf = (x3 == G.L3 - 1) ? s - (G.L3 - 1) : s + 1;
        long long sb = (x3 == 0) ? s + (G.L3 - 1) : s - 1;
        hop_pair<T, RECON, 3>(in, gauge, G, s, sf, sb, T(1), T(1), acc);
    }
    {
        long long sf = (x0 == G.L0 - 1) ? s - (long long)(G.L0 - 1) * G.S0 : s + G.S0;
        long long sb = (x0 == 0) ? s + (long long)(G.L0 - 1) * G.S0 : s - G.S0;
        T pf = (x0 == G.L0 - 1) ? T(G.bc) : T(1);
        T pb = (x0 == 0) ? T(G.bc) : T(1);
        hop_pair<T, RECON, 0>(in, gauge, G, s, sf, sb, pf, pb, acc);
    }

    finish_site<T, EPI>(out, G.V, s, acc, s0, s1, v1, s2, v2, s3, v3);
}

// --------------------------------------------------------------------------------- hop-parallel kernel (tiny lattices)
// On lattices of a few thousand sites (BASELINE config 3, 8^3x16) there are fewer sites than the GPU has lanes and the
// stencil is bound by the latency of its chain of eight dependent load -> multiply steps.  Here a CTA is 8 warps x 32
// sites: warp h computes hop h (h = 2 mu + {0: forward, 1: backward}) of the same 32 sites, so every load of a site is
// in flight at once; the eight contributions are summed through shared memory and warp p finishes plane p (mass term,
// gamma5, fused epilogue, one coalesced 128-bit store).
template <typename T, int RECON, int MU, int SGN>
__device__ __forceinline__ void single_hop(const typename Prec<T>::Vec* __restrict__ in,
                                           const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, long long V,
                                           long long s_spinor, long long s_link, T phase, cx<T> (&acc)[12]) {
    cx<T> psi[12], U[3][3], h[2][3], g[2][3];
    load_spinor<T>(in, V, s_spinor, psi);
    load_link<T, RECON>(gauge, V, MU, s_link, U);
    project<T, MU, SGN>(psi, phase, h);
    if (SGN < 0) mul_U(U, h, g);
    else mul_Udag(U, h, g);
    accumulate<T, MU, SGN>(g, acc);
}

template <typename T, int RECON, bool EPI>
__global__ void __launch_bounds__(256) wilson_Q_hop_kernel(typename Prec<T>::Vec* out,
                                                           const typename Prec<T>::Vec* __restrict__ in,
                                                           const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, Geom G,
                                                           T mass_term, T s0, T s1, const typename Prec<T>::Vec* v1, T s2,
                                                           const typename Prec<T>::Vec* v2, T s3,
                                                           const typename Prec<T>::Vec* v3, long long batch_stride) {
    using Vec = typename Prec<T>::Vec;
    constexpr int NV = Prec<T>::NV;
    constexpr int W = 24 / NV;   // reals per 128-bit word
    {
        const long long off = (long long)blockIdx.y * batch_stride;
        out += off; in += off;
        if (EPI) { if (v1) v1 += off; if (v2) v2 += off; if (v3) v3 += off; }
    }
    __shared__ T red[8][24][32];
    const int lane = threadIdx.x, hop = threadIdx.y;
    const long long s = (long long)blockIdx.x * 32 + lane;
    const bool valid = s < G.V;
    // the planes this warp will finish (hop, hop + 8): the site's own spinor and the fused update's vectors are requested NOW,
    // so that their latency runs concurrently with the hop's own load -> multiply chain instead of after the barrier
    constexpr int NPW = (NV + 7) / 8;
    Vec phi_p[NPW], vp[3][NPW];
    if (valid) {
#pragma unroll
        for (int k = 0; k < NPW; k++) {
            const int p = hop + 8 * k;
            if (p < NV) {
                phi_p[k] = in[p * G.V + s];
                if (EPI) {
                    if (v1) vp[0][k] = v1[p * G.V + s];
                    if (v2) vp[1][k] = v2[p * G.V + s];
                    if (v3) vp[2][k] = v3[p * G.V + s];
                }
            }
        }
    }
    cx<T> acc[12];
#pragma unroll
    for (int i = 0; i < 12; i++) acc[i] = {T(0), T(0)};
    if (valid) {
        const int x3 = (int)(s % G.L3);
        long long r = s / G.L3;
        const int x2 = (int)(r % G.L2);
        r /= G.L2;
        const int x1 = (int)(r % G.L1);
        const int x0 = (int)(r / G.L1);
        switch (hop) {   // warp-uniform
            case 0: single_hop<T, RECON, 0, -1>(in, gauge, G.V, (x0 == G.L0 - 1) ? s - (long long)(G.L0 - 1) * G.S0 : s + G.S0, s,
                                                 (x0 == G.L0 - 1) ? T(G.bc) : T(1), acc); break;
            case 1: { const long long sb = (x0 == 0) ? s + (long long)(G.L0 - 1) * G.S0 : s - G.S0;
                      single_hop<T, RECON, 0, +1>(in, gauge, G.V, sb, sb, (x0 == 0) ? T(G.bc) : T(1), acc); } break;
            case 2: single_hop<T, RECON, 1, -1>(in, gauge, G.V, (x1 == G.L1 - 1) ? s - (long long)(G.L1 - 1) * G.S1 : s + G.S1, s, T(1), acc); break;
            case 3: { const long long sb = (x1 == 0) ? s + (long long)(G.L1 - 1) * G.S1 : s - G.S1;
                      single_hop<T, RECON, 1, +1>(in, gauge, G.V, sb, sb, T(1), acc); } break;
            case 4: single_hop<T, RECON, 2, -1>(in, gauge, G.V, (x2 == G.L2 - 1) ? s - (long long)(G.L2 - 1) * G.S2 : s + G.S2, s, T(1), acc); break;
            case 5: { const long long sb = (x2 == 0) ? s + (long long)(G.L2 - 1) * G.S2 : s - G.S2;
                      single_hop<T, RECON, 2, +1>(in, gauge, G.V, sb, sb, T(1), acc); } break;
            case 6: single_hop<T, RECON, 3, -1>(in, gauge, G.V, (x3 == G.L3 - 1) ? s - (G.L3 - 1) : s + 1, s, T(1), acc); break;
            default: { const long long sb = (x3 == 0) ? s + (G.L3 - 1) : s - 1;
                       single_hop<T, RECON, 3, +1>(in, gauge, G.V, sb, sb, T(1), acc); } break;
        }
    }
#pragma unroll
    for (int i = 0; i < 12; i++) {
        red[hop][2 * i][lane] = acc[i].re;
        red[hop][2 * i + 1][lane] = acc[i].im;
    }
    __syncthreads();
    if (!valid) return;
#pragma unroll
    for (int k = 0; k < NPW; k++) {   // warp `hop` finishes planes hop, hop + 8
        const int p = hop + 8 * k;
        if (p >= NV) break;
        Vec phi = phi_p[k], w;
        const T* pr = reinterpret_cast<const T*>(&phi);
        T* wr = reinterpret_cast<T*>(&w);
        const T sg = (p * W < 12) ? T(1) : T(-1);   // gamma5: reals 0..11 are spin 0, 1
#pragma unroll
        for (int q = 0; q < W; q++) {
            T t = T(0);
#pragma unroll
            for (int h = 0; h < 8; h++) t += red[h][p * W + q][lane];
            wr[q] = sg * fma(T(-0.5), t, mass_term * pr[q]);
        }
        if (EPI) {
#pragma unroll
            for (int q = 0; q < W; q++) wr[q] *= s0;
            const Vec* vs[3] = {v1, v2, v3};
            const T ss[3] = {s1, s2, s3};
#pragma unroll
            for (int j = 0; j < 3; j++)
                if (vs[j]) {
                    const Vec a = vp[j][k];
                    const T* ar = reinterpret_cast<const T*>(&a);
#pragma unroll
                    for (int q = 0; q < W; q++) wr[q] = fma(ss[j], ar[q], wr[q]);
                }
        }
        out[p * G.V + s] = w;
    }
}

template <typename T, int RECON>
int launch_Q(nd_ctx* ctx, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1, double s2,
             const void* v2, double s3, const void* v3, int nrhs) {
    using Vec = typename Prec<T>::Vec;
    using LVec = typename LinkLayout<T, RECON>::LVec;
    Geom G;
    G.L0 = ctx->dims[0]; G.L1 = ctx->dims[1]; G.L2 = ctx->dims[2]; G.L3 = ctx->dims[3];
    G.V = ctx->V;
    G.S2 = G.L3;
    G.S1 = (long long)G.L2 * G.L3;
    G.S0 = (long long)G.L1 * G.L2 * G.L3;
    G.bc = ctx->bc;
    const long long bstride = (long long)Prec<T>::NV * ctx->V;   // one spinor, in 128-bit words
    if (ctx->V * nrhs < (long long)ctx->hop_max_sites) {   // (a batch of right-hand sides counts as one larger lattice)
        // fewer sites than lanes on the chip: one warp per hop (latency-bound regime, BASELINE config 3)
        const dim3 nb((unsigned)((ctx->V + 31) / 32), (unsigned)nrhs, 1);
        const dim3 tb(32, 8, 1);
        if (epi)
            wilson_Q_hop_kernel<T, RECON, true><<<nb, tb, 0, ctx->stream>>>(
                (Vec*)out, (const Vec*)in, (const LVec*)ctx->gauge, G, T(4.0 + m), T(s0), T(s1), (const Vec*)v1, T(s2),
                (const Vec*)v2, T(s3), (const Vec*)v3, bstride);
        else
            wilson_Q_hop_kernel<T, RECON, false><<<nb, tb, 0, ctx->stream>>>(
                (Vec*)out, (const Vec*)in, (const LVec*)ctx->gauge, G, T(4.0 + m), T(1), T(0), nullptr, T(0), nullptr, T(0),
                nullptr, bstride);
        ND_LAUNCHED(ctx);
        return ND_OK;
    }
    // 128 threads per CTA; small lattices get smaller CTAs so that every SM has work
    int threads = 128;
    while (threads > 32 && ctx->V * nrhs / threads < 2 * ctx->num_sms) threads /= 2;
    unsigned blocks1 = (unsigned)((ctx->V + threads - 1) / threads);
    for (int i = 0; i < 3; i++) { G.lb[i] = ctx->tile_lb[i]; G.nt[i] = 0; }
    if (ctx->tile_threads > 0 && ctx->tile_threads <= Q_THREADS && ctx->V * nrhs / ctx->tile_threads >= 2 * ctx->num_sms) {
        threads = ctx->tile_threads;
        blocks1 = (unsigned)G.L0;
        for (int i = 0; i < 3; i++) { G.nt[i] = ctx->dims[i + 1] >> G.lb[i]; blocks1 *= (unsigned)G.nt[i]; }
    }
    const dim3 blocks(blocks1, (unsigned)nrhs, 1);
    if (epi)
        wilson_Q_kernel<T, RECON, true><<<blocks, threads, 0, ctx->stream>>>(
            (Vec*)out, (const Vec*)in, (const LVec*)ctx->gauge, G, T(4.0 + m), T(s0), T(s1), (const Vec*)v1, T(s2),
            (const Vec*)v2, T(s3), (const Vec*)v3, bstride);
    else
        wilson_Q_kernel<T, RECON, false><<<blocks, threads, 0, ctx->stream>>>(
            (Vec*)out, (const Vec*)in, (const LVec*)ctx->gauge, G, T(4.0 + m), T(1), T(0), nullptr, T(0), nullptr, T(0),
            nullptr, bstride);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

}  // namespace

int ndi_apply_Q(nd_ctx* ctx, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1,
                double s2, const void* v2, double s3, const void* v3) {
    return ndi_apply_Q_batch(ctx, 1, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
}

// the same stencil on nrhs right-hand sides stored back to back (out, in and every v_i are batches of nrhs spinors): one
// launch with blockIdx.y = right-hand side; the links are shared through L1 / L2
int ndi_apply_Q_batch(nd_ctx* ctx, int nrhs, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1,
                      double s2, const void* v2, double s3, const void* v3) {
    if (!ctx) return ND_ERR_BAD_ARG;
    if (nrhs < 1 || nrhs > 65535) return nd_fail(ctx, ND_ERR_BAD_ARG, "apply_Q: bad number of right-hand sides");
    if (!out || !in || out == in) return nd_fail(ctx, ND_ERR_BAD_ARG, "apply_Q: out/in null or aliased");
    if (!ctx->gauge_set) return nd_fail(ctx, ND_ERR_BAD_STATE, "apply_Q: gauge field not set");
    if (s1 == 0.0) v1 = nullptr;
    if (s2 == 0.0) v2 = nullptr;
    if (s3 == 0.0) v3 = nullptr;
    if (v1 == in || v2 == in || v3 == in) {
        // allowed (read-only), nothing to do
    }
    if (ctx->shard_n > 1 && !ctx->in_shard_call) {
        // domain decomposition (shard.cu): faces out, the local stencil with the wrapped time hops switched off while the
        // transfer runs, faces in.  One right-hand side at a time (the halo buffers hold one face pair).
        const size_t sb = nd_spinor_bytes(ctx);
        for (int j = 0; j < nrhs; j++) {
            const size_t o = (size_t)j * sb;
            int rc = ndi_halo_pack(ctx, (const char*)in + o);
            if (rc != ND_OK) return rc;
            if (!ctx->peer_own) {   // (peer-to-peer mode: the pack kernel has already stored the faces where they belong)
                if (!ctx->exchange_start) return nd_fail(ctx, ND_ERR_BAD_STATE, "sharding: neither an exchange-start callback nor peer windows");
                if (ctx->exchange_start(ctx->comm_user, ctx->halo[0], ctx->halo[1], ctx->halo[2], ctx->halo[3], nd_halo_bytes(ctx)) != 0)
                    return nd_fail(ctx, ND_ERR_CUDA, "sharding: the exchange-start callback failed");
            }
            ctx->in_shard_call = true;
            const int saved_bc = ctx->bc;
            ctx->bc = 0;   // phase of the hops across the local time boundary: they come from the neighbours instead
            rc = ndi_apply_Q_batch(ctx, 1, (char*)out + o, (const char*)in + o, m, epi, s0, s1, v1 ? (const char*)v1 + o : nullptr, s2,
                                   v2 ? (const char*)v2 + o : nullptr, s3, v3 ? (const char*)v3 + o : nullptr);
            ctx->bc = saved_bc;
            ctx->in_shard_call = false;
            // From here on the exchange is under way on every rank (requests posted / faces stored into the neighbours' windows):
            // whatever happened to the local stencil, complete it and move to the other half of the receive windows, so that
            // no request is left outstanding, no peer waits for ever and halo_parity stays the same on all ranks.  The first
            // error is the one reported.
            if (!ctx->exchange_wait || ctx->exchange_wait(ctx->comm_user) != 0) {
                if (rc == ND_OK) rc = nd_fail(ctx, ND_ERR_CUDA, "sharding: the exchange-wait callback failed");
            } else if (rc == ND_OK) {
                rc = ndi_halo_apply(ctx, (char*)out + o, epi ? s0 : 1.0);
            }
            ctx->halo_parity ^= 1;   // the next application uses the other half of the receive windows
            if (rc != ND_OK) return rc;
        }
        return ND_OK;
    }
    // tiled marching kernels (wilson_tile.cu) or the site-per-thread / hop-parallel kernels of this file: ndi_select_stencil
    if (ndi_select_stencil(ctx, epi, nrhs) != ND_STENCIL_SITE) return ndi_apply_Q_tile(ctx, nrhs, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
#define ND_DISPATCH(T, R) return launch_Q<T, R>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3, nrhs)
    if (ctx->prec == 32) {
        if (ctx->recon == 18) ND_DISPATCH(float, 18);
        if (ctx->recon == 12) ND_DISPATCH(float, 12);
        ND_DISPATCH(float, 8);
    } else {
        if (ctx->recon == 18) ND_DISPATCH(double, 18);
        if (ctx->recon == 12) ND_DISPATCH(double, 12);
        ND_DISPATCH(double, 8);
    }
#undef ND_DISPATCH
}
