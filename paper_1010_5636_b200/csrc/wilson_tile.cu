// wilson_tile.cu - the Wilson-Dirac stencil Q = gamma5 D_W (eq. 2.1-2.2) as a tiled, marching kernel with
// neighbour exchange through shared memory (BASELINE.json north_star subsystem 2: "stages neighbour halos in shared memory").
//
// Why: the site-per-thread kernel (wilson.cu) moves its compulsory bytes through HBM exactly once, but pulls every
// neighbour spinor and every backward link through the L2 -> SM fabric again (822 B/site in fp32 for 384 B compulsory,
// profiles/r01_q_kernel_ncu_full.md) and sits at that fabric's limit, not at the HBM roofline.  Here
//   * a CTA owns a tile of B1 x B2 x L3 sites of one time-slice (x3 in full, so the warp runs along whole x3 rows) and
//     MARCHES along x0 over a segment of time-slices; a thread owns one (x1, x2, x3) column;
//   * every thread loads ITS OWN spinor and ITS OWN four links, once, fully coalesced (288 B/site in fp32 = the compulsory
//     input traffic), reconstructs each link once, and SENDS to its neighbours, through shared memory, what they need:
//         h-_mu(x) = (1 - gamma_mu) phi(x)                 to x - mu^  (which multiplies by its own U_mu(x - mu^))
//         w_mu(x)  = U_mu(x)^dagger (1 + gamma_mu) phi(x)   to x + mu^  (its complete backward hop)
//     as half-spinors (12 reals) - so no thread ever loads a neighbour's link, and every link is rebuilt by its owner only;
//   * the x3 neighbours are in the same warp: exchanged with shuffles; the x0 neighbours are the thread's own column:
//     phi(t+1) is prefetched into registers and the backward time hop w_0 is carried from the previous slice;
//   * only tile-face sites read neighbour data from global memory (the halo: phi for a forward face, phi and the one link
//     for a backward face) and put the resulting half-spinor into their own receive slot, so the receive phase is uniform;
//   * the links of the NEXT slice travel by cp.async straight into a private shared-memory slot of the thread that owns
//     them while the current slice is computed: a whole slice of link data per CTA is in flight without holding registers;
//   * x1 and x2 use separate exchange buffers in turn (send x1, barrier, receive x1, send x2, barrier, receive x2): two
//     __syncthreads per time-slice and no buffer is ever written while it may still be read.
// L2 -> SM traffic per site (fp32, recon 12, tile 2 x 2 x 32, measured): 541 B against 822 B of the site-per-thread kernel.
//
// Three kernels share this scheme:
//   wilson_Q_tile_kernel   the first shipped form (fp32): four link slots, next spinor of the column in registers (ND_STENCIL_TILE4)
//   wilson_Q_tile2_kernel  the default (fp32 and fp64, x3 extent 32 or 16, batches of right-hand sides): two link slots shared by
//                          two directions each, next spinor through a shared-memory slot, four cp.async groups per slice
//   wilson_Q_tile3_kernel  tile2's schedule with TMA tensor-map box loads instead of cp.async (ND_STENCIL_TILE_TMA)
#include <cuda.h>   // CUtensorMap (the tensor-map variant at the end of this file)

#include <cstring>
#include <mutex>

#include "nd_dirac.cuh"

namespace {

struct TileGeom {
    int L0, L1, L2;
    long long V, S0;
    int bc;
    int nt2, ntile;          // tiles along x2, tiles per time-slice
    int seg_base, seg_rem;   // nseg segments of time-slices: the first seg_rem have seg_base + 1 slices, the rest seg_base
};

template <typename T> struct HalfWords { static constexpr int NW = sizeof(T) == 4 ? 3 : 6; };   // 128-bit words of a half-spinor

__device__ __forceinline__ void half_to_words(const cx<float> (&h)[2][3], float4 (&w)[3]) {
    w[0] = make_float4(h[0][0].re, h[0][0].im, h[0][1].re, h[0][1].im);
    w[1] = make_float4(h[0][2].re, h[0][2].im, h[1][0].re, h[1][0].im);
    w[2] = make_float4(h[1][1].re, h[1][1].im, h[1][2].re, h[1][2].im);
}
__device__ __forceinline__ void words_to_half(const float4 (&w)[3], cx<float> (&h)[2][3]) {
    h[0][0] = {w[0].x, w[0].y}; h[0][1] = {w[0].z, w[0].w};
    h[0][2] = {w[1].x, w[1].y}; h[1][0] = {w[1].z, w[1].w};
    h[1][1] = {w[2].x, w[2].y}; h[1][2] = {w[2].z, w[2].w};
}
__device__ __forceinline__ void half_to_words(const cx<double> (&h)[2][3], double2 (&w)[6]) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int c = 0; c < 3; c++) w[3 * s + c] = make_double2(h[s][c].re, h[s][c].im);
}
__device__ __forceinline__ void words_to_half(const double2 (&w)[6], cx<double> (&h)[2][3]) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int c = 0; c < 3; c++) h[s][c] = {w[3 * s + c].x, w[3 * s + c].y};
}
// slot (kind, site) of one exchange buffer: words [kind][w][site], consecutive lanes on consecutive 128-bit words
template <typename T, int NT>
__device__ __forceinline__ void put_half(typename Prec<T>::Vec* buf, int kind, int site, const cx<T> (&h)[2][3]) {
    constexpr int NW = HalfWords<T>::NW;
    typename Prec<T>::Vec w[NW];
    half_to_words(h, w);
#pragma unroll
    for (int i = 0; i < NW; i++) buf[(kind * NW + i) * NT + site] = w[i];
}
template <typename T, int NT>
__device__ __forceinline__ void get_half(const typename Prec<T>::Vec* buf, int kind, int site, cx<T> (&h)[2][3]) {
    constexpr int NW = HalfWords<T>::NW;
    typename Prec<T>::Vec w[NW];
#pragma unroll
    for (int i = 0; i < NW; i++) w[i] = buf[(kind * NW + i) * NT + site];
    words_to_half(w, h);
}

__device__ __forceinline__ float shfl_real(float v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ double shfl_real(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
template <typename T> __device__ __forceinline__ void shfl_half(cx<T> (&h)[2][3], int src) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            h[s][c].re = shfl_real(h[s][c].re, src);
            h[s][c].im = shfl_real(h[s][c].im, src);
        }
}

// a link kept in registers between its two uses (send phase: U^dagger on the own spinor; receive phase: U on the neighbour's).
// fp32 keeps the whole matrix; fp64, short of registers, keeps two rows and rebuilds the third (eq. 2.3) at the second use.
template <typename T> struct KeptLink {
    static constexpr int ROWS = sizeof(T) == 4 ? 3 : 2;
    cx<T> r[ROWS][3];
    __device__ __forceinline__ void keep(const cx<T> (&U)[3][3]) {
#pragma unroll
        for (int i = 0; i < ROWS; i++)
#pragma unroll
            for (int j = 0; j < 3; j++) r[i][j] = U[i][j];
    }
    __device__ __forceinline__ void get(cx<T> (&U)[3][3]) const {
#pragma unroll
        for (int i = 0; i < ROWS; i++)
#pragma unroll
            for (int j = 0; j < 3; j++) U[i][j] = r[i][j];
        if (ROWS == 2) third_row(U);
    }
};

// cp.async (LDGSTS): 16 bytes global -> shared without passing through registers; .cg = cached in L2 only (streamed data)
template <int BYTES> __device__ __forceinline__ void cp_async(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");   // fp32 recon 18: 64-bit words
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// mbarrier helpers of the tensor-map variant (wilson_Q_tile3_kernel): completion of TMA loads is counted in bytes
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(b)),
        "r"(parity)
        : "memory");
}

// The halo slot of a tile-face thread: the spinor (and, for a backward face, the link) of its neighbour outside the tile,
// fetched by cp.async one phase ahead: words [NV spinor planes][NT] then [NL link words][NT].
// (HLN entries per link word, entry `hidx` of this thread: the fp64 kernel keeps link entries for the backward faces only)
template <typename T, int RECON, int MU, int NT, int HLN = NT>
__device__ __forceinline__ void issue_halo(unsigned char* hal, const typename Prec<T>::Vec* __restrict__ in,
                                           const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, long long V, int site,
                                           bool face_bwd, bool face_fwd, long long s_bwd, long long s_fwd, int hidx) {
    using Vec = typename Prec<T>::Vec;
    using LL = LinkLayout<T, RECON>;
    Vec* hs = reinterpret_cast<Vec*>(hal);
    typename LL::LVec* hl = reinterpret_cast<typename LL::LVec*>(hal + (size_t)Prec<T>::NV * NT * sizeof(Vec));
    if (face_fwd || face_bwd) {
        const long long sn = face_fwd ? s_fwd : s_bwd;
#pragma unroll
        for (int p = 0; p < Prec<T>::NV; p++) cp_async<16>(&hs[p * NT + site], in + p * V + sn);
    }
    if (face_bwd) {
#pragma unroll
        for (int p = 0; p < LL::NL; p++) cp_async<sizeof(typename LL::LVec)>(&hl[p * HLN + hidx], gauge + ((long long)MU * LL::NL + p) * V + s_bwd);
    }
}

// One direction mu in {1, 2} of the send phase of a site: the two half-spinors its in-tile neighbours need, and, on a tile
// face, the half-spinor this site itself needs from outside the tile (neighbour data from the halo slot).
//   slot kinds K = "h- of my forward neighbour" (read in the forward hop), K + 1 = "w of my backward neighbour"
template <typename T, int RECON, int MU, int NT, int K, int HLN = NT>
__device__ __forceinline__ void send_dir(typename Prec<T>::Vec* buf, const unsigned char* hal, const cx<T> (&phi)[12],
                                         const cx<T> (&U)[3][3], int site, int slot_bwd, int slot_fwd, bool face_bwd, bool face_fwd,
                                         int hidx) {
    using Vec = typename Prec<T>::Vec;
    using LL = LinkLayout<T, RECON>;
    cx<T> h[2][3], g[2][3];
    if (slot_bwd >= 0) {   // my h- goes to the site behind me: it is ITS forward neighbour's projection
        project<T, MU, -1>(phi, T(1), h);
        put_half<T, NT>(buf, K, slot_bwd, h);
    }
    if (slot_fwd >= 0) {   // my complete backward-hop product goes to the site in front of me
        project<T, MU, +1>(phi, T(1), h);
        mul_Udag(U, h, g);
        put_half<T, NT>(buf, K + 1, slot_fwd, g);
    }
    if (face_fwd || face_bwd) {
        const Vec* hs = reinterpret_cast<const Vec*>(hal);
        Vec w[Prec<T>::NV];
#pragma unroll
        for (int p = 0; p < Prec<T>::NV; p++) w[p] = hs[p * NT + site];
        cx<T> psi[12];
        words_to_cx(w, psi);
        if (face_fwd) {    // forward neighbour outside the tile
            project<T, MU, -1>(psi, T(1), h);
            put_half<T, NT>(buf, K, site, h);
        } else {           // backward neighbour outside the tile: its spinor and its link
            const typename LL::LVec* hl = reinterpret_cast<const typename LL::LVec*>(hal + (size_t)Prec<T>::NV * NT * sizeof(Vec));
            typename LL::LVec lw[LL::NL];
#pragma unroll
            for (int p = 0; p < LL::NL; p++) lw[p] = hl[p * HLN + hidx];
            cx<T> Ub[3][3];
            reconstruct_link<T, RECON>(lw, Ub);
            project<T, MU, +1>(psi, T(1), h);
            mul_Udag(Ub, h, g);
            put_half<T, NT>(buf, K + 1, site, g);
        }
    }
}

template <typename T, int MU, int NT, int K>
__device__ __forceinline__ void recv_dir(const typename Prec<T>::Vec* buf, const cx<T> (&U)[3][3], int site, cx<T> (&acc)[12]) {
    cx<T> h[2][3], g[2][3];
    get_half<T, NT>(buf, K, site, h);        // (1 - gamma_mu) phi(x + mu^)
    mul_U(U, h, g);
    accumulate<T, MU, -1>(g, acc);
    get_half<T, NT>(buf, K + 1, site, g);    // U_mu(x - mu^)^dagger (1 + gamma_mu) phi(x - mu^)
    accumulate<T, MU, +1>(g, acc);
}

// the thread's private link slot: words [mu][w][site].  take_link reads link mu of the current slice from the slot, rebuilds
// the matrix, and (when `next` is a site of the next slice) refills the slot with the next slice's words by cp.async - the
// in-flight link data of a whole time-slice lives in shared memory, not in registers.
template <typename T, int RECON, int NT>
__device__ __forceinline__ void take_link(typename LinkLayout<T, RECON>::LVec* lnk, const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge,
                                          long long V, int mu, int site, bool refill, long long s_next, cx<T> (&U)[3][3]) {
    using LL = LinkLayout<T, RECON>;
    typename LL::LVec w[LL::NL];
#pragma unroll
    for (int p = 0; p < LL::NL; p++) w[p] = lnk[(mu * LL::NL + p) * NT + site];
    reconstruct_link<T, RECON>(w, U);
    if (refill) {
        const typename LL::LVec* src = gauge + (long long)mu * LL::NL * V + s_next;
#pragma unroll
        for (int p = 0; p < LL::NL; p++) cp_async<sizeof(typename LL::LVec)>(&lnk[(mu * LL::NL + p) * NT + site], src + p * V);
    }
}

// The vectors of the fused update out = s0*Q(in) + s1*v1 + s2*v2 + s3*v3 at this thread's site, loaded BEFORE the last barrier
// of the slice and combined after it (out may alias any v_i: every v_i(x) is read before out(x) is written, by the same thread).
// (fp64 has no registers to spare for this: there the vectors are loaded at use, after the barrier.)
template <typename T, bool EPI> struct EpiVectors {
    static constexpr bool EARLY = EPI && sizeof(T) == 4;
    typename Prec<T>::Vec w[EARLY ? 3 : 1][Prec<T>::NV];
    const typename Prec<T>::Vec* vs[3];
    __device__ __forceinline__ void load(long long V, long long s, T s1, const typename Prec<T>::Vec* v1, T s2,
                                         const typename Prec<T>::Vec* v2, T s3, const typename Prec<T>::Vec* v3) {
        vs[0] = v1; vs[1] = v2; vs[2] = v3;
        if (EARLY) {
#pragma unroll
            for (int j = 0; j < 3; j++)
                if (vs[j]) {
#pragma unroll
                    for (int p = 0; p < Prec<T>::NV; p++) w[j][p] = vs[j][p * V + s];
                }
        }
    }
    __device__ __forceinline__ void finish(typename Prec<T>::Vec* out, long long V, long long s, const cx<T> (&acc)[12], T s0, T s1,
                                           T s2, T s3) {
        using Vec = typename Prec<T>::Vec;
        constexpr int NV = Prec<T>::NV;
        cx<T> res[12];
#pragma unroll
        for (int i = 0; i < 12; i++) {
            const T sg = (i < 6) ? T(-0.5) : T(0.5);   // gamma5 [ -1/2 acc ]
            res[i].re = sg * acc[i].re;
            res[i].im = sg * acc[i].im;
        }
        Vec o[NV];
        cx_to_words(res, o);
        if (EPI) {
            T* wr = reinterpret_cast<T*>(o);
#pragma unroll
            for (int i = 0; i < 24; i++) wr[i] *= s0;
            const T ss[3] = {s1, s2, s3};
#pragma unroll
            for (int j = 0; j < 3; j++)
                if (vs[j]) {
                    if (EARLY) {
                        const T* ar = reinterpret_cast<const T*>(w[j]);
#pragma unroll
                        for (int i = 0; i < 24; i++) wr[i] = fma(ss[j], ar[i], wr[i]);
                    } else {
#pragma unroll
                        for (int p = 0; p < NV; p++) {
                            const Vec a = vs[j][p * V + s];
                            const T* ar = reinterpret_cast<const T*>(&a);
#pragma unroll
                            for (int i = 0; i < 24 / NV; i++) wr[p * (24 / NV) + i] = fma(ss[j], ar[i], wr[p * (24 / NV) + i]);
                        }
                    }
                }
        }
#pragma unroll
        for (int p = 0; p < NV; p++) out[p * V + s] = o[p];
    }
};

// Synchronisation of the exchange.  In a 2 x 2 x 32 tile a warp is one x3 row and has exactly ONE partner warp per direction
// (the other row of the pair), so a 64-thread named barrier per pair replaces the CTA-wide barrier, with two meetings per
// direction and slice: "the partner has finished its previous receive" before the send, "data is in place" after it.  The
// first meeting orders EVERYTHING the partner did before it, so x1 and x2 can share one exchange buffer: a site's slots are
// written by its x1 partner only after the site's own x2 receive of the last slice, and by its x2 partner only after its
// own x1 receive of this slice.
template <int B1, int B2, int L3> struct PairSync { static constexpr bool value = (B1 == 2 && B2 == 2 && L3 == 32); };
__device__ __forceinline__ void pair_barrier(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }

template <typename T, int RECON, bool EPI, int B1, int B2, int L3, int MINB>
__global__ void __launch_bounds__(B1* B2* L3, MINB)
    wilson_Q_tile_kernel(typename Prec<T>::Vec* out, const typename Prec<T>::Vec* __restrict__ in,
                         const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, TileGeom G, T mass_term, T s0, T s1,
                         const typename Prec<T>::Vec* v1, T s2, const typename Prec<T>::Vec* v2, T s3,
                         const typename Prec<T>::Vec* v3) {
    using Vec = typename Prec<T>::Vec;
    using LL = LinkLayout<T, RECON>;
    using LVec = typename LL::LVec;
    constexpr int NT = B1 * B2 * L3;
    constexpr int NW = HalfWords<T>::NW;
    // exchange kinds: x1 uses 0, 1; x2 uses 2, 3 - or 0, 1 again where the pair barriers make one buffer enough
    constexpr int NK = PairSync<B1, B2, L3>::value ? 2 : 4;
    constexpr int K2 = PairSync<B1, B2, L3>::value ? 0 : 2;
    constexpr int ROW1 = B2 * L3;   // slot distance of x1 neighbours
    constexpr int ROW2 = L3;        // slot distance of x2 neighbours
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Vec* xbuf = reinterpret_cast<Vec*>(smem_raw);                                  // exchange: [NK kinds][NW][NT]
    LVec* lnk = reinterpret_cast<LVec*>(smem_raw + (size_t)NK * NW * NT * sizeof(Vec));   // links: [4 mu][NL][NT]
    unsigned char* hal = smem_raw + (size_t)NK * NW * NT * sizeof(Vec) + (size_t)4 * LL::NL * NT * sizeof(LVec);   // halo slot

    const int site = threadIdx.x;
    const int x3 = site % L3, r2 = (site / L3) % B2, r1 = site / (L3 * B2);
    const int tile = blockIdx.x % G.ntile, seg = blockIdx.x / G.ntile;
    const int x1 = (tile / G.nt2) * B1 + r1, x2 = (tile % G.nt2) * B2 + r2;
    const long long S1 = (long long)G.L2 * L3, S2 = L3;
    const long long ss = ((long long)x1 * G.L2 + x2) * L3 + x3;
    const int ts = seg * G.seg_base + (seg < G.seg_rem ? seg : G.seg_rem);
    const int len = G.seg_base + (seg < G.seg_rem ? 1 : 0);

    const int lane = threadIdx.x & 31;
    // the links of the segment's first slice start their way into the thread's slot
#pragma unroll
    for (int mu = 0; mu < 4; mu++)
#pragma unroll
        for (int p = 0; p < LL::NL; p++)
            cp_async<sizeof(LVec)>(&lnk[(mu * LL::NL + p) * NT + site], gauge + ((long long)mu * LL::NL + p) * G.V + ts * G.S0 + ss);

    // neighbours in x1 / x2: inside the tile (slot index), or outside (global site offset within the slice)
    const bool wrap1 = (G.L1 == B1), wrap2 = (G.L2 == B2);
    const int slot_b1 = (r1 > 0) ? site - ROW1 : (wrap1 ? site + (B1 - 1) * ROW1 : -1);
    const int slot_f1 = (r1 < B1 - 1) ? site + ROW1 : (wrap1 ? site - (B1 - 1) * ROW1 : -1);
    const int slot_b2 = (r2 > 0) ? site - ROW2 : (wrap2 ? site + (B2 - 1) * ROW2 : -1);
    const int slot_f2 = (r2 < B2 - 1) ? site + ROW2 : (wrap2 ? site - (B2 - 1) * ROW2 : -1);
    const bool face_b1 = slot_b1 < 0, face_f1 = slot_f1 < 0, face_b2 = slot_b2 < 0, face_f2 = slot_f2 < 0;
    const long long ss_b1 = (x1 == 0) ? ss + (long long)(G.L1 - 1) * S1 : ss - S1;
    const long long ss_f1 = (x1 == G.L1 - 1) ? ss - (long long)(G.L1 - 1) * S1 : ss + S1;
    const long long ss_b2 = (x2 == 0) ? ss + (long long)(G.L2 - 1) * S2 : ss - S2;
    const long long ss_f2 = (x2 == G.L2 - 1) ? ss - (long long)(G.L2 - 1) * S2 : ss + S2;
    // x3 neighbours: lanes of the same warp (a warp holds 32 / L3 complete x3 rows)
    const int lane_f3 = (lane & ~(L3 - 1)) | ((lane + 1) & (L3 - 1));
    const int lane_b3 = (lane & ~(L3 - 1)) | ((lane + L3 - 1) & (L3 - 1));

    issue_halo<T, RECON, 1, NT>(hal, in, gauge, G.V, site, face_b1, face_f1, ts * G.S0 + ss_b1, ts * G.S0 + ss_f1, site);
    cp_async_commit();

    cx<T> phi_c[12], w0[2][3];
    {
        // the backward time hop of the segment's first slice: U_0(x, t-1)^dagger (1 + gamma_0) phi(x, t-1)
        const int tp = (ts == 0) ? G.L0 - 1 : ts - 1;
        cx<T> psi[12], U[3][3], h[2][3];
        load_spinor<T>(in, G.V, tp * G.S0 + ss, psi);
        load_link<T, RECON>(gauge, G.V, 0, tp * G.S0 + ss, U);
        project<T, 0, +1>(psi, (ts == 0) ? T(G.bc) : T(1), h);
        mul_Udag(U, h, w0);
        load_spinor<T>(in, G.V, ts * G.S0 + ss, phi_c);
    }

    for (int i = 0; i < len; i++) {
        const int t = ts + i;
        const long long st = t * G.S0;
        const long long s = st + ss;
        const bool more = (i + 1 < len);           // the next slice belongs to this segment: prefetch its links
        const long long s_next = s + G.S0;         // (only used when `more`: t + 1 < L0 then)
        cx<T> phi_n[12];
        load_spinor<T>(in, G.V, ((t == G.L0 - 1) ? 0 : st + G.S0) + ss, phi_n);   // next slice of this column
        // this slice's link words and x1 halo (issued one slice ago) have landed
        cp_async_wait_all();

        cx<T> acc[12];
        {
            const T f = T(-2) * mass_term;   // -1/2 acc = (4+m) phi - 1/2 sum(hops)
#pragma unroll
            for (int k = 0; k < 12; k++) acc[k] = {f * phi_c[k].re, f * phi_c[k].im};
        }
        KeptLink<T> kept;
        // ---- x1: send
        if (PairSync<B1, B2, L3>::value) pair_barrier(1 + r2);   // the partner row has finished last slice's x1 receive
        {
            cx<T> U[3][3];
            take_link<T, RECON, NT>(lnk, gauge, G.V, 1, site, more, s_next, U);
            kept.keep(U);
            send_dir<T, RECON, 1, NT, 0>(xbuf, hal, phi_c, U, site, slot_b1, slot_f1, face_b1, face_f1, site);
            // the halo slot is free again: this slice's x2 halo
            issue_halo<T, RECON, 2, NT>(hal, in, gauge, G.V, site, face_b2, face_f2, st + ss_b2, st + ss_f2, site);
            cp_async_commit();
        }
        // ---- x3: the neighbours are lanes of this warp
        {
            cx<T> U[3][3], h[2][3], g[2][3];
            take_link<T, RECON, NT>(lnk, gauge, G.V, 3, site, more, s_next, U);
            project<T, 3, -1>(phi_c, T(1), h);
            shfl_half(h, lane_f3);             // (1 - gamma_3) phi(x + 3^)
            mul_U(U, h, g);
            accumulate<T, 3, -1>(g, acc);
            project<T, 3, +1>(phi_c, T(1), h);
            mul_Udag(U, h, g);
            shfl_half(g, lane_b3);             // U_3(x - 3^)^dagger (1 + gamma_3) phi(x - 3^)
            accumulate<T, 3, +1>(g, acc);
        }
        if (PairSync<B1, B2, L3>::value) pair_barrier(1 + r2);   // x1 half-spinors are in place
        else __syncthreads();                  // ... (and everybody's x2 receive of the last slice is finished)
        {
            cx<T> U[3][3];
            kept.get(U);
            recv_dir<T, 1, NT, 0>(xbuf, U, site, acc);
        }
        // ---- x2: send
        if (PairSync<B1, B2, L3>::value) pair_barrier(3 + r1);   // the partner row has finished last slice's x2 receive
        {
            cx<T> U[3][3];
            take_link<T, RECON, NT>(lnk, gauge, G.V, 2, site, more, s_next, U);
            kept.keep(U);
            // the x2 halo
            cp_async_wait_all();
            send_dir<T, RECON, 2, NT, K2>(xbuf, hal, phi_c, U, site, slot_b2, slot_f2, face_b2, face_f2, site);
            if (more) issue_halo<T, RECON, 1, NT>(hal, in, gauge, G.V, site, face_b1, face_f1, st + G.S0 + ss_b1, st + G.S0 + ss_f1, site);
        }
        // ---- x0: this thread's own column
        {
            cx<T> U[3][3], h[2][3], g[2][3];
            accumulate<T, 0, +1>(w0, acc);     // carried from the previous slice
            take_link<T, RECON, NT>(lnk, gauge, G.V, 0, site, more, s_next, U);
            project<T, 0, -1>(phi_n, (t == G.L0 - 1) ? T(G.bc) : T(1), h);
            mul_U(U, h, g);
            accumulate<T, 0, -1>(g, acc);
            project<T, 0, +1>(phi_c, (t == G.L0 - 1) ? T(G.bc) : T(1), h);
            mul_Udag(U, h, w0);                // the next slice's backward time hop
        }
        cp_async_commit();
        EpiVectors<T, EPI> ev;
        ev.load(G.V, s, s1, v1, s2, v2, s3, v3);   // the fused update's vectors are on their way while the barrier is met
        if (PairSync<B1, B2, L3>::value) pair_barrier(3 + r1);   // x2 half-spinors are in place
        else __syncthreads();                  // ... (and everybody's x1 receive of this slice is finished)
        {
            cx<T> U[3][3];
            kept.get(U);
            recv_dir<T, 2, NT, K2>(xbuf, U, site, acc);
        }
        ev.finish(out, G.V, s, acc, s0, s1, s2, s3);
#pragma unroll
        for (int k = 0; k < 12; k++) phi_c[k] = phi_n[k];
    }
}

// the number of segments along x0 that fills the machine best: CTAs = ntile * nseg are handed to `slots` resident CTA
// slots in rounds; a short segment pays its prologue (one extra spinor + link read per column) more often
int choose_segments(int L0, int ntile, int slots) {
    int best = 1;
    double best_eff = 0.0;
    for (int nseg = 1; nseg <= L0; nseg++) {
        const long long ctas = (long long)ntile * nseg;
        const long long rounds = (ctas + slots - 1) / slots;
        const int longest = (L0 + nseg - 1) / nseg;
        // time ~ rounds * (longest + prologue), work = L0 * ntile / slots
        const double eff = ((double)L0 * ntile / slots) / ((double)rounds * (longest + 0.6));
        if (eff > best_eff + 1e-9) { best_eff = eff; best = nseg; }
    }
    return best;
}

// fp64 plain stencil, one right-hand side, x3 extent 32: the count measured to be fastest (round-3 rows; 32^3 x 32 / 64 /
// 128 and 96 x 16 x 32^2, every candidate timed from a cooled board).  The round model above is right for fp32 but not here, where
// two CTAs per SM leave the kernel latency-bound and a partly filled last round costs little: the FEWEST segments that still give
// about 3.5 rounds of CTAs win (1024 CTAs on 296 slots in all four lattices: 32^3x64 4 segments 284.9 us against 289.0 for the
// model's 8; 32^3x32 147.1 / 151.9; 96x16x32^2 218.6 / 226.4; 32^3x128 564.3 / 565.3) - the prologue (previous slice's spinor and
// link, read without overlap) is dear in fp64.  Only ever fewer segments than the model, the direction that was measured.
// (The fused-epilogue launch prefers segments of 4 slices from a cooled board, 472.9 against 483.0 us, but loses that and more
// inside a sustained loop at the power cap - 505.6 against 492.8 us - so it stays on the model.)
int choose_segments_fp64_plain(int L0, int ntile, int slots, int model) {
    int nseg = (int)((3.4 * slots + ntile - 1) / ntile);
    if (nseg > model) nseg = model;
    if (nseg > L0 / 3) nseg = L0 / 3;
    return nseg < 1 ? 1 : nseg;
}

// ------------------------------------------------------------------------------------------ the fp64 variant
// In fp64 a site's state is twice as large, and the kernel above neither fits the register file (next spinor of the column
// and a whole kept link on top of accumulators, current spinor and carried time hop: 255 registers and spills) nor shared
// memory (135 KB per 128 sites: one CTA of 4 warps per SM).  Same march, same exchange, different staging:
//   * the NEXT spinor of the column is not held in registers: it travels by cp.async into a private slot and is read at the
//     forward time hop, into the registers of the current spinor, which is dead by then;
//   * TWO link slots instead of four, each shared by two directions in turn (A: x1, then x2; B: x3, then x0): a slot is
//     refilled as soon as its link has been read, so a link is in flight for about half a time-slice (2 CTAs per SM alternate:
//     a few microseconds) instead of a whole one;
//   * the halo slot keeps link entries only for the three rows of the tile that have a backward face;
//   * cp.async groups are committed at four points of a slice and every wait is "all but the newest group".
// Shared memory (recon 12): 24 (exchange) + 24 (links) + 24 + 9 (halo) + 24 (next spinor) = 105 KB: two CTAs per SM.
// Tile 2 x 2 x 32 with the pair barriers of the kernel above; x1 and x2 extents of at least 4 (every site of the tile has
// exactly one neighbour outside the tile per direction).
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename T, int RECON, int NT>
__device__ __forceinline__ void read_link_slot(const typename LinkLayout<T, RECON>::LVec* slot, int site, cx<T> (&U)[3][3]) {
    using LL = LinkLayout<T, RECON>;
    typename LL::LVec w[LL::NL];
#pragma unroll
    for (int p = 0; p < LL::NL; p++) w[p] = slot[p * NT + site];
    reconstruct_link<T, RECON>(w, U);
}
template <typename T, int RECON, int NT>
__device__ __forceinline__ void fill_link_slot(typename LinkLayout<T, RECON>::LVec* slot, const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge,
                                               long long V, int mu, int site, long long s) {
    using LL = LinkLayout<T, RECON>;
    const typename LL::LVec* src = gauge + (long long)mu * LL::NL * V + s;
#pragma unroll
    for (int p = 0; p < LL::NL; p++) cp_async<sizeof(typename LL::LVec)>(&slot[p * NT + site], src + p * V);
}

template <typename T, int RECON, bool EPI, int MINB, int L3>
__global__ void __launch_bounds__(128, MINB)
    wilson_Q_tile2_kernel(typename Prec<T>::Vec* out, const typename Prec<T>::Vec* __restrict__ in,
                          const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, TileGeom G, T mass_term, T s0, T s1,
                          const typename Prec<T>::Vec* v1, T s2, const typename Prec<T>::Vec* v2, T s3,
                          const typename Prec<T>::Vec* v3, long long batch_stride) {
    using Vec = typename Prec<T>::Vec;
    using LL = LinkLayout<T, RECON>;
    using LVec = typename LL::LVec;
    {   // blockIdx.y = right-hand side of a batch stored back to back (the links are shared through L2)
        const long long off = (long long)blockIdx.y * batch_stride;
        out += off; in += off;
        if (EPI) { if (v1) v1 += off; if (v2) v2 += off; if (v3) v3 += off; }
    }
    // x3 extent 32: one 2 x 2 x 32 tile per CTA, a warp is one x3 row; x3 extent 16: two independent 2 x 2 x 16 tiles per CTA
    // (neighbours in x2), a warp is the two rows (r2 = 0, 1) of one r1: the x2 partner of a site is in its own warp
    constexpr int NT = 128, NSUB = 32 / L3, SUBT = NT / NSUB;
    constexpr int HLN = 3 * 32;                // halo link entries: the three rows of a tile that have a backward face
    constexpr int NW = HalfWords<T>::NW, NV = Prec<T>::NV;
    constexpr int ROW1 = 2 * L3, ROW2 = L3;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char* sp = smem_raw;
    Vec* xbuf = reinterpret_cast<Vec*>(sp);   sp += (size_t)2 * NW * NT * sizeof(Vec);        // exchange: [2 kinds][NW][NT]
    LVec* lnkA = reinterpret_cast<LVec*>(sp); sp += (size_t)LL::NL * NT * sizeof(LVec);       // link slot A: x1, then x2
    LVec* lnkB = reinterpret_cast<LVec*>(sp); sp += (size_t)LL::NL * NT * sizeof(LVec);       // link slot B: x3, then x0
    unsigned char* hal = sp;                  sp += (size_t)NV * NT * sizeof(Vec) + (size_t)LL::NL * HLN * sizeof(LVec);   // halo slot
    Vec* phis = reinterpret_cast<Vec*>(sp);                                                    // next spinor of the column: [NV][NT]

    const int site = threadIdx.x;
    const int sub = site / SUBT, x3 = site % L3, r2 = (site / L3) % 2, r1 = (site / (2 * L3)) % 2;
    const int tile = blockIdx.x % G.ntile, seg = blockIdx.x / G.ntile;
    const int x1 = (tile / G.nt2) * 2 + r1, x2 = ((tile % G.nt2) * NSUB + sub) * 2 + r2;
    const long long S1 = (long long)G.L2 * L3, S2 = L3;
    const long long ss = ((long long)x1 * G.L2 + x2) * L3 + x3;
    const int ts = seg * G.seg_base + (seg < G.seg_rem ? seg : G.seg_rem);
    const int len = G.seg_base + (seg < G.seg_rem ? 1 : 0);
    const int lane = threadIdx.x & 31;

    // in-tile neighbours (the other row of the pair) and the neighbours outside the tile
    const bool face_b1 = (r1 == 0), face_f1 = !face_b1, face_b2 = (r2 == 0), face_f2 = !face_b2;
    const int slot_b1 = face_b1 ? -1 : site - ROW1, slot_f1 = face_f1 ? -1 : site + ROW1;
    const int slot_b2 = face_b2 ? -1 : site - ROW2, slot_f2 = face_f2 ? -1 : site + ROW2;
    const long long ss_b1 = (x1 == 0) ? ss + (long long)(G.L1 - 1) * S1 : ss - S1;
    const long long ss_f1 = (x1 == G.L1 - 1) ? ss - (long long)(G.L1 - 1) * S1 : ss + S1;
    const long long ss_b2 = (x2 == 0) ? ss + (long long)(G.L2 - 1) * S2 : ss - S2;
    const long long ss_f2 = (x2 == G.L2 - 1) ? ss - (long long)(G.L2 - 1) * S2 : ss + S2;
    // halo link entry of this thread, the same in both directions (private: no other thread ever touches it): rows
    // (r1, r2) = (0, 0) [backward face in x1 and x2], (0, 1) [x1 only], (1, 0) [x2 only]
    const int hidx1 = sub * 3 * L3 + x3 + L3 * (r1 == 0 ? r2 : 2), hidx2 = hidx1;
    const int lane_f3 = (lane & ~(L3 - 1)) | ((lane + 1) & (L3 - 1)), lane_b3 = (lane & ~(L3 - 1)) | ((lane + L3 - 1) & (L3 - 1));
    const int bar1 = (L3 == 32) ? 1 + r2 : 1 + sub;   // the two warps that are x1 partners

    // group a: link 1 and the x1 halo of the first slice; group b: link 3 of the first slice and the spinor of the second
    fill_link_slot<T, RECON, NT>(lnkA, gauge, G.V, 1, site, ts * G.S0 + ss);
    issue_halo<T, RECON, 1, NT, HLN>(hal, in, gauge, G.V, site, face_b1, face_f1, ts * G.S0 + ss_b1, ts * G.S0 + ss_f1, hidx1);
    cp_async_commit();
    fill_link_slot<T, RECON, NT>(lnkB, gauge, G.V, 3, site, ts * G.S0 + ss);
    {
        const long long sn = ((ts == G.L0 - 1) ? 0 : (ts + 1) * G.S0) + ss;
#pragma unroll
        for (int p = 0; p < NV; p++) cp_async<16>(&phis[p * NT + site], in + p * G.V + sn);
    }
    cp_async_commit();

    cx<T> phi_c[12], w0[2][3];
    {
        // the backward time hop of the segment's first slice: U_0(x, t-1)^dagger (1 + gamma_0) phi(x, t-1)
        const int tp = (ts == 0) ? G.L0 - 1 : ts - 1;
        cx<T> psi[12], U[3][3], h[2][3];
        load_spinor<T>(in, G.V, tp * G.S0 + ss, psi);
        load_link<T, RECON>(gauge, G.V, 0, tp * G.S0 + ss, U);
        project<T, 0, +1>(psi, (ts == 0) ? T(G.bc) : T(1), h);
        mul_Udag(U, h, w0);
        load_spinor<T>(in, G.V, ts * G.S0 + ss, phi_c);
    }

    for (int i = 0; i < len; i++) {
        const int t = ts + i;
        const long long st = t * G.S0;
        const long long s = st + ss;
        const bool more = (i + 1 < len);
        cp_async_wait<1>();                        // link 1 and the x1 halo of this slice have landed
        if (EPI && (lane & 7) == 0) {
            // the fused update's vectors of this slice are read after the last barrier, with no registers to load them early:
            // pull their lines (8 lanes = one 128-byte line per plane) into L2 now, a whole slice ahead
            const Vec* vs[3] = {v1, v2, v3};
#pragma unroll
            for (int j = 0; j < 3; j++)
                if (vs[j]) {
#pragma unroll
                    for (int p = 0; p < NV; p++) asm volatile("prefetch.global.L2 [%0];" ::"l"(vs[j] + p * G.V + s));
                }
        }
        cx<T> acc[12];
        {
            const T f = T(-2) * mass_term;
#pragma unroll
            for (int k = 0; k < 12; k++) acc[k] = {f * phi_c[k].re, f * phi_c[k].im};
        }
        KeptLink<T> kept;
        // ---- x1: send
        pair_barrier(bar1);
        {
            cx<T> U[3][3];
            read_link_slot<T, RECON, NT>(lnkA, site, U);
            fill_link_slot<T, RECON, NT>(lnkA, gauge, G.V, 2, site, s);             // slot A: link 2 of this slice
            kept.keep(U);
            send_dir<T, RECON, 1, NT, 0, HLN>(xbuf, hal, phi_c, U, site, slot_b1, slot_f1, face_b1, face_f1, hidx1);
            issue_halo<T, RECON, 2, NT, HLN>(hal, in, gauge, G.V, site, face_b2, face_f2, st + ss_b2, st + ss_f2, hidx2);
            cp_async_commit();                     // group 1
        }
        // ---- x3: lanes of this warp
        cp_async_wait<1>();                        // link 3 (and the next spinor of the column)
        {
            cx<T> U[3][3], h[2][3], g[2][3];
            read_link_slot<T, RECON, NT>(lnkB, site, U);
            fill_link_slot<T, RECON, NT>(lnkB, gauge, G.V, 0, site, s);             // slot B: link 0 of this slice
            cp_async_commit();                     // group 2
            project<T, 3, -1>(phi_c, T(1), h);
            shfl_half(h, lane_f3);
            mul_U(U, h, g);
            accumulate<T, 3, -1>(g, acc);
            project<T, 3, +1>(phi_c, T(1), h);
            mul_Udag(U, h, g);
            shfl_half(g, lane_b3);
            accumulate<T, 3, +1>(g, acc);
        }
        pair_barrier(bar1);                      // x1 half-spinors are in place
        {
            cx<T> U[3][3];
            kept.get(U);
            recv_dir<T, 1, NT, 0>(xbuf, U, site, acc);
        }
        // ---- x2: send
        if (L3 == 32) pair_barrier(3 + r1); else __syncwarp();
        cp_async_wait<1>();                        // link 2 and the x2 halo
        {
            cx<T> U[3][3];
            read_link_slot<T, RECON, NT>(lnkA, site, U);
            if (more) fill_link_slot<T, RECON, NT>(lnkA, gauge, G.V, 1, site, s + G.S0);   // slot A: link 1 of the next slice
            kept.keep(U);
            send_dir<T, RECON, 2, NT, 0, HLN>(xbuf, hal, phi_c, U, site, slot_b2, slot_f2, face_b2, face_f2, hidx2);
            if (more) issue_halo<T, RECON, 1, NT, HLN>(hal, in, gauge, G.V, site, face_b1, face_f1, st + G.S0 + ss_b1, st + G.S0 + ss_f1, hidx1);
            cp_async_commit();                     // group 3
        }
        // ---- x0: this thread's own column
        cp_async_wait<1>();                        // link 0
        {
            cx<T> U[3][3], h[2][3], g[2][3];
            const T ph = (t == G.L0 - 1) ? T(G.bc) : T(1);
            accumulate<T, 0, +1>(w0, acc);         // carried from the previous slice
            read_link_slot<T, RECON, NT>(lnkB, site, U);
            if (more) fill_link_slot<T, RECON, NT>(lnkB, gauge, G.V, 3, site, s + G.S0);   // slot B: link 3 of the next slice
            project<T, 0, +1>(phi_c, ph, h);
            mul_Udag(U, h, w0);                    // the next slice's backward time hop; phi(t) is dead now
            {
                Vec w[NV];
#pragma unroll
                for (int p = 0; p < NV; p++) w[p] = phis[p * NT + site];
                words_to_cx(w, phi_c);             // phi(t + 1)
            }
            if (more) {                            // the slot takes phi(t + 2) (exists: t + 1 <= L0 - 1)
                const long long sn = ((t + 1 == G.L0 - 1) ? 0 : st + 2 * G.S0) + ss;
#pragma unroll
                for (int p = 0; p < NV; p++) cp_async<16>(&phis[p * NT + site], in + p * G.V + sn);
            }
            cp_async_commit();                     // group 4
            project<T, 0, -1>(phi_c, ph, h);
            mul_U(U, h, g);
            accumulate<T, 0, -1>(g, acc);
        }
        EpiVectors<T, EPI> ev;
        ev.load(G.V, s, s1, v1, s2, v2, s3, v3);
        if (L3 == 32) pair_barrier(3 + r1); else __syncwarp();                      // x2 half-spinors are in place
        {
            cx<T> U[3][3];
            kept.get(U);
            recv_dir<T, 2, NT, 0>(xbuf, U, site, acc);
        }
        ev.finish(out, G.V, s, acc, s0, s1, s2, s3);
    }
}

template <typename T, int RECON, bool EPI, int MINB, int L3>
int launch_tile2(nd_ctx* ctx, int nrhs, void* out, const void* in, double m, double s0, double s1, const void* v1, double s2, const void* v2,
                 double s3, const void* v3) {
    using Vec = typename Prec<T>::Vec;
    using LL = LinkLayout<T, RECON>;
    using LVec = typename LL::LVec;
    constexpr int NT = 128;
    constexpr size_t smem = (size_t)2 * HalfWords<T>::NW * NT * sizeof(Vec) + (size_t)2 * LL::NL * NT * sizeof(LVec) +
                            (size_t)Prec<T>::NV * NT * sizeof(Vec) + (size_t)LL::NL * 96 * sizeof(LVec) +
                            (size_t)Prec<T>::NV * NT * sizeof(Vec);
    TileGeom G;
    G.L0 = ctx->dims[0]; G.L1 = ctx->dims[1]; G.L2 = ctx->dims[2];
    G.V = ctx->V;
    G.S0 = (long long)ctx->dims[1] * ctx->dims[2] * ctx->dims[3];
    G.bc = ctx->bc;
    G.nt2 = G.L2 / (2 * (32 / L3));
    G.ntile = (G.L1 / 2) * G.nt2;
    auto kern = wilson_Q_tile2_kernel<T, RECON, EPI, MINB, L3>;
    int& per_sm = ctx->tile_ctas_per_sm[4 + (EPI ? 1 : 0)];
    if (per_sm == 0) {
        ND_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int n = 0;
        ND_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, NT, smem));
        if (n < 1) return nd_fail(ctx, ND_ERR_CUDA, "tiled fp64 stencil does not fit on an SM");
        per_sm = n;
    }
    int nseg = choose_segments(G.L0, G.ntile * nrhs, per_sm * ctx->num_sms);   // a batch = more columns to march along
    if (sizeof(T) == 8 && !EPI && nrhs == 1 && L3 == 32) nseg = choose_segments_fp64_plain(G.L0, G.ntile, per_sm * ctx->num_sms, nseg);
    G.seg_base = G.L0 / nseg;
    G.seg_rem = G.L0 % nseg;
    const dim3 blocks((unsigned)(G.ntile * nseg), (unsigned)nrhs, 1);
    kern<<<blocks, NT, smem, ctx->stream>>>((Vec*)out, (const Vec*)in, (const LVec*)ctx->gauge, G, T(4.0 + m), T(s0), T(s1),
                                            (const Vec*)v1, T(s2), (const Vec*)v2, T(s3), (const Vec*)v3,
                                            (long long)Prec<T>::NV * ctx->V);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

// ------------------------------------------------------------------------------ the tensor-map (TMA) variant
// wilson_Q_tile2_kernel with every prefetch issued as a TMA tensor-map box load (cp.async.bulk.tensor.5d, SASS UTMALDG) instead of
// per-thread cp.async: the spinor and link arrays are described to the TMA unit as 5D tensors
//     [plane][x0][x1][x2][x3 row of 32 128-bit words]     (plane stride = one lattice volume)
// and ONE request moves all planes of one x3 row (a box of 1 x 1 x 1 x 1 row x NP planes: 1.5 KB for a link, 3 KB for a spinor in
// fp32) into the warp's private slot, laid out [plane][lane].  A warp is one row, so lane 0 of every warp issues for its own row
// after a __syncwarp (all lanes have read the slot) and completion is counted in bytes on four mbarriers per warp, one per group
// of the two-slot schedule above: at most 9 requests per warp and slice (plain bulk copies, one per row-plane, would be 21 of 512
// bytes) and no LDGSTS, no per-thread address arithmetic.  Periodic wrap-around is in the box coordinates.  fp32 / fp64, x3
// extent 32.
struct TileMaps {
    CUtensorMap spinor;   // `in`
    CUtensorMap links;    // the context's gauge field
};
__device__ __forceinline__ void tma_row(void* dst, const CUtensorMap* tm, int x2, int x1, int x0, int plane0, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(
                     smem_u32(dst)),
                 "l"(tm), "r"(0), "r"(x2), "r"(x1), "r"(x0), "r"(plane0), "r"(smem_u32(bar))
                 : "memory");
}

template <typename T, int RECON, bool EPI, int MINB>
__global__ void __launch_bounds__(128, MINB)
    wilson_Q_tile3_kernel(typename Prec<T>::Vec* out, const typename Prec<T>::Vec* __restrict__ in,
                          const typename LinkLayout<T, RECON>::LVec* __restrict__ gauge, const __grid_constant__ TileMaps maps,
                          TileGeom G, T mass_term, T s0, T s1, const typename Prec<T>::Vec* v1, T s2, const typename Prec<T>::Vec* v2,
                          T s3, const typename Prec<T>::Vec* v3) {
    using Vec = typename Prec<T>::Vec;
    using LL = LinkLayout<T, RECON>;
    using LVec = typename LL::LVec;
    constexpr int L3 = 32, NT = 128, NL = LL::NL;
    constexpr int NW = HalfWords<T>::NW, NV = Prec<T>::NV;
    constexpr int ROW1 = 2 * L3, ROW2 = L3;
    constexpr unsigned LROW = NL * 32 * sizeof(LVec), SROW = NV * 32 * sizeof(Vec);   // bytes of one link / spinor row box
    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char* sp = smem_raw;
    Vec* xbuf = reinterpret_cast<Vec*>(sp);   sp += (size_t)2 * NW * NT * sizeof(Vec);   // exchange: [2 kinds][NW][NT]
    LVec* lnkA = reinterpret_cast<LVec*>(sp); sp += (size_t)NL * NT * sizeof(LVec);      // per warp [NL][32]: x1, then x2
    LVec* lnkB = reinterpret_cast<LVec*>(sp); sp += (size_t)NL * NT * sizeof(LVec);      // x3, then x0
    Vec* hals = reinterpret_cast<Vec*>(sp);   sp += (size_t)NV * NT * sizeof(Vec);       // halo spinor, per warp [NV][32]
    LVec* hall = reinterpret_cast<LVec*>(sp); sp += (size_t)NL * NT * sizeof(LVec);      // halo link (backward faces)
    Vec* phis = reinterpret_cast<Vec*>(sp);                                               // next spinor of the column
    __shared__ unsigned long long mbar[4][NT / 32];

    const int site = threadIdx.x, lane = site & 31, warp = site >> 5;
    const int x3 = lane, r2 = warp & 1, r1 = warp >> 1;
    const int tile = blockIdx.x % G.ntile, seg = blockIdx.x / G.ntile;
    const int x1 = (tile / G.nt2) * 2 + r1, x2 = (tile % G.nt2) * 2 + r2;
    const long long ss = ((long long)x1 * G.L2 + x2) * L3 + x3;
    const int ts = seg * G.seg_base + (seg < G.seg_rem ? seg : G.seg_rem);
    const int len = G.seg_base + (seg < G.seg_rem ? 1 : 0);
    const bool face_b1 = (r1 == 0), face_f1 = !face_b1, face_b2 = (r2 == 0), face_f2 = !face_b2;
    const int slot_b1 = face_b1 ? -1 : site - ROW1, slot_f1 = face_f1 ? -1 : site + ROW1;
    const int slot_b2 = face_b2 ? -1 : site - ROW2, slot_f2 = face_f2 ? -1 : site + ROW2;
    const int x1n = face_b1 ? (x1 == 0 ? G.L1 - 1 : x1 - 1) : (x1 == G.L1 - 1 ? 0 : x1 + 1);   // the row outside the tile in x1
    const int x2n = face_b2 ? (x2 == 0 ? G.L2 - 1 : x2 - 1) : (x2 == G.L2 - 1 ? 0 : x2 + 1);   // ... and in x2
    const int lane_f3 = (lane + 1) & 31, lane_b3 = (lane + 31) & 31;
    // this warp's private rows in the slots
    LVec* myA = lnkA + warp * NL * 32;
    LVec* myB = lnkB + warp * NL * 32;
    Vec* myhs = hals + warp * NV * 32;
    LVec* myhl = hall + warp * NL * 32;
    Vec* myphi = phis + warp * NV * 32;
    unsigned long long* barA = &mbar[0][warp];   // link 1 + x1 halo
    unsigned long long* barB = &mbar[1][warp];   // link 3 + next spinor
    unsigned long long* bar1 = &mbar[2][warp];   // link 2 + x2 halo
    unsigned long long* bar2 = &mbar[3][warp];   // link 0
    const unsigned bytesA = LROW + SROW + (face_b1 ? LROW : 0u), bytes1 = LROW + SROW + (face_b2 ? LROW : 0u);
    if (lane == 0) {
        mbar_init(barA, 1); mbar_init(barB, 1); mbar_init(bar1, 1); mbar_init(bar2, 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    if (lane == 0) {
        mbar_expect_tx(barA, bytesA);
        tma_row(myA, &maps.links, x2, x1, ts, 1 * NL, barA);
        tma_row(myhs, &maps.spinor, x2, x1n, ts, 0, barA);
        if (face_b1) tma_row(myhl, &maps.links, x2, x1n, ts, 1 * NL, barA);
        mbar_expect_tx(barB, LROW + SROW);
        tma_row(myB, &maps.links, x2, x1, ts, 3 * NL, barB);
        tma_row(myphi, &maps.spinor, x2, x1, (ts == G.L0 - 1) ? 0 : ts + 1, 0, barB);
    }

    cx<T> phi_c[12], w0[2][3];
    {
        const int tp = (ts == 0) ? G.L0 - 1 : ts - 1;
        cx<T> psi[12], U[3][3], h[2][3];
        load_spinor<T>(in, G.V, tp * G.S0 + ss, psi);
        load_link<T, RECON>(gauge, G.V, 0, tp * G.S0 + ss, U);
        project<T, 0, +1>(psi, (ts == 0) ? T(G.bc) : T(1), h);
        mul_Udag(U, h, w0);
        load_spinor<T>(in, G.V, ts * G.S0 + ss, phi_c);
    }

    for (int i = 0; i < len; i++) {
        const int t = ts + i;
        const long long s = t * G.S0 + ss;
        const bool more = (i + 1 < len);
        const unsigned par = i & 1;
        mbar_wait(barA, par);                      // link 1 and the x1 halo of this slice
        cx<T> acc[12];
        {
            const T f = T(-2) * mass_term;
#pragma unroll
            for (int k = 0; k < 12; k++) acc[k] = {f * phi_c[k].re, f * phi_c[k].im};
        }
        KeptLink<T> kept;
        // ---- x1: send
        pair_barrier(1 + r2);
        {
            cx<T> U[3][3], h[2][3], g[2][3];
            {
                LVec w[NL];
#pragma unroll
                for (int p = 0; p < NL; p++) w[p] = myA[p * 32 + lane];
                reconstruct_link<T, RECON>(w, U);
            }
            kept.keep(U);
            if (!face_b1) { project<T, 1, -1>(phi_c, T(1), h); put_half<T, NT>(xbuf, 0, slot_b1, h); }
            if (!face_f1) { project<T, 1, +1>(phi_c, T(1), h); mul_Udag(U, h, g); put_half<T, NT>(xbuf, 1, slot_f1, g); }
            {
                Vec w[NV];
#pragma unroll
                for (int p = 0; p < NV; p++) w[p] = myhs[p * 32 + lane];
                cx<T> psi[12];
                words_to_cx(w, psi);
                if (face_f1) { project<T, 1, -1>(psi, T(1), h); put_half<T, NT>(xbuf, 0, site, h); }
                else {
                    LVec lw[NL];
#pragma unroll
                    for (int p = 0; p < NL; p++) lw[p] = myhl[p * 32 + lane];
                    cx<T> Ub[3][3];
                    reconstruct_link<T, RECON>(lw, Ub);
                    project<T, 1, +1>(psi, T(1), h);
                    mul_Udag(Ub, h, g);
                    put_half<T, NT>(xbuf, 1, site, g);
                }
            }
            __syncwarp();
            if (lane == 0) {                       // group 1: link 2 and the x2 halo of this slice
                mbar_expect_tx(bar1, bytes1);
                tma_row(myA, &maps.links, x2, x1, t, 2 * NL, bar1);
                tma_row(myhs, &maps.spinor, x2n, x1, t, 0, bar1);
                if (face_b2) tma_row(myhl, &maps.links, x2n, x1, t, 2 * NL, bar1);
            }
        }
        // ---- x3: lanes of this warp
        mbar_wait(barB, par);                      // link 3 (and the next spinor of the column)
        {
            cx<T> U[3][3], h[2][3], g[2][3];
            {
                LVec w[NL];
#pragma unroll
                for (int p = 0; p < NL; p++) w[p] = myB[p * 32 + lane];
                reconstruct_link<T, RECON>(w, U);
            }
            __syncwarp();
            if (lane == 0) {                       // group 2: link 0 of this slice
                mbar_expect_tx(bar2, LROW);
                tma_row(myB, &maps.links, x2, x1, t, 0, bar2);
            }
            project<T, 3, -1>(phi_c, T(1), h);
            shfl_half(h, lane_f3);
            mul_U(U, h, g);
            accumulate<T, 3, -1>(g, acc);
            project<T, 3, +1>(phi_c, T(1), h);
            mul_Udag(U, h, g);
            shfl_half(g, lane_b3);
            accumulate<T, 3, +1>(g, acc);
        }
        pair_barrier(1 + r2);                      // x1 half-spinors are in place
        {
            cx<T> U[3][3];
            kept.get(U);
            recv_dir<T, 1, NT, 0>(xbuf, U, site, acc);
        }
        // ---- x2: send
        pair_barrier(3 + r1);
        mbar_wait(bar1, par);                      // link 2 and the x2 halo
        {
            cx<T> U[3][3], h[2][3], g[2][3];
            {
                LVec w[NL];
#pragma unroll
                for (int p = 0; p < NL; p++) w[p] = myA[p * 32 + lane];
                reconstruct_link<T, RECON>(w, U);
            }
            kept.keep(U);
            if (!face_b2) { project<T, 2, -1>(phi_c, T(1), h); put_half<T, NT>(xbuf, 0, slot_b2, h); }
            if (!face_f2) { project<T, 2, +1>(phi_c, T(1), h); mul_Udag(U, h, g); put_half<T, NT>(xbuf, 1, slot_f2, g); }
            {
                Vec w[NV];
#pragma unroll
                for (int p = 0; p < NV; p++) w[p] = myhs[p * 32 + lane];
                cx<T> psi[12];
                words_to_cx(w, psi);
                if (face_f2) { project<T, 2, -1>(psi, T(1), h); put_half<T, NT>(xbuf, 0, site, h); }
                else {
                    LVec lw[NL];
#pragma unroll
                    for (int p = 0; p < NL; p++) lw[p] = myhl[p * 32 + lane];
                    cx<T> Ub[3][3];
                    reconstruct_link<T, RECON>(lw, Ub);
                    project<T, 2, +1>(psi, T(1), h);
                    mul_Udag(Ub, h, g);
                    put_half<T, NT>(xbuf, 1, site, g);
                }
            }
            __syncwarp();
            if (more && lane == 0) {               // group 3: link 1 and the x1 halo of the next slice
                mbar_expect_tx(barA, bytesA);
                tma_row(myA, &maps.links, x2, x1, t + 1, 1 * NL, barA);
                tma_row(myhs, &maps.spinor, x2, x1n, t + 1, 0, barA);
                if (face_b1) tma_row(myhl, &maps.links, x2, x1n, t + 1, 1 * NL, barA);
            }
        }
        // ---- x0: this thread's own column
        mbar_wait(bar2, par);                      // link 0
        {
            cx<T> U[3][3], h[2][3], g[2][3];
            const T ph = (t == G.L0 - 1) ? T(G.bc) : T(1);
            accumulate<T, 0, +1>(w0, acc);
            {
                LVec w[NL];
#pragma unroll
                for (int p = 0; p < NL; p++) w[p] = myB[p * 32 + lane];
                reconstruct_link<T, RECON>(w, U);
            }
            project<T, 0, +1>(phi_c, ph, h);
            mul_Udag(U, h, w0);
            {
                Vec w[NV];
#pragma unroll
                for (int p = 0; p < NV; p++) w[p] = myphi[p * 32 + lane];
                words_to_cx(w, phi_c);             // phi(t + 1)
            }
            __syncwarp();
            if (more && lane == 0) {               // group 4: link 3 of the next slice, phi(t + 2)
                mbar_expect_tx(barB, LROW + SROW);
                tma_row(myB, &maps.links, x2, x1, t + 1, 3 * NL, barB);
                tma_row(myphi, &maps.spinor, x2, x1, (t + 1 == G.L0 - 1) ? 0 : t + 2, 0, barB);
            }
            project<T, 0, -1>(phi_c, ph, h);
            mul_U(U, h, g);
            accumulate<T, 0, -1>(g, acc);
        }
        EpiVectors<T, EPI> ev;
        ev.load(G.V, s, s1, v1, s2, v2, s3, v3);
        pair_barrier(3 + r1);                      // x2 half-spinors are in place
        {
            cx<T> U[3][3];
            kept.get(U);
            recv_dir<T, 2, NT, 0>(xbuf, U, site, acc);
        }
        ev.finish(out, G.V, s, acc, s0, s1, s2, s3);
    }
}

// tensor map of a plane-SoA array of 128-bit (or 64-bit: fp32 recon 18) words: dims (fastest first) reals of an x3 row, x2, x1, x0,
// planes; box = one x3 row x `box_planes` planes
typedef CUresult (*nd_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time dependency on libcuda), resolved once per process
nd_encode_tiled_fn tensor_map_encoder() {
    static std::once_flag once;
    static nd_encode_tiled_fn encode = nullptr;
    std::call_once(once, [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess && fn && q == cudaDriverEntryPointSuccess)
            encode = (nd_encode_tiled_fn)fn;
    });
    return encode;
}
// The maps are cached in the context (nd_tmap_slot): the link map is encoded once, spinor maps once per `in` pointer among the
// last ND_TMAP_SLOTS arrays - the Clenshaw loop cycles through four - so a launch outside a CUDA graph makes no driver call.
int make_row_map(nd_ctx* ctx, CUtensorMap* tm, const void* base, int word_bytes, int planes, int box_planes) {
    static_assert(sizeof(CUtensorMap) == sizeof(nd_tmap_slot::map), "opaque copy of CUtensorMap in nd_internal.cuh");
    for (int i = 0; i < ND_TMAP_SLOTS; i++) {
        const nd_tmap_slot& c = ctx->tmaps[i];
        if (c.base == base && c.word_bytes == word_bytes && c.planes == planes && c.box_planes == box_planes) {
            memcpy(tm, c.map, sizeof(CUtensorMap));
            return ND_OK;
        }
    }
    const nd_encode_tiled_fn encode = tensor_map_encoder();
    if (!encode) return nd_fail(ctx, ND_ERR_CUDA, "cuTensorMapEncodeTiled is not available in this driver");
    const int rb = ctx->prec / 8;                                   // bytes of a real
    const cuuint64_t row = (cuuint64_t)ctx->dims[3] * word_bytes;   // bytes of an x3 row of one plane
    const cuuint64_t dims[5] = {row / rb, (cuuint64_t)ctx->dims[2], (cuuint64_t)ctx->dims[1], (cuuint64_t)ctx->dims[0], (cuuint64_t)planes};
    const cuuint64_t strides[4] = {row, row * ctx->dims[2], row * ctx->dims[2] * ctx->dims[1], (cuuint64_t)ctx->V * word_bytes};
    const cuuint32_t box[5] = {(cuuint32_t)(row / rb), 1, 1, 1, (cuuint32_t)box_planes};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = encode(tm, ctx->prec == 32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<void*>(base),
                              dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return nd_fail(ctx, ND_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    nd_tmap_slot& c = ctx->tmaps[ctx->tmap_next];
    ctx->tmap_next = (ctx->tmap_next + 1) % ND_TMAP_SLOTS;
    c.base = base; c.word_bytes = word_bytes; c.planes = planes; c.box_planes = box_planes;
    memcpy(c.map, tm, sizeof(CUtensorMap));
    return ND_OK;
}

template <typename T, int RECON, bool EPI, int MINB>
int launch_tile3(nd_ctx* ctx, void* out, const void* in, double m, double s0, double s1, const void* v1, double s2, const void* v2,
                 double s3, const void* v3) {
    using Vec = typename Prec<T>::Vec;
    using LL = LinkLayout<T, RECON>;
    using LVec = typename LL::LVec;
    constexpr int NT = 128;
    constexpr size_t smem = (size_t)2 * HalfWords<T>::NW * NT * sizeof(Vec) + (size_t)3 * LL::NL * NT * sizeof(LVec) +
                            (size_t)2 * Prec<T>::NV * NT * sizeof(Vec);
    TileGeom G;
    G.L0 = ctx->dims[0]; G.L1 = ctx->dims[1]; G.L2 = ctx->dims[2];
    G.V = ctx->V;
    G.S0 = (long long)ctx->dims[1] * ctx->dims[2] * ctx->dims[3];
    G.bc = ctx->bc;
    G.nt2 = G.L2 / 2;
    G.ntile = (G.L1 / 2) * G.nt2;
    TileMaps maps;
    int rc = make_row_map(ctx, &maps.spinor, in, (int)sizeof(Vec), Prec<T>::NV, Prec<T>::NV);
    if (rc == ND_OK) rc = make_row_map(ctx, &maps.links, ctx->gauge, (int)sizeof(LVec), 4 * LL::NL, LL::NL);
    if (rc != ND_OK) return rc;
    auto kern = wilson_Q_tile3_kernel<T, RECON, EPI, MINB>;
    int& per_sm = ctx->tile_ctas_per_sm[6 + (EPI ? 1 : 0)];
    if (per_sm == 0) {
        ND_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int n = 0;
        ND_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, NT, smem));
        if (n < 1) return nd_fail(ctx, ND_ERR_CUDA, "tensor-map stencil does not fit on an SM");
        per_sm = n;
    }
    const int nseg = choose_segments(G.L0, G.ntile, per_sm * ctx->num_sms);
    G.seg_base = G.L0 / nseg;
    G.seg_rem = G.L0 % nseg;
    const unsigned blocks = (unsigned)(G.ntile * nseg);
    kern<<<blocks, NT, smem, ctx->stream>>>((Vec*)out, (const Vec*)in, (const LVec*)ctx->gauge, maps, G, T(4.0 + m), T(s0), T(s1),
                                            (const Vec*)v1, T(s2), (const Vec*)v2, T(s3), (const Vec*)v3);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

template <typename T, int RECON, bool EPI, int B1, int B2, int L3, int MINB>
int launch_tile(nd_ctx* ctx, void* out, const void* in, double m, double s0, double s1, const void* v1, double s2, const void* v2,
                double s3, const void* v3) {
    using Vec = typename Prec<T>::Vec;
    using LVec = typename LinkLayout<T, RECON>::LVec;
    constexpr int NT = B1 * B2 * L3;
    constexpr int NW = HalfWords<T>::NW;
    // exchange buffer(s) + 4 link slots + halo slot (spinor + 1 link)
    constexpr size_t smem = (size_t)(PairSync<B1, B2, L3>::value ? 2 : 4) * NW * NT * sizeof(Vec) +
                            (size_t)5 * LinkLayout<T, RECON>::NL * NT * sizeof(LVec) + (size_t)Prec<T>::NV * NT * sizeof(Vec);
    TileGeom G;
    G.L0 = ctx->dims[0]; G.L1 = ctx->dims[1]; G.L2 = ctx->dims[2];
    G.V = ctx->V;
    G.S0 = (long long)ctx->dims[1] * ctx->dims[2] * ctx->dims[3];
    G.bc = ctx->bc;
    G.nt2 = G.L2 / B2;
    G.ntile = (G.L1 / B1) * G.nt2;
    auto kern = wilson_Q_tile_kernel<T, RECON, EPI, B1, B2, L3, MINB>;
    int& per_sm = ctx->tile_ctas_per_sm[EPI ? 1 : 0];
    if (per_sm == 0) {
        ND_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int n = 0;
        ND_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, NT, smem));
        if (n < 1) return nd_fail(ctx, ND_ERR_CUDA, "tiled stencil does not fit on an SM");
        per_sm = n;
    }
    const int nseg = choose_segments(G.L0, G.ntile, per_sm * ctx->num_sms);
    G.seg_base = G.L0 / nseg;
    G.seg_rem = G.L0 % nseg;
    const unsigned blocks = (unsigned)(G.ntile * nseg);
    kern<<<blocks, NT, smem, ctx->stream>>>((Vec*)out, (const Vec*)in, (const LVec*)ctx->gauge, G, T(4.0 + m), T(s0), T(s1),
                                            (const Vec*)v1, T(s2), (const Vec*)v2, T(s3), (const Vec*)v3);
    ND_LAUNCHED(ctx);
    return ND_OK;
}

// The four-slot kernel, fp32 only (ND_STENCIL_TILE4; the default is the two-slot kernel, which grew out of it).  Registers per
// thread: the plain kernel fits 3 CTAs of 128 threads per SM (168 registers), the fused-epilogue kernel holds the three update
// vectors of its site as well and runs 2 CTAs per SM.  (Its variant with TMA bulk copies - cp.async.bulk, one 512-byte row-plane
// per lane, 21 requests per warp and slice: 188 / 257 us against 144 / 224 us on 32^3x64 - has been replaced by the tensor-map
// kernel above.)
template <int RECON>
int launch_tile_shape(nd_ctx* ctx, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1, double s2,
                      const void* v2, double s3, const void* v3) {
    if (epi) return launch_tile<float, RECON, true, 2, 2, 32, 2>(ctx, out, in, m, s0, s1, v1, s2, v2, s3, v3);
    return launch_tile<float, RECON, false, 2, 2, 32, 3>(ctx, out, in, m, 1, 0, nullptr, 0, nullptr, 0, nullptr);
}

}  // namespace

// Lattices the tiled kernels take: x3 extent 32 (tile 2 x 2 x 32: a warp is one x3 row), even x1 / x2 extents, and enough tiles
// to give every SM work; x1, x2 extents >= 4 for the two-slot kernel (every site of a tile has exactly one outside neighbour
// per direction); fp64: recon 12 / 8 only (with 9 link words per slot two CTAs no longer fit an SM).
// (at least ND_TILE_MIN_CTA_SLICES_PER_SM slices of 128 sites per SM: below that the segments along x0 get so short that their
// prologue - one extra spinor and link per column - eats the gain; 16^3x32 has 6.9 and runs 12.3 us site vs 14.4 us tiled in fp32)
constexpr long long ND_TILE_MIN_CTA_SLICES_PER_SM = 8;
bool ndi_tile_geometry(const nd_ctx* ctx) {
    const int L1 = ctx->dims[1], L2 = ctx->dims[2], L3 = ctx->dims[3];
    if (L3 != 32 && L3 != 16) return false;
    if (L1 % 2 != 0 || L2 % (64 / L3) != 0) return false;      // x3 extent 16: a CTA takes two tiles side by side in x2
    if (L1 < 4 || L2 < 4) return false;
    if (ctx->prec == 64 && ctx->recon == 18) return false;
    return true;
}
// ... for nrhs right-hand sides per launch (a batch on a small lattice is as good as one source on a large one)
bool ndi_tile_worthwhile(const nd_ctx* ctx, int nrhs) { return ctx->V * nrhs / 128 >= ND_TILE_MIN_CTA_SLICES_PER_SM * ctx->num_sms; }
bool ndi_tile_supported(const nd_ctx* ctx) { return ndi_tile_geometry(ctx) && ndi_tile_worthwhile(ctx, 1); }

// fp32: 3 CTAs of 128 threads per SM for the plain stencil (145 - 161 registers), 2 for the fused epilogue (the three update vectors of
// the site are loaded before the last barrier); fp64: 2 CTAs per SM (255 registers, 105 KB shared memory)
template <typename T, int RECON, int MINB, int MINB_EPI>
static int launch_tile2_shape(nd_ctx* ctx, int nrhs, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1,
                              double s2, const void* v2, double s3, const void* v3) {
    if (ctx->dims[3] == 16) {
        if (epi) return launch_tile2<T, RECON, true, MINB_EPI, 16>(ctx, nrhs, out, in, m, s0, s1, v1, s2, v2, s3, v3);
        return launch_tile2<T, RECON, false, MINB, 16>(ctx, nrhs, out, in, m, 1, 0, nullptr, 0, nullptr, 0, nullptr);
    }
    if (epi) return launch_tile2<T, RECON, true, MINB_EPI, 32>(ctx, nrhs, out, in, m, s0, s1, v1, s2, v2, s3, v3);
    return launch_tile2<T, RECON, false, MINB, 32>(ctx, nrhs, out, in, m, 1, 0, nullptr, 0, nullptr, 0, nullptr);
}

template <typename T, int RECON, int MINB, int MINB_EPI>
static int launch_tile3_shape(nd_ctx* ctx, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1, double s2,
                              const void* v2, double s3, const void* v3) {
    if (epi) return launch_tile3<T, RECON, true, MINB_EPI>(ctx, out, in, m, s0, s1, v1, s2, v2, s3, v3);
    return launch_tile3<T, RECON, false, MINB>(ctx, out, in, m, 1, 0, nullptr, 0, nullptr, 0, nullptr);
}

// Which kernel one stencil call runs.  Auto = the fastest measured on 32^3x64 (us per launch, tile vs site):
//   fp32 recon 12 / 8 / 18: plain 139 / 148 / 171 vs 167 / 185 / 196, fused epilogue 224 / 226 / 252 vs 247 / 239 / 279
//   fp64 recon 12 / 8: plain 289 / 382 vs 344 / 417; fused 491 / 539 vs 502 / 535 (all at 87-89 % of the HBM peak): fused with recon 12 only
//   fp64 recon 8, plain, one source, x3 extent 32: the tensor-map loads (363 vs 382 us) - the per-thread cp.async address arithmetic
//   competes with the 8-parameter reconstruction for issue slots
// A batch of right-hand sides on a small lattice marches as many columns as one source on a large one (ndi_tile_worthwhile): 16^3x32
// takes the tiled kernel from 2 sources on.
int ndi_select_stencil(const nd_ctx* ctx, bool epi, int nrhs) {
    const int v = ctx->stencil_variant;
    if (v != ND_STENCIL_AUTO) return (v == ND_STENCIL_TILE4 && ctx->prec == 64) ? (int)ND_STENCIL_TILE : v;   // (nd_set_stencil_variant refuses that pair)
    if (!(ndi_tile_geometry(ctx) && ndi_tile_worthwhile(ctx, nrhs) && (ctx->prec == 32 || !epi || ctx->recon == 12))) return ND_STENCIL_SITE;
    if (ctx->prec == 64 && ctx->recon == 8 && !epi && nrhs == 1 && ctx->dims[3] == 32) return ND_STENCIL_TILE_TMA;
    return ND_STENCIL_TILE;
}

// ND_STENCIL_TILE: the two-slot kernel wilson_Q_tile2_kernel; ND_STENCIL_TILE_TMA: the same schedule with tensor-map
// loads, wilson_Q_tile3_kernel (x3 extent 32); ND_STENCIL_TILE4 (fp32, x3 extent 32): the four-slot kernel wilson_Q_tile_kernel
int ndi_apply_Q_tile(nd_ctx* ctx, int nrhs, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1, double s2,
                     const void* v2, double s3, const void* v3) {
    if (nrhs > 1 && (ctx->stencil_variant == ND_STENCIL_TILE_TMA || ctx->stencil_variant == ND_STENCIL_TILE4)) {
        // the variants kept for comparison take one right-hand side per launch
        const size_t sb = nd_spinor_bytes(ctx);
        for (int j = 0; j < nrhs; j++) {
            const size_t o = (size_t)j * sb;
            const int rc = ndi_apply_Q_tile(ctx, 1, (char*)out + o, (const char*)in + o, m, epi, s0, s1, v1 ? (const char*)v1 + o : nullptr, s2,
                                            v2 ? (const char*)v2 + o : nullptr, s3, v3 ? (const char*)v3 + o : nullptr);
            if (rc != ND_OK) return rc;
        }
        return ND_OK;
    }
    const int sel = ndi_select_stencil(ctx, epi, nrhs);
    if (sel == ND_STENCIL_TILE_TMA) {
        if (ctx->prec == 64) {
            if (ctx->recon == 12) return launch_tile3_shape<double, 12, 2, 2>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
            return launch_tile3_shape<double, 8, 2, 2>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
        }
        if (ctx->recon == 18) return launch_tile3_shape<float, 18, 3, 2>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
        if (ctx->recon == 12) return launch_tile3_shape<float, 12, 3, 2>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
        return launch_tile3_shape<float, 8, 3, 2>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
    }
    if (ctx->prec == 64) {
        if (ctx->recon == 12) return launch_tile2_shape<double, 12, 2, 2>(ctx, nrhs, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
        return launch_tile2_shape<double, 8, 2, 2>(ctx, nrhs, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
    }
    if (sel == ND_STENCIL_TILE4) {
        if (ctx->recon == 18) return launch_tile_shape<18>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
        if (ctx->recon == 12) return launch_tile_shape<12>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
        return launch_tile_shape<8>(ctx, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
    }
    if (ctx->recon == 18) return launch_tile2_shape<float, 18, 3, 2>(ctx, nrhs, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
    if (ctx->recon == 12) return launch_tile2_shape<float, 12, 3, 2>(ctx, nrhs, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
    return launch_tile2_shape<float, 8, 3, 2>(ctx, nrhs, out, in, m, epi, s0, s1, v1, s2, v2, s3, v3);
}
