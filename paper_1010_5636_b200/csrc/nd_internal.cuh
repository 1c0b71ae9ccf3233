// nd_internal.cuh - shared declarations of the CUDA path (context, device layout traits, complex helpers).
// Product code: nothing here is shared with oracle/.
//
// Device layout ("the data layout ... coalescing"):
//   site index s = ((x0*L1 + x1)*L2 + x2)*L3 + x3  (x3 fastest, the warp runs along x3)
//   spinor : NV planes of 128-bit words, word (p, s) at  f[p*V + s]
//            fp32: NV = 6,  float4  = reals 4p..4p+3 of the 24 reals (spin-major, colour, re/im)
//            fp64: NV = 12, double2 = complex component p = spin*3 + colour
//   links  : word (mu, p, s) at g[(mu*NL + p)*V + s]; the P = recon reals of a link in NL words of LVec
//            P=18: rows a,b,c (9 complex); P=12: rows a,b (eq. 2.3 on rows); P=8: a2,a3,b1,theta1,theta2
#pragma once
#include <cuda_runtime.h>

#include <cstdio>
#include <string>
#include <vector>

#include "../../include/nd_b200.h"

struct nd_graph_entry {
    void* out;
    const void* in;
    void* work;
    int kind;            // 0 sign, 1 D_N / D_N^m
    double pa, pb;       // out = pa*in + pb*gamma5 sign(Q) in
    cudaGraphExec_t exec;
    long long nodes;     // kernel launches one replay stands for
    int nrhs;
};

// A cached CUtensorMap of the tensor-map stencil (wilson_tile.cu): the map encodes only the base address and the shape of the
// array, so it stays valid for as long as an array of that shape lives at that address (nd_set_gauge rewrites the links in place).
struct nd_tmap_slot {
    const void* base;       // nullptr: empty
    int word_bytes, planes, box_planes;
    alignas(64) unsigned char map[128];   // CUtensorMap, kept opaque here (cuda.h is included by wilson_tile.cu only)
};
constexpr int ND_TMAP_SLOTS = 8;

struct nd_ctx {
    int dims[4];
    long long V;
    int prec, recon, bc;
    int device;
    cudaStream_t stream;
    void* gauge;
    size_t gauge_bytes;
    bool gauge_set;
    double gstats[4];
    // reductions
    double* d_partial;   // [ND_MAX_RED_BLOCKS * 2 * ND_MAX_BLOCK_L]
    double* d_result;    // [2 * ND_MAX_BLOCK_L * 2]
    double* h_result;    // pinned, same size
    double* d_coef;      // [2 * ND_MAX_BLOCK_L] device copy of block-axpy coefficients
    double* d_nu;        // [ND_MAX_BLOCK_L] Ritz values on the device (sign of nu_k)
    // sign polynomial
    std::vector<double> cheb;
    int n;
    double eps, qnorm, m_sign;
    bool poly_set;
    // low modes
    int l;
    const void* u;
    std::vector<double> nu;
    std::vector<nd_graph_entry> graphs;
    long long launches;
    bool capturing;
    int num_sms;
    int hop_max_sites;  // lattices below this volume use the hop-parallel stencil (wilson.cu)
    int tile_lb[3];     // stencil CTA tile: log2 extents along x1, x2, x3
    int tile_threads;   // sites per tile (0: linear mapping)
    bool dot_configured;        // block_dot_cols_kernel shared-memory attributes set
    bool tile_ok;               // the tiled marching stencil (wilson_tile.cu) takes this lattice
    int stencil_variant;        // ND_STENCIL_* (nd_set_stencil_variant)
    nd_tmap_slot tmaps[ND_TMAP_SLOTS];   // link map + the spinor maps of the last few `in` pointers, replaced round robin
    int tmap_next;
    int tile_ctas_per_sm[8];    // resident CTAs per SM of the tiled kernels ({four-slot, -, two-slot, tensor map} x {plain, fused}), 0 = not queried yet
    // domain decomposition along x0 (shard.cu): this context is the local lattice of rank shard_rank of shard_n
    int shard_rank, shard_n;
    bool in_shard_call;         // the local stencil of a sharded application is being enqueued
    void* halo[4];              // send_next, send_prev, recv_prev, recv_next: half-spinor faces (nd_halo_bytes each)
    // peer-to-peer mode (nd_set_halo_peers): faces are STORED by halo_pack straight into the neighbours' receive windows
    // [parity 2][from_prev, from_next][nd_halo_bytes]; nullptr = callback transfers through halo[0..3]
    void* peer_own;             // this rank's receive window
    void* peer_next;            // the next rank's window (its from_prev faces are written by this rank)
    void* peer_prev;            // the previous rank's window (its from_next faces)
    int halo_parity;
    nd_exchange_start_fn exchange_start;
    nd_exchange_wait_fn exchange_wait;
    nd_allreduce_fn allreduce;
    void* comm_user;
    char err[512];
};

constexpr int ND_MAX_BLOCK_L = 256;     // max vectors in a block dot / block axpy
constexpr int ND_MAX_RED_BLOCKS = 1184; // 8 x 148
constexpr int ND_MAX_RHS = 16;          // right-hand sides of one nd_apply_*_multi call

int nd_fail(nd_ctx* ctx, int code, const char* fmt, ...);
int nd_cuda_check(nd_ctx* ctx, cudaError_t e, const char* what);
#define ND_CUDA(ctx, call)                                         \
    do {                                                           \
        int _rc = nd_cuda_check((ctx), (call), #call);             \
        if (_rc != ND_OK) return _rc;                              \
    } while (0)
#define ND_LAUNCHED(ctx)                                           \
    do {                                                           \
        (ctx)->launches++;                                         \
        int _rc = nd_cuda_check((ctx), cudaGetLastError(), "launch"); \
        if (_rc != ND_OK) return _rc;                              \
    } while (0)

// ---------------------------------------------------------------------------------------- layout traits
template <typename T> struct Prec;
template <> struct Prec<float> {
    using Vec = float4;
    static constexpr int NV = 6;
};
template <> struct Prec<double> {
    using Vec = double2;
    static constexpr int NV = 12;
};

template <typename T, int RECON> struct LinkLayout;
template <> struct LinkLayout<float, 18> { using LVec = float2;  static constexpr int NL = 9; };
template <> struct LinkLayout<float, 12> { using LVec = float4;  static constexpr int NL = 3; };
template <> struct LinkLayout<float, 8>  { using LVec = float4;  static constexpr int NL = 2; };
template <> struct LinkLayout<double, 18> { using LVec = double2; static constexpr int NL = 9; };
template <> struct LinkLayout<double, 12> { using LVec = double2; static constexpr int NL = 6; };
template <> struct LinkLayout<double, 8>  { using LVec = double2; static constexpr int NL = 4; };

// ---------------------------------------------------------------------------------------------- complex
template <typename T> struct cx {
    T re, im;
};
template <typename T> __host__ __device__ __forceinline__ cx<T> mk(T re, T im) { return cx<T>{re, im}; }
template <typename T> __host__ __device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return {a.re + b.re, a.im + b.im}; }
template <typename T> __host__ __device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return {a.re - b.re, a.im - b.im}; }
template <typename T> __host__ __device__ __forceinline__ cx<T> operator*(cx<T> a, cx<T> b) {
    return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re};
}
template <typename T> __host__ __device__ __forceinline__ cx<T> cj(cx<T> a) { return {a.re, -a.im}; }
template <typename T> __host__ __device__ __forceinline__ cx<T> times_i(cx<T> a) { return {-a.im, a.re}; }
template <typename T> __host__ __device__ __forceinline__ cx<T> times_mi(cx<T> a) { return {a.im, -a.re}; }
// acc += a * b
template <typename T> __host__ __device__ __forceinline__ void cfma(cx<T>& acc, cx<T> a, cx<T> b) {
    acc.re = fma(a.re, b.re, acc.re);
    acc.re = fma(-a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im);
    acc.im = fma(a.im, b.re, acc.im);
}
// acc += conj(a) * b
template <typename T> __host__ __device__ __forceinline__ void cfma_cj(cx<T>& acc, cx<T> a, cx<T> b) {
    acc.re = fma(a.re, b.re, acc.re);
    acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im);
    acc.im = fma(-a.im, b.re, acc.im);
}

// 12 complex components of a spinor <-> the 128-bit words of its planes
__device__ __forceinline__ void words_to_cx(const float4 (&w)[6], cx<float> (&c)[12]) {
#pragma unroll
    for (int p = 0; p < 6; p++) {
        c[2 * p] = {w[p].x, w[p].y};
        c[2 * p + 1] = {w[p].z, w[p].w};
    }
}
__device__ __forceinline__ void words_to_cx(const double2 (&w)[12], cx<double> (&c)[12]) {
#pragma unroll
    for (int p = 0; p < 12; p++) c[p] = {w[p].x, w[p].y};
}
__device__ __forceinline__ void cx_to_words(const cx<float> (&c)[12], float4 (&w)[6]) {
#pragma unroll
    for (int p = 0; p < 6; p++) w[p] = make_float4(c[2 * p].re, c[2 * p].im, c[2 * p + 1].re, c[2 * p + 1].im);
}
__device__ __forceinline__ void cx_to_words(const cx<double> (&c)[12], double2 (&w)[12]) {
#pragma unroll
    for (int p = 0; p < 12; p++) w[p] = make_double2(c[p].re, c[p].im);
}

// ---------------------------------------------------------------------------- internal entry points (per TU)
int ndi_apply_Q(nd_ctx* ctx, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1,
                double s2, const void* v2, double s3, const void* v3);
bool ndi_tile_supported(const nd_ctx* ctx);                 // geometry and, for one right-hand side, enough sites
bool ndi_tile_geometry(const nd_ctx* ctx);
bool ndi_tile_worthwhile(const nd_ctx* ctx, int nrhs);
// THE choice of stencil kernel for one call (plain / fused epilogue, nrhs right-hand sides): ND_STENCIL_SITE, _TILE, _TILE_TMA or
// _TILE4, never _AUTO.  The dispatch in wilson.cu / wilson_tile.cu and nd_get_stencil_variant_for both go through it.
int ndi_select_stencil(const nd_ctx* ctx, bool epi, int nrhs);
int ndi_apply_Q_tile(nd_ctx* ctx, int nrhs, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1, double s2,
                     const void* v2, double s3, const void* v3);
int ndi_apply_Q_batch(nd_ctx* ctx, int nrhs, void* out, const void* in, double m, bool epi, double s0, double s1, const void* v1,
                      double s2, const void* v2, double s3, const void* v3);
int ndi_halo_pack(nd_ctx* ctx, const void* in);                 // faces of `in` -> halo[0], halo[1]
int ndi_halo_apply(nd_ctx* ctx, void* out, double s0);          // halo[2], halo[3] -> the boundary slices of out
int ndi_allreduce(nd_ctx* ctx, double* d_buf, int n);           // sum over ranks (no-op unless sharded)
int ndi_block_dot_dev(nd_ctx* ctx, int l, const void* v, const void* x, double* d_out);   // d_out: 2l doubles (device)
int ndi_block_dot_cols_dev(nd_ctx* ctx, int l, const void* v, int nc, const void* const* cols, double* d_out);   // d_out[(c*l+k)*2+ri]
int ndi_block_axpy_batch_dev(nd_ctx* ctx, int l, int nb, const double* d_coef, const void* v, void* y, int mode, const void* eta,
                             double pa, double pb);
int ndi_block_dot2_dev(nd_ctx* ctx, int l, const void* v, const void* x0, const void* x1, double* d_out);  // 4l doubles
int ndi_block_axpy_dev(nd_ctx* ctx, int l, const double* d_coef, const void* v, void* y, int mode, const void* eta, double pa,
                       double pb);   // mode 1: y <- pa*eta + pb*gamma5(y + sum_k a_k v_k)
int ndi_apply_DNm(nd_ctx* ctx, void* out, const void* in, double pa, double pb, void* work, int use_graph);
int ndi_block_gram_dev(nd_ctx* ctx, int l, const void* v, int nx, const void* x, double* d_out);      // d_out[(j*l+k)*2+c]
int ndi_block_rotate_dev(nd_ctx* ctx, int l, const double* d_coef, const void* v, int ny, void* y);  // coef[(j*l+i)*2+c]
int ndi_block_resid(nd_ctx* ctx, int k, const void* x, const void* y, const double* nu, double* rho);   // rho_j = ||y_j - nu_j x_j||
int ndi_chiral_combine(nd_ctx* ctx, int sigma, void* y, const void* u, double c);   // y <- P_sigma u + c y
int ndi_read_result(nd_ctx* ctx, const double* d_src, double* h_dst, int n);              // sync copy to host
int ndi_drop_graphs(nd_ctx* ctx);
constexpr int ND_RESULT_DOUBLES = 4 * ND_MAX_BLOCK_L;
