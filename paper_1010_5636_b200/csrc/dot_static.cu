// dot_static.cu - nd_dot_static: the spinor inner product <x, y> (BLAS-1 of BASELINE.json north_star; the reductions behind
// PAPER.md:L66 / L79-84) for callers that are not allowed to allocate device memory.
//
// Who needs this.  Every other reduction of the library goes through a context, and nd_create reserves the context's
// partial-sum buffer with cudaMalloc.  Some hosts of this library cannot do that at all:
//   - a plug-in living inside an application whose own pool has already claimed the GPU's memory (a cudaMalloc there fails,
//     or takes memory the application believes it owns);
//   - code running in a phase where the allocator must not be touched - cudaMalloc and cudaFree synchronise the whole device
//     and take driver locks, which a latency-bound measurement loop or a region between other people's asynchronous work
//     cannot afford;
//   - processes under a fixed memory budget (MPS limits, a shared GPU) that want the library's footprint known at load time.
// For them this file offers one call that needs no context and performs no allocation of any kind: its partial sums live
// in a file-scope __device__ array that is part of the library image.  Every GPU on which the library's kernels are loaded
// holds that array (ND_DOT_STATIC_SCRATCH_BYTES = 256 KiB) from module load until the process exits; it is never freed.
//
// The kernel is a variant of block_dot_cols_kernel (blas.cu) for one vector and one column: a CTA owns one range of
// DOT_RANGE consecutive sites, accumulates conj(x) y in fp64 registers (both precisions), reduces through warp shuffles and
// shared memory and writes ONE (re, im) pair into its own slot of the static array; a second single-CTA kernel adds the
// slots in a fixed order.  No atomics, so the result is bitwise reproducible and does not depend on the GPU's SM count.
// One slot per range is what bounds the lattice size: ND_DOT_STATIC_MAX_SITES = slots * DOT_RANGE.
//
// Sharing.  All calls on a device use the same array.  Nothing in it has to start at zero: a call writes slots
// [0, nblocks) and afterwards reads exactly those, so whatever an earlier call left behind (also in slots >= nblocks) is
// never looked at.  Two calls whose kernels may run at the same time on one GPU (different streams, different host threads,
// different processes do NOT share - each process has its own module image) would overwrite each other's slots: the caller
// must order them, e.g. by issuing them on one stream.
//
// Address of the array.  In host code the name g_dot_scratch is only a handle for the runtime, not a device pointer - passed
// to a kernel it would fault (or, on systems where the GPU can reach host memory, quietly use host memory).  The device
// address is looked up with cudaGetSymbolAddress once per device, with that device current, the first time the entry point
// is used on it, and cached.  That first call on a device should be made outside any stream capture.
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "nd_internal.cuh"

namespace {

constexpr int DOT_THREADS = 128;
constexpr int DOT_WARPS = DOT_THREADS / 32;
constexpr int DOT_SITES_PER_THREAD = 2;
constexpr int DOT_RANGE = DOT_THREADS * DOT_SITES_PER_THREAD;                       // sites per CTA
constexpr long long DOT_SLOTS = ND_DOT_STATIC_MAX_SITES / DOT_RANGE;                // 16384 CTAs at most
constexpr int FINAL_THREADS = 256;
constexpr int MAX_DEVICES = 64;

static_assert(ND_DOT_STATIC_MAX_SITES % DOT_RANGE == 0, "whole ranges");
static_assert(DOT_SLOTS * 2 * sizeof(double) == ND_DOT_STATIC_SCRATCH_BYTES, "header states the size of the static array");

// partial sums: slot b = (re, im) of CTA b.  Lives in the library image on every device; see the file header.
static __device__ __align__(256) double g_dot_scratch[2 * DOT_SLOTS];

// device address of g_dot_scratch per device ordinal (nullptr: not looked up yet), guarded by g_mu
std::mutex g_mu;
double* g_scratch_addr[MAX_DEVICES];

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// re, im += conj(a) b for the complex numbers of one 128-bit word, in fp64
__device__ __forceinline__ void acc_word(double& re, double& im, const float4& a, const float4& b) {
    const double ar0 = a.x, ai0 = a.y, ar1 = a.z, ai1 = a.w, br0 = b.x, bi0 = b.y, br1 = b.z, bi1 = b.w;
    re = fma(ar0, br0, re); re = fma(ai0, bi0, re); im = fma(ar0, bi0, im); im = fma(-ai0, br0, im);
    re = fma(ar1, br1, re); re = fma(ai1, bi1, re); im = fma(ar1, bi1, im); im = fma(-ai1, br1, im);
}
__device__ __forceinline__ void acc_word(double& re, double& im, const double2& a, const double2& b) {
    re = fma(a.x, b.x, re); re = fma(a.y, b.y, re); im = fma(a.x, b.y, im); im = fma(-a.y, b.x, im);
}

// slot[blockIdx.x] = sum over the CTA's DOT_RANGE sites of conj(x) y.  `slots` is the device address of g_dot_scratch.
template <typename T>
__global__ void __launch_bounds__(DOT_THREADS) dot_static_kernel(double* __restrict__ slots, const typename Prec<T>::Vec* __restrict__ x,
                                                                 const typename Prec<T>::Vec* __restrict__ y, long long V) {
    using Vec = typename Prec<T>::Vec;
    constexpr int NV = Prec<T>::NV;
    __shared__ double wred[DOT_WARPS][2];
    const long long base = (long long)blockIdx.x * DOT_RANGE;
    double re = 0.0, im = 0.0;
#pragma unroll
    for (int j = 0; j < DOT_SITES_PER_THREAD; j++) {
        const long long s = base + j * DOT_THREADS + threadIdx.x;
        if (s < V) {
            Vec a[NV], b[NV];
#pragma unroll
            for (int p = 0; p < NV; p++) { a[p] = x[p * V + s]; b[p] = y[p * V + s]; }   // all loads of the site in flight together
#pragma unroll
            for (int p = 0; p < NV; p++) acc_word(re, im, a[p], b[p]);
        }
    }
    re = warp_sum(re);
    im = warp_sum(im);
    if ((threadIdx.x & 31) == 0) { wred[threadIdx.x >> 5][0] = re; wred[threadIdx.x >> 5][1] = im; }
    __syncthreads();
    if (threadIdx.x < 2) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < DOT_WARPS; w++) t += wred[w][threadIdx.x];
        slots[2 * (long long)blockIdx.x + threadIdx.x] = t;
    }
}

// out[0..1] = sum_{b < nblocks} slot b, one CTA, fixed order
__global__ void __launch_bounds__(FINAL_THREADS) dot_static_final_kernel(double* __restrict__ out, const double* __restrict__ slots, int nblocks) {
    __shared__ double wred[FINAL_THREADS / 32][2];
    double re = 0.0, im = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += FINAL_THREADS) { re += slots[2 * b]; im += slots[2 * b + 1]; }
    re = warp_sum(re);
    im = warp_sum(im);
    if ((threadIdx.x & 31) == 0) { wred[threadIdx.x >> 5][0] = re; wred[threadIdx.x >> 5][1] = im; }
    __syncthreads();
    if (threadIdx.x < 2) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < FINAL_THREADS / 32; w++) t += wred[w][threadIdx.x];
        out[threadIdx.x] = t;
    }
}

int fail(char* errbuf, size_t errbuf_len, int code, const char* fmt, ...) {
    if (errbuf && errbuf_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// Device address of g_dot_scratch on `device`, which must be the current device.  Looked up once per device.
cudaError_t scratch_address(int device, double** addr) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[device]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_dot_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[device] = p;
    }
    *addr = g_scratch_addr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" int nd_dot_static(const void* x, const void* y, long long V, int prec, int device, void* stream, double* d_out2,
                             char* errbuf, size_t errbuf_len) {
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    if (!x || !y || !d_out2) return fail(errbuf, errbuf_len, ND_ERR_BAD_ARG, "nd_dot_static: null pointer (x, y and d_out2 are required)");
    if (prec != 32 && prec != 64) return fail(errbuf, errbuf_len, ND_ERR_BAD_ARG, "nd_dot_static: prec = %d, must be 32 or 64", prec);
    if (V < 1 || V > ND_DOT_STATIC_MAX_SITES)
        return fail(errbuf, errbuf_len, ND_ERR_BAD_ARG,
                    "nd_dot_static: V = %lld sites is outside [1, %lld]: the static scratch array holds one partial sum per %d sites; "
                    "larger fields need a context (nd_create + nd_dot_dev)",
                    V, (long long)ND_DOT_STATIC_MAX_SITES, DOT_RANGE);
    if (device < 0 || device >= MAX_DEVICES) return fail(errbuf, errbuf_len, ND_ERR_BAD_ARG, "nd_dot_static: device = %d, must be in [0, %d)", device, MAX_DEVICES);

    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
    double* slots = nullptr;
    if (e == cudaSuccess) e = scratch_address(device, &slots);
    if (e == cudaSuccess) {
        const int nblocks = (int)((V + DOT_RANGE - 1) / DOT_RANGE);
        const cudaStream_t st = (cudaStream_t)stream;
        if (prec == 32) dot_static_kernel<float><<<nblocks, DOT_THREADS, 0, st>>>(slots, (const float4*)x, (const float4*)y, V);
        else dot_static_kernel<double><<<nblocks, DOT_THREADS, 0, st>>>(slots, (const double2*)x, (const double2*)y, V);
        e = cudaGetLastError();
        if (e == cudaSuccess) {
            dot_static_final_kernel<<<1, FINAL_THREADS, 0, st>>>(d_out2, slots, nblocks);
            e = cudaGetLastError();
        }
    }
    if (prev >= 0 && prev != device) cudaSetDevice(prev);   // leave the caller's current device as it was
    if (e != cudaSuccess) return fail(errbuf, errbuf_len, ND_ERR_CUDA, "nd_dot_static: CUDA error %d (%s)", (int)e, cudaGetErrorString(e));
    return ND_OK;
}
