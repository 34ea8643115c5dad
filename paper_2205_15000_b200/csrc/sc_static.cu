// sc_static.cu — sc_residual_norm_static: the one entry point of the library that allocates nothing.
//
// The residual of Eq. 27 ||x_new - x_old||_p / ||x_old||_p of a complex field is what the driver
// evaluates once per self-consistency iteration (sc_field_kernels.cuh: reduce_stage1 / reduce_stage2 with the
// per-block partial sums in the context's cudaMalloc'ed `red` buffer).  Callers that may not allocate — code under
// CUDA graph capture, tight serving loops — get the same two-stage, fixed-order reduction here with the partial sums
// in a file-scope device array instead.  Every GPU that loads the library holds the array (64.25 KiB) until exit.
//
// The array is shared by every call on a device and keeps the last call's contents: the block counter is cleared at
// the start of each call (a memset node on the caller's stream), the partial sums are overwritten before they are
// read.  Two calls that overlap on one GPU (different streams, or two host threads) race on it.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/sc_riccati.h"

namespace {

constexpr int ST_THREADS = 256;
constexpr int ST_ITEMS = 8;                          // elements per thread
constexpr int ST_TILE = ST_THREADS * ST_ITEMS;       // one block reduces one tile of 2048 elements
constexpr int ST_MAX_BLOCKS = 4096;                  // tiles the scratch has room for
constexpr int ST_COUNTER = 2 * ST_MAX_BLOCKS;        // offset (in doubles) of the block counter behind the partial sums
static_assert((long long)ST_MAX_BLOCKS * ST_TILE == SC_RESIDUAL_STATIC_MAX_ELEMENTS, "header and kernel disagree on the maximum size");

// [2 * b], [2 * b + 1]: partial norms of tile b (numerator, denominator); [ST_COUNTER]: blocks finished (unsigned)
static __device__ __align__(256) double g_static_scratch[2 * ST_MAX_BLOCKS + 32];

// P: 2 = sum of |element|^2 (root at the end), 1 = sum of |element|, -1 = maximum of |element|; one element is one complex number
template <int P> __device__ __forceinline__ double term(double a, double b) { return P == 2 ? a * a + b * b : sqrt(a * a + b * b); }
template <int P> __device__ __forceinline__ double join(double s, double v) { return P < 0 ? fmax(s, v) : s + v; }

template <int P>
__device__ __forceinline__ void block_join(double (&sh)[2][ST_THREADS], double& a, double& b) {
    sh[0][threadIdx.x] = a; sh[1][threadIdx.x] = b;
    __syncthreads();
    for (int o = ST_THREADS / 2; o; o >>= 1) {
        if (threadIdx.x < o) {
            sh[0][threadIdx.x] = join<P>(sh[0][threadIdx.x], sh[0][threadIdx.x + o]);
            sh[1][threadIdx.x] = join<P>(sh[1][threadIdx.x], sh[1][threadIdx.x + o]);
        }
        __syncthreads();
    }
    a = sh[0][0]; b = sh[1][0];
    __syncthreads();
}

// One launch: every block writes the partial norms of its tile, the block that finishes last joins them in tile order
// (so the result does not depend on which block that is) and writes out[0..2].
template <int P>
__global__ void __launch_bounds__(ST_THREADS) residual_static_kernel(const double2* __restrict__ x_new, const double2* __restrict__ x_old,
                                                                     size_t n, double* scratch, double* __restrict__ out) {
    __shared__ double sh[2][ST_THREADS];
    __shared__ bool last;
    double a = 0.0, b = 0.0;
    const size_t base = (size_t)blockIdx.x * ST_TILE;
#pragma unroll
    for (int q = 0; q < ST_ITEMS; ++q) {
        const size_t i = base + (size_t)q * ST_THREADS + threadIdx.x;
        if (i < n) {
            const double2 u = x_new[i], v = x_old[i];
            a = join<P>(a, term<P>(u.x - v.x, u.y - v.y));
            b = join<P>(b, term<P>(v.x, v.y));
        }
    }
    block_join<P>(sh, a, b);
    if (threadIdx.x == 0) {
        scratch[2 * blockIdx.x] = a; scratch[2 * blockIdx.x + 1] = b;
        __threadfence();
        const unsigned done = atomicAdd(reinterpret_cast<unsigned*>(scratch + ST_COUNTER), 1u);
        last = done + 1 == gridDim.x;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    a = 0.0; b = 0.0;
    for (unsigned t = threadIdx.x; t < gridDim.x; t += ST_THREADS) {
        a = join<P>(a, __ldcg(scratch + 2 * t)); b = join<P>(b, __ldcg(scratch + 2 * t + 1));
    }
    block_join<P>(sh, a, b);
    if (threadIdx.x == 0) {
        if (P == 2) { a = sqrt(a); b = sqrt(b); }
        out[0] = a; out[1] = b; out[2] = b > 0 ? a / b : a;
    }
}

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
double* g_scratch_addr[MAX_DEVICES] = {};     // device address of g_static_scratch on each device, set once per device

sc_status fail(char* err, int err_len, sc_status s, const char* what, const char* detail = "") {
    if (err && err_len > 0) std::snprintf(err, (size_t)err_len, "sc_residual_norm_static: %s%s", what, detail);
    return s;
}

}  // namespace

extern "C" sc_status sc_residual_norm_static(const void* x_new, const void* x_old, long long n, int norm_p, double* out,
                                             int device, void* cuda_stream, char* err, int err_len) {
    if (err && err_len > 0) err[0] = 0;
    if (!x_new || !x_old || !out) return fail(err, err_len, SC_ERR_ARG, "null argument");
    if (n < 1) return fail(err, err_len, SC_ERR_ARG, "n < 1");
    if (n > SC_RESIDUAL_STATIC_MAX_ELEMENTS) {
        char d[96];
        std::snprintf(d, sizeof d, "%lld elements exceed the static scratch's maximum of %lld", n, (long long)SC_RESIDUAL_STATIC_MAX_ELEMENTS);
        return fail(err, err_len, SC_ERR_ARG, d);
    }
    if (norm_p == 0) norm_p = 2;
    if (norm_p != 2 && norm_p != 1 && norm_p != -1) return fail(err, err_len, SC_ERR_ARG, "norm_p must be 2 (or 0), 1, or -1 (maximum norm)");
    cudaError_t e;
    if (device < 0) { if ((e = cudaGetDevice(&device)) != cudaSuccess) return fail(err, err_len, SC_ERR_CUDA, "cudaGetDevice: ", cudaGetErrorString(e)); }
    else if ((e = cudaSetDevice(device)) != cudaSuccess) return fail(err, err_len, SC_ERR_CUDA, "cudaSetDevice: ", cudaGetErrorString(e));
    if (device >= MAX_DEVICES) return fail(err, err_len, SC_ERR_ARG, "device ordinal out of range");
    double* scratch;
    {   // set-up, once per device, with that device current: in host code the array's name is not a device address
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        if (!g_scratch_addr[device]) {
            double* p = nullptr;
            if ((e = cudaGetSymbolAddress((void**)&p, g_static_scratch)) != cudaSuccess || !p)
                return fail(err, err_len, SC_ERR_CUDA, "cudaGetSymbolAddress: ", cudaGetErrorString(e));
            g_scratch_addr[device] = p;
        }
        scratch = g_scratch_addr[device];
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if ((e = cudaMemsetAsync(scratch + ST_COUNTER, 0, sizeof(double), s)) != cudaSuccess)
        return fail(err, err_len, SC_ERR_CUDA, "cudaMemsetAsync: ", cudaGetErrorString(e));
    const unsigned blocks = (unsigned)((n + ST_TILE - 1) / ST_TILE);
    const double2 *a = (const double2*)x_new, *b = (const double2*)x_old;
    if (norm_p == 2) residual_static_kernel<2><<<blocks, ST_THREADS, 0, s>>>(a, b, (size_t)n, scratch, out);
    else if (norm_p == 1) residual_static_kernel<1><<<blocks, ST_THREADS, 0, s>>>(a, b, (size_t)n, scratch, out);
    else residual_static_kernel<-1><<<blocks, ST_THREADS, 0, s>>>(a, b, (size_t)n, scratch, out);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail(err, err_len, SC_ERR_CUDA, "kernel launch: ", cudaGetErrorString(e));
    return SC_OK;
}
