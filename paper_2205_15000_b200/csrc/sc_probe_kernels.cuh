// sc_probe_kernels.cuh — measurement kernels that are not part of the sweep (kept apart from sc_kernels.cuh so that the
// march kernel's sources, whose hash stamps the ncu captures in profiles/, do not change when a probe is added).
#pragma once
#include <cuda_runtime.h>

namespace sck {

// What other instructions cost next to half-rate DFMA: the 8-chain DFMA loop with NI integer (LOP3) and NL shared-memory
// loads (each followed by one DADD) per 8 DFMA.  Reported as DFMA per second (DESIGN.md §6 "what bounds the march").
template <int NI, int NL>
__global__ void __launch_bounds__(256) fp64_mix_kernel(int iters, double* sink) {
    __shared__ double sh[1024];
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double b = 0.999999, c = 1e-7;
    int x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3;
    for (int q = threadIdx.x; q < 1024; q += blockDim.x) sh[q] = q * 1e-12;
    __syncthreads();
    const unsigned base = (unsigned)__cvta_generic_to_shared(sh);
    double l = 0;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
#pragma unroll
            for (int q = 0; q < NI; ++q) {
                if (q % 4 == 0) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x0) : "r"(x1), "r"(i));
                if (q % 4 == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x1) : "r"(x2), "r"(i));
                if (q % 4 == 2) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x2) : "r"(x3), "r"(i));
                if (q % 4 == 3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x3) : "r"(x0), "r"(i));
            }
#pragma unroll
            for (int q = 0; q < NL; ++q) {
                double v;
                asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(base + ((threadIdx.x + 32 * q + 8 * u) & 1023) * 8));
                l += v;
            }
        }
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7 + l;
    if (s == 123.456 || (x0 ^ x1 ^ x2 ^ x3) == 0x12345) sink[0] = s;
}

// DFMA whose three source operands are all different registers that change from instruction to instruction (the march's
// DFMAs look like this; the peak loop above re-uses two constant operands): 8 chains a_i <- a_i * b_j + c_k with rotating j, k.
__global__ void __launch_bounds__(256) fp64_operand_kernel(int iters, double* sink) {
    double a[8], b[8], c[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = threadIdx.x * 1e-9 + i; b[i] = 0.999999 - 1e-9 * i; c[i] = 1e-7 * (i + 1); }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = fma(a[i], b[(i + u) & 7], c[(i + 3 * u + 1) & 7]);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    if (s == 123.456) sink[0] = s;
}

}  // namespace sck
