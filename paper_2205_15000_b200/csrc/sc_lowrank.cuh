// sc_lowrank.cuh — the paper's own vector-potential solve (App. D, D7-D9 :1023-1038): the Green's-function
// table G_{m,n} (D3-D6) is eigendecomposed, G = sum_k lambda_k V^(k) V^(k)T (D7), only the N* eigenpairs of largest
// |lambda| that satisfy sqrt(1 - sum_{n<N*} lambda_n^2 / sum_n lambda_n^2) < eps (D9) are kept, and the 2-D cross-correlation
// becomes N* pairs of separable 1-D cross-correlations (D8):
//     A_ind = -(1/kappa^2) sum_k lambda_k  Ty_k . J . Tx_k,    (T_k)_{a,b} = V^(k)_{|a-b|}   (symmetric Toeplitz),
// with J = (j - <j>_mask) on the mask.  The paper does the eigendecomposition on the CPU (Armadillo) and the
// correlations on the GPU; here both run on the device — cuSOLVER syevd once per geometry, two cuBLAS DGEMMs per kept
// eigenpair and current component (library routines, off the roofline-judged path).  This is an APPROXIMATION chosen
// with sc_set_vector_potential_error(eps > 0); eps = 0 (default) is the exact FFT correlation of sc_field_kernels.cuh,
// which is also faster (0.5 ms against ~1 ms per kept eigenpair at 1600 x 1600).
#pragma once
#include <cublas_v2.h>
#include <cuda_runtime.h>
#include <cusolverDn.h>

#include <algorithm>
#include <cmath>
#include <numeric>
#include <string>
#include <vector>

namespace scf {

// G_closed(m, n, h) (D3-D6) is defined in sc_field_kernels.cuh, which includes this header after it.

struct LowRank {
    int N = 0, nx = 0, ny = 0, nstar = 0; double eps = 0.0;
    std::vector<double> lam;            // kept eigenvalues, |lambda| descending
    double* V = nullptr;                // device, [nstar][N]: kept eigenvectors
    double *Tx = nullptr, *Ty = nullptr, *J = nullptr, *W = nullptr;
    cublasHandle_t blas = nullptr;
    bool ready = false;
};

inline void release(LowRank& L) {
    void* ptrs[] = {L.V, L.Tx, L.Ty, L.J, L.W};
    for (void* p : ptrs) if (p) cudaFree(p);
    if (L.blas) cublasDestroy(L.blas);
    L = LowRank();
}

__global__ void toeplitz_kernel(int n, const double* v, double* T) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i < n) T[(size_t)j * n + i] = v[i > j ? i - j : j - i];
}
// J = (j - mean) on the mask, 0 elsewhere
__global__ void masked_current_kernel(size_t ng, const unsigned char* mask, const double* j, const double* mean, int comp, double* J) {
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < ng) J[q] = mask[q] ? j[q] - mean[comp] : 0.0;
}

#define SCL_CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { err = std::string(#call) + ": " + cudaGetErrorString(e_); return e_ == cudaErrorMemoryAllocation ? 2 : 1; } } while (0)
#define SCL_LIB(call) do { int r_ = (int)(call); if (r_ != 0) { err = std::string(#call) + ": library error " + std::to_string(r_); return 1; } } while (0)

// eigendecomposition of G (once per geometry and tolerance) and the D9 truncation
inline int ensure_lowrank(LowRank& L, int nx, int ny, double h, double eps, cudaStream_t s, std::string& err) {
    if (L.ready && L.nx == nx && L.ny == ny && L.eps == eps) return 0;
    release(L);
    const int N = std::max(nx, ny);
    L.N = N; L.nx = nx; L.ny = ny; L.eps = eps;
    std::vector<double> G((size_t)N * N);
    for (int n = 0; n < N; ++n) for (int m = n; m < N; ++m) G[(size_t)n * N + m] = G[(size_t)m * N + n] = G_closed(m, n, h);   // G_{m,n} = G_{n,m}
    double *dG = nullptr, *dW = nullptr, *work = nullptr; int* info = nullptr; int lwork = 0;
    cusolverDnHandle_t sol = nullptr;
    // temporaries and the solver handle are released on every return path (the error macros below return early)
    struct Temps { double*& a; double*& b; double*& c; int*& i; cusolverDnHandle_t& h;
                   ~Temps() { cudaFree(a); cudaFree(b); cudaFree(c); cudaFree(i); if (h) cusolverDnDestroy(h); } } temps{dG, dW, work, info, sol};
    SCL_CU(cudaMalloc((void**)&dG, G.size() * sizeof(double))); SCL_CU(cudaMalloc((void**)&dW, N * sizeof(double))); SCL_CU(cudaMalloc((void**)&info, sizeof(int)));
    SCL_CU(cudaMemcpyAsync(dG, G.data(), G.size() * sizeof(double), cudaMemcpyHostToDevice, s));
    SCL_LIB(cusolverDnCreate(&sol)); SCL_LIB(cusolverDnSetStream(sol, s));
    SCL_LIB(cusolverDnDsyevd_bufferSize(sol, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, N, dG, N, dW, &lwork));
    SCL_CU(cudaMalloc((void**)&work, (size_t)lwork * sizeof(double)));
    SCL_LIB(cusolverDnDsyevd(sol, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, N, dG, N, dW, work, lwork, info));
    std::vector<double> lam(N); int hinfo = 0;
    SCL_CU(cudaMemcpyAsync(lam.data(), dW, N * sizeof(double), cudaMemcpyDeviceToHost, s));
    SCL_CU(cudaMemcpyAsync(&hinfo, info, sizeof(int), cudaMemcpyDeviceToHost, s));
    SCL_CU(cudaStreamSynchronize(s));
    if (hinfo != 0) { err = "cusolverDnDsyevd did not converge"; return 1; }
    // D9 (:1036): eigenvalues sorted by |lambda| descending; N* = smallest count with sqrt(1 - kept/total) < eps
    std::vector<int> ord(N); std::iota(ord.begin(), ord.end(), 0);
    std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return std::fabs(lam[a]) > std::fabs(lam[b]); });
    double tot = 0.0; for (double v : lam) tot += v * v;
    double kept = 0.0; int nstar = N;
    for (int k = 0; k < N; ++k) {
        kept += lam[ord[k]] * lam[ord[k]];
        if (std::sqrt(std::max(0.0, 1.0 - kept / tot)) < eps) { nstar = k + 1; break; }
    }
    L.nstar = nstar; L.lam.resize(nstar);
    SCL_CU(cudaMalloc((void**)&L.V, (size_t)nstar * N * sizeof(double)));
    for (int k = 0; k < nstar; ++k) {       // syevd returns the eigenvectors as the columns of dG (column-major): column c = dG + c*N
        L.lam[k] = lam[ord[k]];
        SCL_CU(cudaMemcpyAsync(L.V + (size_t)k * N, dG + (size_t)ord[k] * N, N * sizeof(double), cudaMemcpyDeviceToDevice, s));
    }
    SCL_CU(cudaMalloc((void**)&L.Tx, (size_t)nx * nx * sizeof(double))); SCL_CU(cudaMalloc((void**)&L.Ty, (size_t)ny * ny * sizeof(double)));
    SCL_CU(cudaMalloc((void**)&L.J, (size_t)nx * ny * sizeof(double))); SCL_CU(cudaMalloc((void**)&L.W, (size_t)nx * ny * sizeof(double)));
    SCL_LIB(cublasCreate(&L.blas)); SCL_LIB(cublasSetStream(L.blas, s));
    SCL_LIB(cublasSetMathMode(L.blas, CUBLAS_PEDANTIC_MATH));      // plain fp64 DGEMM, no reduced-precision paths
    SCL_CU(cudaStreamSynchronize(s));
    L.ready = true;
    return 0;
}

// one current component: out[ny][nx] = scale * sum_k lambda_k Ty_k . J . Tx_k  (row-major fields; as column-major
// matrices of size nx x ny: out^T = sum_k lambda_k Tx_k . J^T . Ty_k)
inline int lowrank_apply(LowRank& L, double scale, double* out, cudaStream_t s, std::string& err) {
    const int nx = L.nx, ny = L.ny, N = L.N;
    const double one = 1.0, zero = 0.0;
    SCL_CU(cudaMemsetAsync(out, 0, (size_t)nx * ny * sizeof(double), s));
    for (int k = 0; k < L.nstar; ++k) {
        ++sck::g_launches, toeplitz_kernel<<<dim3((nx + 127) / 128, nx), 128, 0, s>>>(nx, L.V + (size_t)k * N, L.Tx);
        ++sck::g_launches, toeplitz_kernel<<<dim3((ny + 127) / 128, ny), 128, 0, s>>>(ny, L.V + (size_t)k * N, L.Ty);
        const double a = scale * L.lam[k];
        SCL_LIB(cublasDgemm(L.blas, CUBLAS_OP_N, CUBLAS_OP_N, nx, ny, nx, &one, L.Tx, nx, L.J, nx, &zero, L.W, nx));
        SCL_LIB(cublasDgemm(L.blas, CUBLAS_OP_N, CUBLAS_OP_N, nx, ny, ny, &a, L.W, nx, L.Ty, ny, &one, out, nx));
    }
    SCL_CU(cudaGetLastError());
    return 0;
}

}  // namespace scf
