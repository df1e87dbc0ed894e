// approx.cu -- SURVEY.md §8(f) NEXT-4: factorisation-free APPROXIMATE projection onto the PSD cone (PAPER.md:181-183:
// "the corresponding spectral map can be approximated by a composite matrix polynomial constructed solely from
// matrix-matrix products").  The paper points to ref. [81] for the optimised coefficients; they are not in this
// container, so the composite polynomial built here is the K-fold composition of the Newton-Schulz cubic
// g(t) = (3 t - t^3) / 2 (DESIGN.md §4 reading):
//     S_0 = X / ||X||_F,    S_{k+1} = (3 S_k - S_k^3) / 2,    P_K = (X + X S_K) / 2,
// i.e. the filter lambda -> lambda (1 + g^K(lambda / s)) / 2 on the spectrum of X.  2 K + 1 complex n^3 GEMMs on the
// FP64 tensor pipe (DMMA, gemm.cuh), nothing else: no reduction, no eigensolver.  In FP64 this is slower than the exact
// path (K ~ 30 for eigenvalues down to 1e-5 ||X||); the paper proposes it for low-precision tensor cores.  Every S_k is a
// polynomial in X, hence Hermitian; the products are formed in full (both triangles).
#include "kernels.h"
#include "gemm.cuh"
#include "approx.h"

namespace hpsd {

constexpr int AP_MI = 4, AP_NI = 4, AP_WM = 2, AP_WN = 2;       // 64 x 64 CTA tile, 4 warps
constexpr int AP_THREADS = AP_WM * AP_WN * 32;
constexpr size_t kSmemAp = gemm_smem_bytes<cplx, cplx, MNMAJ, KMAJ, AP_MI, AP_NI, AP_WM, AP_WN>();

// ||svec||_2 = ||X||_F (the encoding preserves the inner product): one CTA, fixed summation order
__global__ void __launch_bounds__(1024) approx_norm_kernel(size_t len, const double *__restrict__ sv, double *__restrict__ out) {
    __shared__ double red[32];
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    size_t i = threadIdx.x;
    for (; i + 3 * 1024 < len; i += 4 * 1024) {
        const double x0 = sv[i], x1 = sv[i + 1024], x2 = sv[i + 2048], x3 = sv[i + 3072];
        a0 = fma(x0, x0, a0); a1 = fma(x1, x1, a1); a2 = fma(x2, x2, a2); a3 = fma(x3, x3, a3);
    }
    for (; i < len; i += 1024) { const double x = sv[i]; a0 = fma(x, x, a0); }
    double s = warp_sum((a0 + a1) + (a2 + a3));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = warp_sum(red[threadIdx.x]);
        if (threadIdx.x == 0) { const double nrm = sqrt(s); out[0] = nrm; out[1] = nrm > 0.0 ? 1.0 / nrm : 0.0; }
    }
}

// X (full, column-major) from the svec, and S_0 = X / s
__global__ void __launch_bounds__(256) approx_unpack_kernel(int n, const double *__restrict__ sv, const double *__restrict__ scal,
                                                            cplx *__restrict__ X, cplx *__restrict__ S, int ld) {
    const int j = blockIdx.y;
    const double *c = sv + svec_col_off(n, j);
    const double inv = scal[1];
    for (int i = j + blockIdx.x * 256 + threadIdx.x; i < n; i += gridDim.x * 256) {
        cplx v;
        if (i == j) v = mk(c[0], 0.0);
        else { const int k = i - j - 1; v = mk(c[1 + 2 * k] / kSqrt2, c[2 + 2 * k] / kSqrt2); }
        const cplx s = mk(v.x * inv, v.y * inv);
        X[(size_t)j * ld + i] = v; S[(size_t)j * ld + i] = s;
        if (i != j) { X[(size_t)i * ld + j] = conj_(v); S[(size_t)i * ld + j] = conj_(s); }
    }
}

struct ApStoreEpi {            // C = acc
    cplx *C; int ld;
    __device__ __forceinline__ void operator()(int i, int j, double re, double im) const { C[(size_t)j * ld + i] = mk(re, im); }
};
struct ApCubicEpi {            // C = 3/2 S - 1/2 acc        (acc = S T = S^3)
    cplx *C; const cplx *S; int ld;
    __device__ __forceinline__ void operator()(int i, int j, double re, double im) const {
        const cplx s = S[(size_t)j * ld + i];
        C[(size_t)j * ld + i] = mk(1.5 * s.x - 0.5 * re, 1.5 * s.y - 0.5 * im);
    }
};
struct ApPackEpi {             // svec out = vec_R((X + acc) / 2), lower triangle      (acc = X S_K)
    double *out; const cplx *X; int ld, n;
    __device__ __forceinline__ void operator()(int i, int j, double re, double im) const {
        const cplx x = X[(size_t)j * ld + i];
        const size_t c = svec_col_off(n, j);
        if (i == j) out[c] = 0.5 * (x.x + re);
        else { const size_t k = c + 1 + 2 * (size_t)(i - j - 1); out[k] = kSqrt2 * 0.5 * (x.x + re); out[k + 1] = kSqrt2 * 0.5 * (x.y + im); }
    }
};

// C = A B for full column-major n x n operands: A as (m, k) at A[m + k ld] (MNMAJ), B as (n, k) at B[k + n ld] (KMAJ)
template <class Epi, bool LOWER>
__global__ void __launch_bounds__(AP_THREADS) approx_gemm_kernel(int n, const cplx *__restrict__ A, const cplx *__restrict__ B, int ld, Epi epi) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (LOWER && blockIdx.y > blockIdx.x) return;
    GemmProblem<cplx, cplx> p;
    p.A = A; p.lda = ld; p.B = B; p.ldb = ld;
    p.A2 = nullptr; p.B2 = nullptr; p.lda2 = p.ldb2 = 0; p.M = n; p.N = n; p.K = n; p.K2 = 0;
    gemm_tile_body<cplx, cplx, MNMAJ, KMAJ, false, false, AP_MI, AP_NI, AP_WM, AP_WN, LOWER>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
}

static int g_ap_init_dev = -1;
static int approx_init() {
    int dev = 0;
    cudaGetDevice(&dev);
    if (g_ap_init_dev == dev) return 0;
    if (cudaFuncSetAttribute(approx_gemm_kernel<ApStoreEpi, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemAp) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(approx_gemm_kernel<ApCubicEpi, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemAp) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(approx_gemm_kernel<ApPackEpi, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemAp) != cudaSuccess) return HPSD_ECUDA_;
    g_ap_init_dev = dev;
    return 0;
}

size_t approx_ws_bytes(int n) {
    const size_t N = align_up((size_t)n, 8);
    return 4 * align_up(sizeof(cplx) * N * n, 256) + 256;
}

int launch_project_approx(int n, const double *in, double *out, int iterations, unsigned char *scratch, cudaStream_t st) {
    int rc = approx_init();
    if (rc) return rc;
    const int ld = (int)align_up((size_t)n, 8);
    const size_t mat = align_up(sizeof(cplx) * (size_t)ld * n, 256);
    double *scal = reinterpret_cast<double *>(scratch);
    cplx *X = reinterpret_cast<cplx *>(scratch + 256);
    cplx *S = reinterpret_cast<cplx *>(scratch + 256 + mat);
    cplx *S2 = reinterpret_cast<cplx *>(scratch + 256 + 2 * mat);
    cplx *T = reinterpret_cast<cplx *>(scratch + 256 + 3 * mat);
    approx_norm_kernel<<<1, 1024, 0, st>>>((size_t)n * n, in, scal);
    HPSD_LAUNCH_CHECK();
    approx_unpack_kernel<<<dim3((n + 1023) / 1024, n), 256, 0, st>>>(n, in, scal, X, S, ld);
    HPSD_LAUNCH_CHECK();
    const int nt = (n + 63) / 64;
    for (int k = 0; k < iterations; ++k) {
        approx_gemm_kernel<ApStoreEpi, false><<<dim3(nt, nt), AP_THREADS, kSmemAp, st>>>(n, S, S, ld, ApStoreEpi{T, ld});            // T = S^2
        HPSD_LAUNCH_CHECK();
        approx_gemm_kernel<ApCubicEpi, false><<<dim3(nt, nt), AP_THREADS, kSmemAp, st>>>(n, S, T, ld, ApCubicEpi{S2, S, ld});        // S' = 3/2 S - 1/2 S T
        HPSD_LAUNCH_CHECK();
        cplx *t = S; S = S2; S2 = t;
    }
    approx_gemm_kernel<ApPackEpi, true><<<dim3(nt, nt), AP_THREADS, kSmemAp, st>>>(n, X, S, ld, ApPackEpi{out, X, ld, n});           // (X + X S_K) / 2
    HPSD_LAUNCH_CHECK();
    return 0;
}

}  // namespace hpsd
