// affine.cu -- SURVEY.md §8(f) NEXT-3: the affine-projection step of the paper's SCS iteration on the device,
//     z_x = (a_x - A^T a_y) / 2,      z_y = a_y + A z_x
// with  A x = - sum_mu x_mu F_mu,  (A^T Z)_mu = - tr[F_mu Z]  (Eq. D3) over the orthonormal
// product basis  F_mu = sigma_alpha (x) sigma_beta (x) sigma_gamma (x) sigma_delta  of the process-matrix subspace:
// generalized Gell-Mann matrices (Eq. A10) on A_i, A_o, B_i, B_o (all of dimension d), restricted to
// the allowed multi-indices of Eq. (B14), all-identity index excluded.  Because A^T A = 1 (D4) no
// linear solve is needed.
//
// "Neither the basis matrices F_mu nor the operator A are formed explicitly": the paper contracts
// dense local basis tensors with einsum.  Here the contraction is four mode-wise transforms of the d^2 x d^2 x d^2 x d^2
// coefficient tensor that use the SPARSITY of the Gell-Mann matrices directly: an off-diagonal matrix position (a, a')
// receives two basis elements, a diagonal one at most d.  Every pass streams the tensor once (HBM-bound: 16 n^2 bytes
// in, 16 n^2 out; no GEMM), the svec <-> tensor index permutation is fused into the first / last pass.
#include <new>
#include <vector>
#include "../../include/hpsd.h"
#include "kernels.h"

namespace hpsd {

struct AffineDims {
    int d, q;           // local dimension, q = d^2 basis elements per subsystem
    int n;              // d^4
    long long t;        // q^4 = n^2 tensor elements
    int npairs;         // d (d - 1) / 2
};

__device__ __forceinline__ int pair_index(int d, int j, int k) { return j * (2 * d - j - 1) / 2 + (k - j - 1); }   // j < k
__device__ __forceinline__ double diag_scale(int l) { return rsqrt((double)((l + 1) * (l + 2))); }
constexpr double kRsqrt2 = 0.70710678118654752440;

__device__ __forceinline__ cplx ld_c(const cplx *p, long long i) { return p[i]; }
__device__ __forceinline__ cplx ld_c(const double *p, long long i) { return mk(p[i], 0.0); }

// out[l, p, r] = sum_alpha sigma_alpha[a, a'] in[l, alpha, r],  p = a d + a'   (mode j: L = q^j, R = q^(3-j))
template <typename TIN>
__global__ void __launch_bounds__(256) affine_mode_fwd_kernel(AffineDims D, long long R, const TIN *__restrict__ in, cplx *__restrict__ out) {
    const long long e = (long long)blockIdx.x * 256 + threadIdx.x;
    if (e >= D.t) return;
    const long long r = e % R, lp = e / R;
    const int p = (int)(lp % D.q);
    const long long l = lp / D.q;
    const int a = p / D.d, b = p % D.d;
    const long long base = l * D.q * R + r;                 // + alpha R
    cplx acc;
    if (a == b) {
        acc = rsqrt((double)D.d) * ld_c(in, base);
        if (a >= 1) { const cplx v = ld_c(in, base + (long long)a * R); const double c = -(double)a * diag_scale(a - 1); acc.x += c * v.x; acc.y += c * v.y; }
        for (int l2 = a; l2 <= D.d - 2; ++l2) { const cplx v = ld_c(in, base + (long long)(1 + l2) * R); const double c = diag_scale(l2); acc.x += c * v.x; acc.y += c * v.y; }
    } else {
        const int j = a < b ? a : b, k = a < b ? b : a;
        const int pi = pair_index(D.d, j, k);
        const cplx s = ld_c(in, base + (long long)(D.d + pi) * R);
        const cplx t = ld_c(in, base + (long long)(D.d + D.npairs + pi) * R);
        // sigma_sym[a, b] = 1/sqrt2;  sigma_asym[j, k] = -i/sqrt2, sigma_asym[k, j] = +i/sqrt2
        const cplx it = a < b ? mk(t.y, -t.x) : mk(-t.y, t.x);
        acc = mk(kRsqrt2 * (s.x + it.x), kRsqrt2 * (s.y + it.y));
    }
    out[e] = acc;
}

// out[l, alpha, r] = sum_p conj(sigma_alpha[a, a']) in[l, p, r]
__global__ void __launch_bounds__(256) affine_mode_adj_kernel(AffineDims D, long long R, const cplx *__restrict__ in, cplx *__restrict__ out) {
    const long long e = (long long)blockIdx.x * 256 + threadIdx.x;
    if (e >= D.t) return;
    const long long r = e % R, lp = e / R;
    const int al = (int)(lp % D.q);
    const long long l = lp / D.q;
    const long long base = l * D.q * R + r;                 // + p R
    const int d = D.d;
    cplx acc = mk(0.0, 0.0);
    if (al == 0) {
        for (int a = 0; a < d; ++a) acc = acc + in[base + (long long)(a * d + a) * R];
        const double c = rsqrt((double)d);
        acc = mk(c * acc.x, c * acc.y);
    } else if (al < d) {
        const int l2 = al - 1;
        for (int a = 0; a <= l2; ++a) acc = acc + in[base + (long long)(a * d + a) * R];
        const cplx v = in[base + (long long)((l2 + 1) * d + l2 + 1) * R];
        const double c = diag_scale(l2);
        acc = mk(c * (acc.x - (l2 + 1) * v.x), c * (acc.y - (l2 + 1) * v.y));
    } else {
        const bool asym = al >= d + D.npairs;
        int pi = al - d - (asym ? D.npairs : 0);
        int j = 0;
        while (pi >= d - 1 - j) { pi -= d - 1 - j; ++j; }    // pair_index inverse
        const int k = j + 1 + pi;
        const cplx u = in[base + (long long)(j * d + k) * R], v = in[base + (long long)(k * d + j) * R];
        if (!asym) acc = mk(kRsqrt2 * (u.x + v.x), kRsqrt2 * (u.y + v.y));
        else { const cplx w = mk(u.x - v.x, u.y - v.y); acc = mk(-kRsqrt2 * w.y, kRsqrt2 * w.x); }      // i (u - v) / sqrt2
    }
    out[e] = acc;
}

// tensor index of the matrix element (row, col): digits (a1..a4), (a1'..a4') -> p_i = a_i d + a_i'
__device__ __forceinline__ long long tensor_index(const AffineDims &D, int row, int col) {
    const int d = D.d;
    long long idx = 0, mul = 1;
    for (int s = 0; s < 4; ++s) {                            // from the last subsystem (B_o) to the first
        const int a = row % d, b = col % d;
        row /= d; col /= d;
        idx += (long long)(a * d + b) * mul;
        mul *= D.q;
    }
    return idx;
}

// T[p1..p4] = Z[(a1 a2 a3 a4), (a1' a2' a3' a4')] from the svec of the Hermitian matrix Z (Eq. D10 inverted)
__global__ void __launch_bounds__(256) affine_svec_to_tensor_kernel(AffineDims D, const double *__restrict__ sv, cplx *__restrict__ T) {
    const int j = blockIdx.y;                                // matrix column
    const double *c = sv + svec_col_off(D.n, j);
    for (int i = j + blockIdx.x * 256 + threadIdx.x; i < D.n; i += gridDim.x * 256) {
        cplx v;
        if (i == j) v = mk(c[0], 0.0);
        else { const int k = i - j - 1; v = mk(c[1 + 2 * k] / kSqrt2, c[2 + 2 * k] / kSqrt2); }
        T[tensor_index(D, i, j)] = v;
        if (i != j) T[tensor_index(D, j, i)] = conj_(v);
    }
}

// svec out = base_svec (or 0) + sign * vec_R(T as a matrix): lower triangle only (T is Hermitian as a matrix)
__global__ void __launch_bounds__(256) affine_tensor_to_svec_kernel(AffineDims D, const cplx *__restrict__ T, const double *base,
                                                                     double sign, double *out) {
    const int j = blockIdx.y;
    const size_t o = svec_col_off(D.n, j);
    for (int i = j + blockIdx.x * 256 + threadIdx.x; i < D.n; i += gridDim.x * 256) {
        const cplx v = T[tensor_index(D, i, j)];
        if (i == j) out[o] = (base ? base[o] : 0.0) + sign * v.x;
        else {
            const size_t k = o + 1 + 2 * (size_t)(i - j - 1);
            out[k] = (base ? base[k] : 0.0) + sign * kSqrt2 * v.x;
            out[k + 1] = (base ? base[k + 1] : 0.0) + sign * kSqrt2 * v.y;
        }
    }
}

__global__ void __launch_bounds__(256) affine_scatter_kernel(int m, const int *__restrict__ idx, const double *__restrict__ x, double *__restrict__ w) {
    const int k = blockIdx.x * 256 + threadIdx.x;
    if (k < m) w[idx[k]] = x[k];
}
// x_out[mu] = scale_a * a[mu] + scale_t * Re T[idx[mu]]
__global__ void __launch_bounds__(256) affine_gather_kernel(int m, const int *__restrict__ idx, const cplx *__restrict__ T,
                                                            const double *a, double scale_a, double scale_t, double *out) {
    const int k = blockIdx.x * 256 + threadIdx.x;
    if (k < m) out[k] = (a ? scale_a * a[k] : 0.0) + scale_t * T[idx[k]].x;
}

}  // namespace hpsd

using namespace hpsd;

struct hpsd_affine {
    AffineDims D;
    int m = 0, dev = -1;
    int *idx = nullptr;           // device: tensor index of every allowed multi-index, lexicographic in (alpha, beta, gamma, delta)
    double *w = nullptr;          // device: coefficient tensor (real, q^4)
    cplx *T0 = nullptr, *T1 = nullptr;
};

namespace {

int affine_forward(hpsd_affine *h, const double *x, const double *base, double *out_svec, cudaStream_t st) {
    // w <- scatter(x);  four forward modes (first reads the real tensor);  svec <- base - T
    const AffineDims &D = h->D;
    const unsigned nb = (unsigned)((D.t + 255) / 256);
    HPSD_CUDA_OK(cudaMemsetAsync(h->w, 0, sizeof(double) * (size_t)D.t, st));
    affine_scatter_kernel<<<(h->m + 255) / 256, 256, 0, st>>>(h->m, h->idx, x, h->w);
    HPSD_LAUNCH_CHECK();
    long long R = (long long)D.q * D.q * D.q;
    affine_mode_fwd_kernel<double><<<nb, 256, 0, st>>>(D, R, h->w, h->T0);
    HPSD_LAUNCH_CHECK();
    cplx *src = h->T0, *dst = h->T1;
    for (int mode = 1; mode < 4; ++mode) {
        R /= D.q;
        affine_mode_fwd_kernel<cplx><<<nb, 256, 0, st>>>(D, R, src, dst);
        HPSD_LAUNCH_CHECK();
        cplx *t = src; src = dst; dst = t;
    }
    affine_tensor_to_svec_kernel<<<dim3((D.n + 1023) / 1024, D.n), 256, 0, st>>>(D, src, base, -1.0, out_svec);
    HPSD_LAUNCH_CHECK();
    return 0;
}

// leaves the fully transformed tensor (alpha-space on all four modes) in *result
int affine_adjoint(hpsd_affine *h, const double *y_svec, cplx **result, cudaStream_t st) {
    const AffineDims &D = h->D;
    const unsigned nb = (unsigned)((D.t + 255) / 256);
    affine_svec_to_tensor_kernel<<<dim3((D.n + 1023) / 1024, D.n), 256, 0, st>>>(D, y_svec, h->T0);
    HPSD_LAUNCH_CHECK();
    cplx *src = h->T0, *dst = h->T1;
    long long R = (long long)D.q * D.q * D.q;
    for (int mode = 0; mode < 4; ++mode) {
        affine_mode_adj_kernel<<<nb, 256, 0, st>>>(D, R, src, dst);
        HPSD_LAUNCH_CHECK();
        cplx *t = src; src = dst; dst = t;
        R /= D.q;
    }
    *result = src;
    return 0;
}

}  // namespace

extern "C" {

int hpsd_affine_create(int d, hpsd_affine **out) {
    if (!out) return HPSD_EINVAL;
    *out = nullptr;
    if (d < 2 || d > 9) return HPSD_EINVAL;
    int dev;
    if (cudaGetDevice(&dev) != cudaSuccess) return HPSD_ECUDA;
    hpsd_affine *h = new (std::nothrow) hpsd_affine();
    if (!h) return HPSD_EALLOC;
    h->dev = dev;
    AffineDims &D = h->D;
    D.d = d; D.q = d * d; D.n = D.q * D.q; D.t = (long long)D.n * D.n; D.npairs = d * (d - 1) / 2;
    // allowed multi-indices of Eq. (B14): w_{alpha 0, gamma 0}, w_{i 0, gamma l}, w_{alpha j, k 0}; not (0,0,0,0)
    std::vector<int> idx;
    const int q = D.q;
    for (int al = 0; al < q; ++al)
        for (int be = 0; be < q; ++be)
            for (int ga = 0; ga < q; ++ga)
                for (int de = 0; de < q; ++de) {
                    if (!(al | be | ga | de)) continue;
                    const bool ok = (be == 0 && de == 0) || (al >= 1 && be == 0 && de >= 1) || (be >= 1 && ga >= 1 && de == 0);
                    if (ok) idx.push_back(((al * q + be) * q + ga) * q + de);
                }
    h->m = (int)idx.size();
    bool ok = cudaMalloc(&h->idx, sizeof(int) * idx.size()) == cudaSuccess &&
              cudaMalloc(&h->w, sizeof(double) * (size_t)D.t) == cudaSuccess &&
              cudaMalloc(&h->T0, sizeof(cplx) * (size_t)D.t) == cudaSuccess &&
              cudaMalloc(&h->T1, sizeof(cplx) * (size_t)D.t) == cudaSuccess &&
              cudaMemcpy(h->idx, idx.data(), sizeof(int) * idx.size(), cudaMemcpyHostToDevice) == cudaSuccess;
    if (!ok) { hpsd_affine_destroy(h); cudaGetLastError(); return HPSD_EALLOC; }
    *out = h;
    return HPSD_OK;
}

int hpsd_affine_destroy(hpsd_affine *h) {
    if (!h) return HPSD_OK;
    if (h->idx) cudaFree(h->idx);
    if (h->w) cudaFree(h->w);
    if (h->T0) cudaFree(h->T0);
    if (h->T1) cudaFree(h->T1);
    delete h;
    return HPSD_OK;
}

int hpsd_affine_dims(const hpsd_affine *h, int *n, int *m) {
    if (!h) return HPSD_EINVAL;
    if (n) *n = h->D.n;
    if (m) *m = h->m;
    return HPSD_OK;
}

int hpsd_affine_apply_a(hpsd_affine *h, const double *x, double *y_svec, void *stream) {
    if (!h || !x || !y_svec) return HPSD_EINVAL;
    g_launches = 0;
    return affine_forward(h, x, nullptr, y_svec, (cudaStream_t)stream);
}

int hpsd_affine_apply_at(hpsd_affine *h, const double *y_svec, double *x, void *stream) {
    if (!h || !x || !y_svec) return HPSD_EINVAL;
    g_launches = 0;
    cudaStream_t st = (cudaStream_t)stream;
    cplx *t;
    int rc = affine_adjoint(h, y_svec, &t, st);
    if (rc) return rc;
    affine_gather_kernel<<<(h->m + 255) / 256, 256, 0, st>>>(h->m, h->idx, t, nullptr, 0.0, -1.0, x);       // (A^T Z)_mu = - tr[F_mu Z]
    HPSD_LAUNCH_CHECK();
    return HPSD_OK;
}

int hpsd_affine_project(hpsd_affine *h, const double *a_x, const double *a_y, double *z_x, double *z_y, void *stream) {
    if (!h || !a_x || !a_y || !z_x || !z_y) return HPSD_EINVAL;
    g_launches = 0;
    cudaStream_t st = (cudaStream_t)stream;
    cplx *t;
    int rc = affine_adjoint(h, a_y, &t, st);
    if (rc) return rc;
    // z_x = (a_x - A^T a_y) / 2 = (a_x + tr[F_mu a_y]) / 2
    affine_gather_kernel<<<(h->m + 255) / 256, 256, 0, st>>>(h->m, h->idx, t, a_x, 0.5, 0.5, z_x);
    HPSD_LAUNCH_CHECK();
    // z_y = a_y + A z_x = a_y - sum_mu z_x,mu F_mu
    return affine_forward(h, z_x, a_y, z_y, st);
}

}  // extern "C"
