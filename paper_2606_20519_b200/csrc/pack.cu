// pack.cu -- S1 (mat_R) and S8 (vec_R) of SURVEY.md §8(a); Eq. (D10).
// HBM-bound streaming kernels: every svec double is read/written exactly once,
// consecutive threads walk consecutive rows of one column (coalesced on both sides).
#include "kernels.h"

namespace hpsd {

// One CTA handles a chunk of one column j: rows i = j .. n-1.
// svec column j: [X_jj, s Re X_{j+1,j}, s Im X_{j+1,j}, ...]
template <int FULL>
__global__ void __launch_bounds__(256) unpack_kernel(int n, const double *__restrict__ sv, const double *__restrict__ sub, cplx *__restrict__ A, int lda,
                                                     int *__restrict__ nf, int f32) {
    const int j = blockIdx.y;
    const size_t o = svec_col_off(n, j);
    for (int i = j + blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        cplx v;
        if (i == j) {
            v = mk(sub ? sv_ld(sv, o, f32) - sv_ld(sub, o, f32) : sv_ld(sv, o, f32), 0.0);
        } else {
            const size_t k = o + 1 + 2 * (size_t)(i - j - 1);
            double re = sv_ld(sv, k, f32), im = sv_ld(sv, k + 1, f32);
            if (sub) { re -= sv_ld(sub, k, f32); im -= sv_ld(sub, k + 1, f32); }     // u~ - v of Eq. (D33)
            // division, not multiplication by 1/sqrt2: bit-identical to vec_R^-1 as defined
            v = mk(re / kSqrt2, im / kSqrt2);
        }
        if (nonfinite(v.x) || nonfinite(v.y)) {       // the path computes on a sanitised copy; the flag turns the output into NaN
            v = mk(0.0, 0.0);
            if (nf) *nf = 1;
        }
        A[(size_t)j * lda + i] = v;
        if (FULL && i != j) A[(size_t)i * lda + j] = conj_(v);
    }
}

__global__ void __launch_bounds__(256) pack_kernel(int n, const cplx *__restrict__ A, int lda, double *__restrict__ sv) {
    const int j = blockIdx.y;
    double *c = sv + svec_col_off(n, j);
    for (int i = j + blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const cplx v = A[(size_t)j * lda + i];
        if (i == j) {
            c[0] = v.x;
        } else {
            const int k = i - j - 1;
            c[1 + 2 * k] = kSqrt2 * v.x;
            c[2 + 2 * k] = kSqrt2 * v.y;
        }
    }
}

__global__ void clamp_scalars_kernel(int count, const long long *__restrict__ offs, SvecIo io) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) {
        const double v = io_load(io, offs[i]);
        io_store(io, offs[i], v > 0.0 ? v : (v != v ? v : 0.0));   // NaN propagates
    }
}

__global__ void __launch_bounds__(256) svec_convert_kernel(size_t count, const void *__restrict__ src, void *__restrict__ dst, int to_f32) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (size_t)gridDim.x * blockDim.x) {
        if (to_f32) reinterpret_cast<float *>(dst)[i] = (float)reinterpret_cast<const double *>(src)[i];
        else reinterpret_cast<double *>(dst)[i] = (double)reinterpret_cast<const float *>(src)[i];
    }
}

int launch_svec_convert(size_t count, const void *src, void *dst, int to_f32, cudaStream_t st) {
    if (count == 0) return 0;
    size_t blocks = (count + 1023) / 1024;           // four entries per thread
    if (blocks > 148 * 32) blocks = 148 * 32;
    svec_convert_kernel<<<(unsigned)blocks, 256, 0, st>>>(count, src, dst, to_f32);
    HPSD_LAUNCH_CHECK();
    return 0;
}

static dim3 col_grid(int n) {
    int gx = (n + 1023) / 1024;  // up to 4 rows per thread before the grid-stride loop wraps
    if (gx < 1) gx = 1;
    return dim3(gx, n, 1);
}

int launch_unpack(int n, const double *svec, const double *sub, cplx *A, int lda, int full, cudaStream_t st, int *nf, int f32) {
    if (n <= 0) return 0;
    if (n > 65535) return -1;
    if (full) unpack_kernel<1><<<col_grid(n), 256, 0, st>>>(n, svec, sub, A, lda, nf, f32);
    else unpack_kernel<0><<<col_grid(n), 256, 0, st>>>(n, svec, sub, A, lda, nf, f32);
    HPSD_LAUNCH_CHECK();
    return 0;
}

int launch_pack(int n, const cplx *A, int lda, double *svec, cudaStream_t st) {
    if (n <= 0) return 0;
    if (n > 65535) return -1;
    pack_kernel<<<col_grid(n), 256, 0, st>>>(n, A, lda, svec);
    HPSD_LAUNCH_CHECK();
    return 0;
}

int launch_clamp_scalars(int count, const long long *offs_dev, const SvecIo &io, cudaStream_t st) {
    if (count <= 0) return 0;
    clamp_scalars_kernel<<<(count + 127) / 128, 128, 0, st>>>(count, offs_dev, io);
    HPSD_LAUNCH_CHECK();
    return 0;
}

}  // namespace hpsd
