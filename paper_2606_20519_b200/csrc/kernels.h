// kernels.h -- internal launcher declarations (host side) of the hpsd library.
#pragma once
#include "common.cuh"

namespace hpsd {

// ---- pack.cu (S1 / S8) ------------------------------------
// svec -> column-major complex.  full=0: lower triangle incl. diagonal only.
// sub != nullptr: unpack svec - sub (the ADMM argument u~ - v of Eq. D33)
// nf != nullptr: non-finite entries are replaced by zero and *nf (device) is set to 1
int launch_svec_convert(size_t count, const void *src, void *dst, int to_f32, cudaStream_t st);
int launch_unpack(int n, const double *svec, const double *sub, cplx *A, int lda, int full, cudaStream_t st, int *nf = nullptr, int f32 = 0);
int launch_pack(int n, const cplx *A, int lda, double *svec, cudaStream_t st);
// n = 1 blocks: out = max(in, 0) for `count` scattered scalars
int launch_clamp_scalars(int count, const long long *offs_dev, const SvecIo &io, cudaStream_t st);

// ---- jacobi.cu (S9 / S10) --------------------------------------------------
// Batched one-CTA-per-matrix cyclic Jacobi projection for blocks of one size n
// (2 <= n <= kJacobiMaxN).  offs_dev[i] = svec offset (doubles) of matrix i;
// info_dev may be NULL; info_idx_dev[i] = index into info_dev.
constexpr int kJacobiMaxN = 84;
int launch_jacobi_project(int n, int count, const long long *offs_dev, const SvecIo &io,
                          int *info_dev, const int *info_idx_dev, cudaStream_t st);
int jacobi_init();  // set kernel attributes once per device

// ---- medium.cu (S10) ----------------------------------------------------------
// Batched one-CTA-per-matrix Householder + implicit-QL projection for blocks of one size n,
// jacobi_max_n < n <= kMediumMaxN (the matrix must fit in shared memory: 16 n (n|1) + O(n) bytes).
constexpr int kMediumMaxN = 116;
int launch_hhql_project(int n, int count, const long long *offs_dev, const SvecIo &io,
                        int *info_dev, const int *info_idx_dev, cudaStream_t st);
int medium_init();
// Batched divide-and-conquer variant (n <= kMedDcMaxN: reflectors and kept eigenvectors both fit in shared memory);
// scratch >= meddc_ws_bytes(n, count), 256-byte aligned.
constexpr int kMedDcMaxN = 83;
size_t meddc_ws_bytes(int n, int count);
int launch_meddc_project(int n, int count, const long long *offs_dev, const SvecIo &io, unsigned char *scratch,
                         int *info_dev, const int *info_idx_dev, cudaStream_t st);

// ---- peak.cu ---------------------------------------------------------------
int launch_fp64_probe(int kind, int iters, double *flops_host, cudaStream_t st);

}  // namespace hpsd
