// backherk.cu -- S5..S8 of SURVEY.md §8(a) for large blocks.
//   S6 (first, because everything after is linear): W_T = Z_T[:, lambda>0] diag(sqrt(lambda_+))
//      ("setting all negative eigenvalues to zero"); eigenvalues are ascending so the
//      positive eigenpairs are the trailing columns: no compaction.
//   S5: W = Q W_T with Q = H_0 ... H_{n-2} applied as compact-WY blocks of 64 reflectors,
//      Z <- Z - (V_b T_b)(V_b^H Z), last block first.  All products are complex DMMA GEMMs.
//   S7+S8: lower triangle of P = W W^H ("matrix reconstruction") with the vec_R
//      scaling of Eq. (D10) applied in the epilogue, written straight into the output svec.
// The number of positive eigenvalues lives in device memory (cnt[1]); grids are worst-case.
#include "kernels.h"
#include "gemm.cuh"
#include "large.h"
#include "twostage.h"
#include "prof.h"

namespace hpsd {

constexpr int BG_MI = 4, BG_NI = 4, BG_WM = 2, BG_WN = 2;   // 64 x 64 CTA tile, 4 warps
constexpr int BG_THREADS = BG_WM * BG_WN * 32;

__global__ void count_pos_kernel(int n, const double *__restrict__ lam, int *cnt) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        int lo = 0, hi = n;   // first index with lam > 0
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (lam[mid] > 0.0) hi = mid; else lo = mid + 1; }
        cnt[0] = lo; cnt[1] = n - lo;
    }
}

// S6: Zc[:, j] = sqrt(lam[p0+j]) * Zt[:, p0+j]
__global__ void __launch_bounds__(256) scale_convert_kernel(int n, const double *__restrict__ lam, const double *__restrict__ Zt, int ldzt,
                                                            cplx *__restrict__ Zc, int ldz, const int *__restrict__ cnt) {
    const int p0 = cnt[0], kpos = cnt[1];
    const int j = blockIdx.y;
    if (j >= kpos) return;
    const double s = sqrt(lam[p0 + j]);
    for (int r = blockIdx.x * 256 + threadIdx.x; r < n; r += gridDim.x * 256) Zc[(size_t)j * ldz + r] = mk(s * Zt[(size_t)(p0 + j) * ldzt + r], 0.0);
}

struct StoreEpi {      // C[i + j*ld] = acc
    cplx *C; int ld;
    __device__ __forceinline__ void operator()(int i, int j, double re, double im) const { C[(size_t)j * ld + i] = mk(re, im); }
};
struct SubEpi {        // C[i + j*ld] -= acc
    cplx *C; int ld;
    static constexpr bool kRmw = true;
    __device__ __forceinline__ cplx load(int i, int j) const { return C[(size_t)j * ld + i]; }
    __device__ __forceinline__ void store(int i, int j, cplx v, double re, double im) const {
        v.x -= re; v.y -= im; C[(size_t)j * ld + i] = v;
    }
};

// Gram matrices G_b = V_b^H V_b for every block (blockIdx.z = b), K split over kSplitK CTAs (blockIdx.x);
// the partial Grams go to Xp (free at this point), bt_tfactor_kernel sums them.
__global__ void __launch_bounds__(BG_THREADS) bt_gram_kernel(BackWs w) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int b = blockIdx.z, cb = b * kNBT;
    const int nbw = min(kNBT, w.n - cb), m = w.n - cb - w.voff;
    if (m <= 0) return;
    const int chunk = (((m + kSplitK - 1) / kSplitK) + 15) & ~15;
    const int k0 = blockIdx.x * chunk;
    const int klen = min(chunk, m - k0);
    GemmProblem<cplx, cplx> p;
    p.A = w.A + (size_t)cb * w.lda + cb + w.voff + k0; p.lda = w.lda; p.B = p.A; p.ldb = w.lda;
    p.A2 = nullptr; p.B2 = nullptr; p.lda2 = p.ldb2 = 0; p.M = nbw; p.N = nbw; p.K = klen > 0 ? klen : 0; p.K2 = 0;
    StoreEpi epi{w.Xp + ((size_t)b * kSplitK + blockIdx.x) * kNBT * kNBT, kNBT};
    gemm_tile_body<cplx, cplx, KMAJ, KMAJ, true, false, BG_MI, BG_NI, BG_WM, BG_WN, false>(p, 0, 0, smem_raw, epi);
}

// T_b from the Gram matrix by the forward recurrence  T(0:j, j) = -tau_j T(0:j,0:j) G(0:j, j), T(j,j) = tau_j,
// in shared memory (64 KB): thread t owns row t of T and only re-reads its own earlier writes.
__global__ void __launch_bounds__(kNBT) bt_tfactor_kernel(BackWs w) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *T = reinterpret_cast<cplx *>(smem_raw);       // kNBT x kNBT, column-major; holds G first
    const int b = blockIdx.x, cb = b * kNBT, t = threadIdx.x;
    const int nbw = min(kNBT, w.n - cb);
    const cplx *part = w.Xp + (size_t)b * kSplitK * kNBT * kNBT;
    for (int e = t; e < kNBT * kNBT; e += kNBT) {
        const int r = e % kNBT, c = e / kNBT;
        cplx s = mk(0.0, 0.0);
        if (r < nbw && c < nbw) {
#pragma unroll
            for (int k = 0; k < kSplitK; ++k) s = s + part[(size_t)k * kNBT * kNBT + e];
        }
        T[e] = s;
    }
    __syncthreads();
    for (int j = 0; j < kNBT; ++j) {
        const cplx tj = (j < nbw) ? w.tau[cb + j] : mk(0.0, 0.0);
        cplx v = mk(0.0, 0.0);
        if (j < nbw) {
            if (t < j) {
                cplx s = mk(0.0, 0.0);
                for (int k = t; k < j; ++k) cfma(s, T[k * kNBT + t], T[j * kNBT + k]);     // row t of T(0:j,0:j) times G(0:j,j)
                v = mk(-tj.x, -tj.y) * s;
            } else if (t == j) v = tj;
        }
        __syncthreads();              // every thread has read column j of G
        T[j * kNBT + t] = v;
        __syncthreads();
    }
    cplx *Tg = w.Tm + (size_t)b * kNBT * kNBT;
    for (int e = t; e < kNBT * kNBT; e += kNBT) Tg[e] = T[e];
}

// VT_b = V_b T_b  (blockIdx.z = b, blockIdx.x = row tile)
__global__ void __launch_bounds__(BG_THREADS) bt_vt_kernel(BackWs w) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int b = blockIdx.z, cb = b * kNBT;
    const int nbw = min(kNBT, w.n - cb), m = w.n - cb - w.voff;
    if (m <= 0 || (int)blockIdx.x * 64 >= m) return;
    GemmProblem<cplx, cplx> p;
    p.A = w.A + (size_t)cb * w.lda + cb + w.voff; p.lda = w.lda;
    p.B = w.Tm + (size_t)b * kNBT * kNBT; p.ldb = kNBT;
    p.A2 = nullptr; p.B2 = nullptr; p.lda2 = p.ldb2 = 0; p.M = m; p.N = nbw; p.K = nbw; p.K2 = 0;
    StoreEpi epi{w.VT + (size_t)cb * w.lda + cb + w.voff, w.lda};
    gemm_tile_body<cplx, cplx, MNMAJ, KMAJ, false, false, BG_MI, BG_NI, BG_WM, BG_WN, false>(p, blockIdx.x, 0, smem_raw, epi);
}

// X_part[s] = V_b^H Z over the s-th chunk of rows (blockIdx.x = column tile, blockIdx.y = s, blockIdx.z = row tile)
// ST = 2: two CTAs (eight warps) per SM; three stages of the 64 x 64 instance need 122 KB of shared memory, one CTA per SM
template <int MI, int NI, int ST = kGemmStages>
__global__ void __launch_bounds__(BG_THREADS, (ST == 2 ? 2 : 1)) bt_vhz_kernel(BackWs w, int b) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int BN = BG_WN * NI * 8;
    const int kpos = w.cnt[1];
    if ((int)blockIdx.x * BN >= kpos) return;
    const int cb = b * kNBT, nbw = min(kNBT, w.n - cb), m = w.n - cb - w.voff;
    const int chunk = (((m + kSplitK - 1) / kSplitK) + 15) & ~15;
    const int k0 = blockIdx.y * chunk;
    const int klen = min(chunk, m - k0);
    GemmProblem<cplx, cplx> p;
    p.A = w.A + (size_t)cb * w.lda + cb + w.voff + k0; p.lda = w.lda;
    p.B = w.Zc + cb + w.voff + k0; p.ldb = w.ldz;
    p.A2 = nullptr; p.B2 = nullptr; p.lda2 = p.ldb2 = 0; p.M = nbw; p.N = kpos; p.K = klen > 0 ? klen : 0; p.K2 = 0;
    StoreEpi epi{w.Xp + (size_t)blockIdx.y * kNBT * w.n, kNBT};
    gemm_tile_body<cplx, cplx, KMAJ, KMAJ, true, false, MI, NI, BG_WM, BG_WN, false, ST>(p, blockIdx.z, blockIdx.x, smem_raw, epi);
}

__global__ void __launch_bounds__(256) bt_reduce_kernel(BackWs w) {
    const int kpos = w.cnt[1];
    const size_t tot = (size_t)kNBT * kpos;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < tot; i += (size_t)gridDim.x * 256) {
        cplx s = w.Xp[i];
#pragma unroll
        for (int k = 1; k < kSplitK; ++k) s = s + w.Xp[(size_t)k * kNBT * w.n + i];
        w.X[i] = s;
    }
}

// Z[cb+1:, :] -= VT_b X
template <int MI, int NI>
__global__ void __launch_bounds__(BG_THREADS, 3) bt_update_kernel(BackWs w, int b) {      // K = 64: two stages, 3 CTAs/SM
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int BM = BG_WM * MI * 8, BN = BG_WN * NI * 8;
    const int kpos = w.cnt[1];
    const int cb = b * kNBT, nbw = min(kNBT, w.n - cb), m = w.n - cb - w.voff;
    if ((int)blockIdx.y * BN >= kpos || (int)blockIdx.x * BM >= m) return;
    GemmProblem<cplx, cplx> p;
    p.A = w.VT + (size_t)cb * w.lda + cb + w.voff; p.lda = w.lda;
    p.B = w.X; p.ldb = kNBT;
    p.A2 = nullptr; p.B2 = nullptr; p.lda2 = p.ldb2 = 0; p.M = m; p.N = kpos; p.K = nbw; p.K2 = 0;
    SubEpi epi{w.Zc + cb + w.voff, w.ldz};
    gemm_tile_body<cplx, cplx, MNMAJ, KMAJ, false, false, MI, NI, BG_WM, BG_WN, false, 2>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
}

// ---- S7 + S8: lower triangle of W W^H packed as vec_R (Eq. D10) --------------------------------
struct PackEpi {
    SvecIo io; int n;
    bool bad;          // non-finite input (flag of S1): the block's output is NaN
    __device__ __forceinline__ void operator()(int i, int j, double re, double im) const {
        if (bad) { re = nan_(); im = nan_(); }
        const size_t c = svec_col_off(n, j);
        if (i == j) io_store(io, c, re);
        else { const int k = i - j - 1; io_store(io, c + 1 + 2 * k, kSqrt2 * re); io_store(io, c + 2 + 2 * k, kSqrt2 * im); }
    }
};

__global__ void __launch_bounds__(BG_THREADS) herk_pack_kernel(BackWs w, SvecIo io) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (blockIdx.y > blockIdx.x) return;
    GemmProblem<cplx, cplx> p;
    p.A = w.Zc; p.lda = w.ldz; p.B = w.Zc; p.ldb = w.ldz;
    p.A2 = nullptr; p.B2 = nullptr; p.lda2 = p.ldb2 = 0; p.M = w.n; p.N = w.n; p.K = w.cnt[1]; p.K2 = 0;
    const bool bad = w.cnt[2] != 0;
    if (bad && w.info != nullptr && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) *w.info = kInfoNonFinite;
    PackEpi epi{io, w.n, bad};
    gemm_tile_body<cplx, cplx, MNMAJ, MNMAJ, false, true, BG_MI, BG_NI, BG_WM, BG_WN, true>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
}

// ---- host driver -------------------------------------------------------------------------------
static int g_bh_init_dev = -1;
constexpr size_t kSmemKK = gemm_smem_bytes<cplx, cplx, KMAJ, KMAJ, BG_MI, BG_NI, BG_WM, BG_WN>();
constexpr size_t kSmemKK2 = gemm_smem_bytes<cplx, cplx, KMAJ, KMAJ, BG_MI, BG_NI, BG_WM, BG_WN, 2>();
constexpr size_t kSmemMK = gemm_smem_bytes<cplx, cplx, MNMAJ, KMAJ, BG_MI, BG_NI, BG_WM, BG_WN>();
constexpr size_t kSmemMK2 = gemm_smem_bytes<cplx, cplx, MNMAJ, KMAJ, BG_MI, BG_NI, BG_WM, BG_WN, 2>();
constexpr size_t kSmemKKs = gemm_smem_bytes<cplx, cplx, KMAJ, KMAJ, 2, 2, BG_WM, BG_WN>();
constexpr size_t kSmemMKs = gemm_smem_bytes<cplx, cplx, MNMAJ, KMAJ, 2, 2, BG_WM, BG_WN, 2>();
constexpr size_t kSmemMM = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, BG_MI, BG_NI, BG_WM, BG_WN>();

int backherk_init() {
    int dev = 0;
    cudaGetDevice(&dev);
    if (g_bh_init_dev == dev) return 0;
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bt_gram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemKK);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bt_tfactor_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(cplx) * kNBT * kNBT));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bt_vhz_kernel<4, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemKK);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bt_vhz_kernel<4, 4, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemKK2);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bt_vhz_kernel<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemKKs);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bt_update_kernel<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMKs);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bt_vt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMK);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bt_update_kernel<4, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMK2);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(herk_pack_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMM);
    if (e != cudaSuccess) return HPSD_ECUDA_;
    g_bh_init_dev = dev;
    return 0;
}

// Compact-WY factors of all reflector blocks (Gram matrices, T_b, V_b T_b): they depend on the reflectors only,
// so the large path runs them on a side stream next to the divide & conquer (S4).
int launch_bt_factors(const BackWs &w, cudaStream_t st) {
    const int n = w.n;
    int rc = backherk_init();
    if (rc) return rc;
    const int nblocks = (n + kNBT - 1) / kNBT;
    const int nt = (n + 63) / 64;
    bt_gram_kernel<<<dim3(kSplitK, 1, nblocks), BG_THREADS, kSmemKK, st>>>(w);
    HPSD_LAUNCH_CHECK();
    bt_tfactor_kernel<<<nblocks, kNBT, sizeof(cplx) * kNBT * kNBT, st>>>(w);
    HPSD_LAUNCH_CHECK();
    bt_vt_kernel<<<dim3(nt, 1, nblocks), BG_THREADS, kSmemMK, st>>>(w);
    HPSD_LAUNCH_CHECK();
    return 0;
}

int launch_back_herk(const BackWs &w, const double *lam, const double *Zt, int ldzt, const SvecIo &io, cudaStream_t st, bool factors_done,
                     const TwoStageWs *ts) {
    const int n = w.n;
    int rc = backherk_init();
    if (rc) return rc;
    const int nblocks = (n + kNBT - 1) / kNBT;
    const int nt = (n + 63) / 64;
    const bool small = n <= 1536;          // 32 x 32 CTA tiles keep the grid wide and the CTAs short
    prof_begin(ST_BACK, st);
    count_pos_kernel<<<1, 32, 0, st>>>(n, lam, w.cnt);
    HPSD_LAUNCH_CHECK();
    scale_convert_kernel<<<dim3((n + 1023) / 1024, n), 256, 0, st>>>(n, lam, Zt, ldzt, w.Zc, w.ldz, w.cnt);
    HPSD_LAUNCH_CHECK();
    if (!factors_done) {
        if (ts) { rc = launch_q2_factors(*ts, st); if (rc) return rc; }
        rc = launch_bt_factors(w, st);
        if (rc) return rc;
    }
    if (ts) {
        prof_end(ST_BACK, st);
        rc = launch_q2_apply(*ts, w.Zc, w.ldz, w.cnt, st);
        if (rc) return rc;
        prof_begin(ST_BACK, st);
    }
    for (int b = nblocks - 1; b >= 0; --b) {
        const int m = n - b * kNBT - w.voff;
        if (m <= 0) continue;
        if (small) bt_vhz_kernel<2, 2><<<dim3((n + 31) / 32, kSplitK, 2), BG_THREADS, kSmemKKs, st>>>(w, b);
        else if (n >= 3072) bt_vhz_kernel<4, 4, 2><<<dim3(nt, kSplitK, 1), BG_THREADS, kSmemKK2, st>>>(w, b);   // > 148 live CTAs: two per SM
        else bt_vhz_kernel<4, 4><<<dim3(nt, kSplitK, 1), BG_THREADS, kSmemKK, st>>>(w, b);
        HPSD_LAUNCH_CHECK();
        bt_reduce_kernel<<<(kNBT * n + 255) / 256 < 1184 ? (kNBT * n + 255) / 256 : 1184, 256, 0, st>>>(w);
        HPSD_LAUNCH_CHECK();
        if (small) bt_update_kernel<2, 2><<<dim3((m + 31) / 32, (n + 31) / 32), BG_THREADS, kSmemMKs, st>>>(w, b);
        else bt_update_kernel<4, 4><<<dim3((m + 63) / 64, nt), BG_THREADS, kSmemMK2, st>>>(w, b);
        HPSD_LAUNCH_CHECK();
    }
    prof_end(ST_BACK, st);
    prof_begin(ST_HERK_PACK, st);
    herk_pack_kernel<<<dim3(nt, nt), BG_THREADS, kSmemMM, st>>>(w, io);
    prof_end(ST_HERK_PACK, st);
    HPSD_LAUNCH_CHECK();
    return 0;
}

}  // namespace hpsd
