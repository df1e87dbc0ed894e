// backq2.cu -- the second back-transformation of the two-stage reduction (part of S5):
// Z <- Q2 Z, where Q2 is the product of the b-long reflectors H(s, k) of the bulge chasing (hb2st.cu), in the order
// they were applied: Q2 = prod_s prod_k H(s, k).
//
// Diamond blocking: the reflectors of hop k of g = kQ2G consecutive sweeps s0 .. s0+g-1 act on rows shifted by one
// each, so together they are one compact-WY block  I - V T V^H  with a parallelogram-shaped V ((b + g - 1) x g,
// column i non-zero in rows i .. i + b - 1).  Q2 Z is applied group by group from the last group of sweeps to the
// first, and inside a group in ascending k (the order that respects every pair of non-commuting reflectors).
//   q2_tfactor_kernel : T of every diamond block from V^H V (needs the reflectors only: runs next to S4)
//   q2_apply_kernel   : each CTA owns 32 columns of Z and walks over all diamond blocks; per block the window of
//                       b + g - 1 rows of Z is staged in shared memory and X = V^H Z_w, X <- T X, Z_w -= V X run as
//                       complex DMMA (mma.sync m8n8k4 f64) tiles that skip the all-zero 8 x 4 pieces of V and T.
#include "kernels.h"
#include "gemm.cuh"
#include "twostage.h"
#include "prof.h"

namespace hpsd {

constexpr int kQ2Threads = 128;
constexpr int kQ2NC = 32;                  // columns of Z per CTA
constexpr int kQ2Rows = kBW + kQ2G;        // window rows held in shared memory (b + g - 1, padded)
constexpr int kQ2VP = kBW + 5;             // pitch of the compact reflectors  Vs[i][t]
constexpr int kQ2TP = kQ2G + 4;            // pitch of T[i][k]
constexpr int kQ2ZP = kQ2NC + 2;           // pitch of the row-major window / X / X2
static_assert(kBW == 32 && kQ2G == 32 && kQ2NC == 32, "tiling of the Q2 kernels");

struct Q2Args {
    int n, ldz, nk, ng;
    const cplx *V2, *tau2;
    cplx *T2;
    cplx *Zc;
    const int *cnt;
    int *flags;          // per (slab, group): blocks finished (release/acquire)
};

__device__ __forceinline__ bool q2_exists(int n, int s, int k) { return s < n - 1 && s + 1 + k * kBW < n; }

// T factor of diamond block (gi = blockIdx.y, k = blockIdx.x), stored row-major [i][j] (upper triangular)
__global__ void __launch_bounds__(kQ2Threads) q2_tfactor_kernel(Q2Args a) {
    __shared__ cplx Vc[kQ2G][kBW + 1];        // the compact reflectors; T once the Gram matrix is formed
    __shared__ cplx G[kQ2G][kQ2G + 1];
    __shared__ cplx taus[kQ2G];
    cplx (*T)[kBW + 1] = Vc;
    const int k = blockIdx.x, gi = blockIdx.y, tid = threadIdx.x;
    const int n = a.n, s0 = gi * kQ2G;
    cplx *Tg = a.T2 + ((size_t)gi * a.nk + k) * kQ2G * kQ2G;
    if (!q2_exists(n, s0, k)) return;                    // the whole block is empty (never read)
    for (int e = tid; e < kQ2G * kBW; e += kQ2Threads) {
        const int i = e / kBW, t = e % kBW;
        Vc[i][t] = q2_exists(n, s0 + i, k) ? a.V2[((size_t)k * n + s0 + i) * kBW + t] : mk(0.0, 0.0);
    }
    if (tid < kQ2G) taus[tid] = q2_exists(n, s0 + tid, k) ? a.tau2[(size_t)k * n + s0 + tid] : mk(0.0, 0.0);
    __syncthreads();
    // G[i][j] = V[:, i]^H V[:, j] for i < j: rows i + t = j + t'
    for (int e = tid; e < kQ2G * kQ2G; e += kQ2Threads) {
        const int i = e / kQ2G, j = e % kQ2G;
        cplx acc = mk(0.0, 0.0);
        if (i < j) {
            const int sh = j - i;
            for (int t = sh; t < kBW; ++t) cfma_conj(acc, Vc[i][t], Vc[j][t - sh]);
        }
        G[i][j] = acc;
    }
    __syncthreads();
    for (int e = tid; e < kQ2G * kQ2G; e += kQ2Threads) T[e / kQ2G][e % kQ2G] = mk(0.0, 0.0);
    __syncthreads();
    // zlarft, forward columnwise:  T(0:j, j) = -tau_j T(0:j, 0:j) G(0:j, j),  T(j, j) = tau_j.  Lane r owns row r.
    if (tid < kQ2G) {
        const int r = tid;
        for (int j = 0; j < kQ2G; ++j) {
            const cplx tj = taus[j];
            if (r < j) {
                cplx s = mk(0.0, 0.0);
                for (int kk = r; kk < j; ++kk) cfma(s, T[r][kk], G[kk][j]);
                T[r][j] = mk(-tj.x, -tj.y) * s;
            } else if (r == j) T[r][j] = tj;
        }
    }
    __syncthreads();
    for (int e = tid; e < kQ2G * kQ2G; e += kQ2Threads) Tg[e] = T[e / kQ2G][e % kQ2G];
}

struct Q2Smem {
    cplx Zw[kQ2Rows * kQ2ZP];
    cplx X[kQ2G * kQ2ZP];
    cplx X2[kQ2G * kQ2ZP];
    cplx Vs[kQ2G * kQ2VP];
    cplx T[kQ2G * kQ2TP];
};

__device__ __forceinline__ int q2_ld_acquire(const int *p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void q2_st_release(int *p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
constexpr int kQ2Done = 1 << 30;

// Each slab of 32 columns of Z is served by P = gridDim.x / (active slabs) CTAs: CTA (slab, p) takes the sweep groups
// ng-1-p, ng-1-p-P, ...  Group gi follows group gi+1 (it must see gi+1's result wherever their rows overlap): block
// (gi, k) overlaps (gi+1, k-2 .. k), so it waits until group gi+1 has published k+1 finished blocks; the P CTAs of a
// slab therefore run as a pipeline one block apart.  Cooperative launch (all CTAs resident: a CTA spins on another's flag).
__global__ void __launch_bounds__(kQ2Threads, 2) q2_apply_kernel(Q2Args a) {
    extern __shared__ __align__(16) unsigned char q2_smem[];
    Q2Smem &S = *reinterpret_cast<Q2Smem *>(q2_smem);
    const int kpos = a.cnt[1];
    const int nact = (kpos + kQ2NC - 1) / kQ2NC;           // active slabs
    if (nact == 0) return;
    int P = (int)gridDim.x / nact; if (P < 1) P = 1;
    if (P > a.ng) P = a.ng;
    const int slab = blockIdx.x % nact, p = blockIdx.x / nact;
    if (p >= P) return;
    const int c0 = slab * kQ2NC;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int fr = lane >> 2, fk = lane & 3;
    const int n = a.n;
    cplx *Zg = a.Zc + (size_t)c0 * a.ldz;
    const int ncol = (kpos - c0 < kQ2NC) ? kpos - c0 : kQ2NC;
    int *flags = a.flags + (size_t)slab * a.ng;

    for (int gi = a.ng - 1 - p; gi >= 0; gi -= P) {
        const int s0 = gi * kQ2G;
        for (int k = 0; k < a.nk; ++k) {
            if (!q2_exists(n, s0, k)) break;
            const int R0 = s0 + 1 + k * kBW;
            const int wlen = (n - R0 < kBW + kQ2G - 1) ? n - R0 : kBW + kQ2G - 1;
            // ---- reflectors and T of this block: read-only data, no dependency
            for (int e = tid; e < kQ2G * kBW; e += kQ2Threads) {
                const int i = e / kBW, t = e % kBW;
                const bool ok = q2_exists(n, s0 + i, k);
                cp_async_16(&S.Vs[i * kQ2VP + t], ok ? a.V2 + ((size_t)k * n + s0 + i) * kBW + t : a.V2, ok);
            }
            {
                const cplx *Tg = a.T2 + ((size_t)gi * a.nk + k) * kQ2G * kQ2G;
                for (int e = tid; e < kQ2G * kQ2G; e += kQ2Threads) cp_async_16(&S.T[(e / kQ2G) * kQ2TP + (e % kQ2G)], Tg + e, true);
            }
            // ---- the window of Z: after the previous group has finished its blocks up to k
            if (gi + 1 < a.ng) {
                if (tid == 0) {
                    const int *pf = flags + gi + 1;
                    while (q2_ld_acquire(pf) < k + 1) { }
                }
                __syncthreads();
            }
            {
                const int rr = tid & 63, ch = tid >> 6;
#pragma unroll 4
                for (int t = 0; t < 16; ++t) {
                    const int c = ch * 16 + t;
                    const bool ok = rr < wlen && c < ncol;
                    cp_async_16(&S.Zw[rr * kQ2ZP + c], ok ? Zg + (size_t)c * a.ldz + R0 + rr : Zg, ok);
                }
            }
            cp_async_commit();
            cp_async_wait<0>();
            __syncthreads();
            // ---- X = V^H Zw: warp = 8 rows i of X, all 32 columns; K runs over window rows 8 warp .. 8 warp + 39
            {
                double re[4][2], im[4][2];
#pragma unroll
                for (int cb = 0; cb < 4; ++cb) { re[cb][0] = re[cb][1] = im[cb][0] = im[cb][1] = 0.0; }
                const int i = 8 * warp + fr;
#pragma unroll
                for (int ks = 0; ks < (kBW + 8) / 4; ++ks) {
                    const int rw = 8 * warp + 4 * ks + fk;           // window row
                    const int t = rw - i;
                    cplx av = mk(0.0, 0.0);
                    if (t >= 0 && t < kBW) av = S.Vs[i * kQ2VP + t];
                    const double ar = av.x, ai = -av.y;              // conj
#pragma unroll
                    for (int cb = 0; cb < 4; ++cb) {
                        const cplx bv = S.Zw[rw * kQ2ZP + cb * 8 + fr];
                        dmma(re[cb][0], re[cb][1], ar, bv.x);
                        dmma(re[cb][0], re[cb][1], -ai, bv.y);
                        dmma(im[cb][0], im[cb][1], ar, bv.y);
                        dmma(im[cb][0], im[cb][1], ai, bv.x);
                    }
                }
#pragma unroll
                for (int cb = 0; cb < 4; ++cb)
#pragma unroll
                    for (int e = 0; e < 2; ++e) S.X[i * kQ2ZP + cb * 8 + 2 * fk + e] = mk(re[cb][e], im[cb][e]);
            }
            __syncthreads();
            // ---- X2 = T X (T upper triangular: K from the diagonal block on)
            {
                double re[4][2], im[4][2];
#pragma unroll
                for (int cb = 0; cb < 4; ++cb) { re[cb][0] = re[cb][1] = im[cb][0] = im[cb][1] = 0.0; }
                const int i = 8 * warp + fr;
                for (int kk = 8 * warp; kk < kQ2G; kk += 4) {
                    const cplx av = S.T[i * kQ2TP + kk + fk];
#pragma unroll
                    for (int cb = 0; cb < 4; ++cb) {
                        const cplx bv = S.X[(kk + fk) * kQ2ZP + cb * 8 + fr];
                        dmma(re[cb][0], re[cb][1], av.x, bv.x);
                        dmma(re[cb][0], re[cb][1], -av.y, bv.y);
                        dmma(im[cb][0], im[cb][1], av.x, bv.y);
                        dmma(im[cb][0], im[cb][1], av.y, bv.x);
                    }
                }
#pragma unroll
                for (int cb = 0; cb < 4; ++cb)
#pragma unroll
                    for (int e = 0; e < 2; ++e) S.X2[i * kQ2ZP + cb * 8 + 2 * fk + e] = mk(re[cb][e], im[cb][e]);
            }
            __syncthreads();
            // ---- Zw -= V X2: warp takes the row blocks (warp, warp + 4): 8 k-steps of non-zero V pieces in total
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int Rb = warp + 4 * h;
                const int rw = 8 * Rb + fr;
                int ilo = 8 * Rb - (kBW - 1); if (ilo < 0) ilo = 0; ilo &= ~3;
                int ihi = 8 * Rb + 7; if (ihi > kQ2G - 1) ihi = kQ2G - 1;
                double re[4][2], im[4][2];
#pragma unroll
                for (int cb = 0; cb < 4; ++cb) { re[cb][0] = re[cb][1] = im[cb][0] = im[cb][1] = 0.0; }
                for (int is = ilo; is <= ihi; is += 4) {
                    const int i = is + fk;
                    const int t = rw - i;
                    cplx av = mk(0.0, 0.0);
                    if (t >= 0 && t < kBW) av = S.Vs[i * kQ2VP + t];
#pragma unroll
                    for (int cb = 0; cb < 4; ++cb) {
                        const cplx bv = S.X2[i * kQ2ZP + cb * 8 + fr];
                        dmma(re[cb][0], re[cb][1], av.x, bv.x);
                        dmma(re[cb][0], re[cb][1], -av.y, bv.y);
                        dmma(im[cb][0], im[cb][1], av.x, bv.y);
                        dmma(im[cb][0], im[cb][1], av.y, bv.x);
                    }
                }
                // straight from the accumulators to global memory (C fragment: row rw, column pairs)
                if (rw < wlen) {
#pragma unroll
                    for (int cb = 0; cb < 4; ++cb)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int c = cb * 8 + 2 * fk + e;
                            if (c < ncol) {
                                cplx z = S.Zw[rw * kQ2ZP + c];
                                z.x -= re[cb][e]; z.y -= im[cb][e];
                                Zg[(size_t)c * a.ldz + R0 + rw] = z;
                            }
                        }
                }
            }
            __syncthreads();                                     // all stores issued; the staging buffers are free
            if (tid == 0) q2_st_release(flags + gi, q2_exists(n, s0, k + 1) && k + 1 < a.nk ? k + 1 : kQ2Done);
        }
    }
}

static int g_q2_init_dev = -1;
int backq2_init() {
    int dev = 0;
    cudaGetDevice(&dev);
    if (g_q2_init_dev == dev) return 0;
    if (cudaFuncSetAttribute(q2_apply_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Q2Smem)) != cudaSuccess) return HPSD_ECUDA_;
    g_q2_init_dev = dev;
    return 0;
}

static int q2_groups(int n) { return n > 1 ? (n - 1 + kQ2G - 1) / kQ2G : 0; }
size_t twostage_q2_blocks(int n) { return (size_t)q2_groups(n) * twostage_hops(n); }

int launch_q2_factors(const TwoStageWs &w, cudaStream_t st) {
    const int n = w.n;
    if (n <= 1) return 0;
    Q2Args a{n, 0, (int)twostage_hops(n), q2_groups(n), w.V2, w.tau2, w.T2, nullptr, nullptr, nullptr};
    q2_tfactor_kernel<<<dim3(a.nk, a.ng), kQ2Threads, 0, st>>>(a);
    HPSD_LAUNCH_CHECK();
    return 0;
}

int launch_q2_apply(const TwoStageWs &w, cplx *Zc, int ldz, const int *cnt, cudaStream_t st) {
    const int n = w.n;
    if (n <= 1) return 0;
    int rc = backq2_init();
    if (rc) return rc;
    Q2Args a{n, ldz, (int)twostage_hops(n), q2_groups(n), w.V2, w.tau2, w.T2, Zc, cnt, w.q2flags};
    const int nslab = (n + kQ2NC - 1) / kQ2NC;
    HPSD_CUDA_OK(cudaMemsetAsync(w.q2flags, 0, sizeof(int) * (size_t)nslab * a.ng, st));
    int dev = 0, sms = 148, per_sm = 1;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, q2_apply_kernel, kQ2Threads, sizeof(Q2Smem)) != cudaSuccess || per_sm < 1) per_sm = 1;
    if (per_sm > 2) per_sm = 2;
    void *args[] = {&a};
    prof_begin(ST_BACKQ2, st);
    const cudaError_t e = cudaLaunchCooperativeKernel((void *)q2_apply_kernel, dim3(sms * per_sm), dim3(kQ2Threads), args, sizeof(Q2Smem), st);
    prof_end(ST_BACKQ2, st);
    g_launches++;
    return e == cudaSuccess ? 0 : HPSD_ECUDA_;
}

}  // namespace hpsd
