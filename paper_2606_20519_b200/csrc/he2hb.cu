// he2hb.cu -- S2 of SURVEY.md §8(a): dense Hermitian -> Hermitian band of width b = kBW, A = Q1 B Q1^H.
// First half of the "eigendecomposition" of PAPER.md:1536 in its two-stage form (BASELINE.json north star (c)).
//
// Per panel k (columns j0 = k b .. j0 + b - 1, trailing size m = n - j0 - b):
//   [QR]   Householder QR of the m x b panel A[j0+b:, j0:j0+b] inside ONE 16-CTA cluster (he2hb_panel_kernel):
//          rows are dealt to the CTAs and live in shared memory, every column step needs ONE all-to-all exchange
//          (st.async + mbarrier, cluster.cuh): the CTAs exchange the b inner products of the raw column with all
//          panel columns; norm, v^H P and the column V^H v of the T recurrence all follow from them.
//          R goes to the band, V (explicit unit diagonal) to V1, T to Tk.
//   [HEMM] Zp[s] = A22[:, K_s] V[K_s, :]           split-K complex DMMA GEMM over all SMs (A22 is stored in full)
//   [ZSUM] Z = sum_s Zp[s];  [GRAM] G = V^H Z (split-K DMMA);  [S] S = -1/2 T^H G T
//   [X]    X = Z T + V S                            (= A22 V T - 1/2 V T^H V^H A22 V T)
//   [HER2K] A22 -= X V^H + V X^H                    lower tiles on DMMA, each element mirrored into the upper triangle
// so that all (16/3) n^3 flops of the reduction are BLAS-3 and the dependent chain is n cluster exchanges instead of
// 2 n grid-wide barriers.
#include "kernels.h"
#include "gemm.cuh"
#include "cluster.cuh"
#include "large.h"
#include "twostage.h"
#include "prof.h"

namespace hpsd {

constexpr int kQrCl = 16;                 // CTAs per cluster (non-portable size)
constexpr int kQrWarps = 10;              // warp 0: top b x b block (kept by every CTA), warps 1..8: one row per thread, warp 9: T
constexpr int kQrThreads = kQrWarps * 32;
constexpr int kQrRows = 256;              // ordinary rows per CTA
constexpr int kQrP = kBW + 1;             // shared-memory pitch (elements): row-wise and column-wise accesses conflict free
static_assert(kBW == 32, "the panel kernel maps lane = panel column");

struct QrArgs {
    int n, lda, ldv, ldab, j0;
    const cplx *A;
    cplx *V1, *tau1, *Tk, *AB;
};

struct QrSmem {
    static constexpr size_t mbar = 0;                                            // two mbarriers
    static constexpr size_t land = 16;                                           // [2][kQrCl][kBW]
    static constexpr size_t part = land + sizeof(cplx) * 2 * kQrCl * kBW;        // [2][kQrWarps][kBW]
    static constexpr size_t row = part + sizeof(cplx) * 2 * kQrWarps * kBW;      // [2][kBW]
    static constexpr size_t qw = row + sizeof(cplx) * 2 * kBW;                   // [kBW]
    static constexpr size_t tau = qw + sizeof(cplx) * kBW;                       // [kBW]
    static constexpr size_t scl = tau + sizeof(cplx) * kBW;                      // [kBW]
    static constexpr size_t top = scl + sizeof(cplx) * kBW;                      // [kBW][kQrP]
    static constexpr size_t tf = top + sizeof(cplx) * kBW * kQrP;                // [kBW][kQrP]
    static constexpr size_t fb = tf + sizeof(cplx) * kBW * kQrP;                 // [kQrWarps][kBW]: update coefficients per warp
    static constexpr size_t total = fb + sizeof(cplx) * kQrWarps * kBW;
};

// zlarfg scalars: H = I - tau v v^H with v = [1; x scale] maps [alpha; x] to [beta; 0], beta real
__device__ __forceinline__ void qr_householder(cplx alpha, double xnorm2, double &beta, cplx &tau, cplx &scale) {
    if (xnorm2 == 0.0 && alpha.y == 0.0) {
        beta = alpha.x; tau = mk(0.0, 0.0); scale = mk(0.0, 0.0);
    } else {
        // one reciprocal square root (refined by a Newton step to full accuracy) and one reciprocal on the dependent chain
        const double s = alpha.x * alpha.x + alpha.y * alpha.y + xnorm2;
        double rinv = rsqrt(s);
        rinv = fma(0.5 * rinv, fma(-s * rinv, rinv, 1.0), rinv);
        const double nrm = s * rinv;
        beta = -copysign(nrm, alpha.x);
        const double ib = -copysign(rinv, alpha.x);
        tau = mk((beta - alpha.x) * ib, -alpha.y * ib);
        const cplx den = mk(alpha.x - beta, alpha.y);
        const double id2 = __drcp_rn(abs2(den));
        scale = mk(den.x * id2, -den.y * id2);
    }
}

// acc_lane += sum over rows r0 <= r < r1 of conj(P[r][j]) P[r][lane]
__device__ __forceinline__ cplx qr_dots(const cplx *P, int r0, int r1, int j, int lane) {
    cplx a0 = mk(0.0, 0.0), a1 = a0, a2 = a0, a3 = a0;
    int r = r0;
    for (; r + 3 < r1; r += 4) {
        const cplx x0 = P[(r + 0) * kQrP + j], p0 = P[(r + 0) * kQrP + lane];
        const cplx x1 = P[(r + 1) * kQrP + j], p1 = P[(r + 1) * kQrP + lane];
        const cplx x2 = P[(r + 2) * kQrP + j], p2 = P[(r + 2) * kQrP + lane];
        const cplx x3 = P[(r + 3) * kQrP + j], p3 = P[(r + 3) * kQrP + lane];
        cfma_conj(a0, x0, p0); cfma_conj(a1, x1, p1); cfma_conj(a2, x2, p2); cfma_conj(a3, x3, p3);
    }
    for (; r < r1; ++r) cfma_conj(a0, P[r * kQrP + j], P[r * kQrP + lane]);
    return (a0 + a1) + (a2 + a3);
}

// rows r0 <= r < r1:  P[r][lane] -= f (P[r][j] scale)   for lane > j   (f = 0 on the other lanes)
__device__ __forceinline__ void qr_update(cplx *P, int r0, int r1, int j, int lane, cplx f, cplx scale) {
    const cplx nf = mk(-f.x, -f.y);
    if (lane <= j) return;
#pragma unroll 4
    for (int r = r0; r < r1; ++r) {
        const cplx v = P[r * kQrP + j] * scale;
        cplx p = P[r * kQrP + lane];
        cfma(p, nf, v);
        P[r * kQrP + lane] = p;
    }
}

// ---- ordinary rows: thread = row, the 32 panel entries of the row live in REGISTERS (shared memory cannot feed one
// pass over 256 x 32 complex per column step: 3000 cycles of LDS/STS wavefronts per step, measured).  The array is
// rotated by one position per step, so that the active column is always p[0] and every index is static:
// after step j, p[k] holds panel column (j + 1 + k) mod 32.
//
// Warp-wide sums of the 32 products conj(p[0]) p[k] by a depth-first halving butterfly: the recursion keeps only
// log2(32) partial sums alive.  Lane L ends up with the sum of index L.
template <int A, int LEN>
__device__ __forceinline__ cplx qr_reduce(const cplx (&p)[kBW], cplx x, int lane) {
    if constexpr (LEN == 1) {
        cplx c = mk(0.0, 0.0);
        cfma_conj(c, x, p[A]);
        return c;
    } else {
        const cplx lo = qr_reduce<A, LEN / 2>(p, x, lane);
        const cplx hi = qr_reduce<A + LEN / 2, LEN / 2>(p, x, lane);
        const bool up = (lane & (LEN / 2)) != 0;
        const cplx keep = up ? hi : lo, send = up ? lo : hi;
        return mk(keep.x + __shfl_xor_sync(0xffffffffu, send.x, LEN / 2), keep.y + __shfl_xor_sync(0xffffffffu, send.y, LEN / 2));
    }
}

__global__ void __launch_bounds__(kQrThreads, 1) he2hb_panel_kernel(QrArgs a) {
    extern __shared__ __align__(16) unsigned char sm[];
    cplx *s_land = reinterpret_cast<cplx *>(sm + QrSmem::land);
    cplx *s_part = reinterpret_cast<cplx *>(sm + QrSmem::part);
    cplx *s_row = reinterpret_cast<cplx *>(sm + QrSmem::row);
    cplx *s_qw = reinterpret_cast<cplx *>(sm + QrSmem::qw);
    cplx *s_tau = reinterpret_cast<cplx *>(sm + QrSmem::tau);
    cplx *s_scl = reinterpret_cast<cplx *>(sm + QrSmem::scl);
    cplx *s_top = reinterpret_cast<cplx *>(sm + QrSmem::top);
    cplx *s_T = reinterpret_cast<cplx *>(sm + QrSmem::tf);
    cplx *s_f = reinterpret_cast<cplx *>(sm + QrSmem::fb);
    const unsigned mbar0 = cx_smem_u32(sm + QrSmem::mbar);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int rank = (int)cx_rank();
    const int n = a.n, j0 = a.j0, lda = a.lda;
    const int g0 = j0 + kBW;                     // global row of panel row 0
    const int m = n - g0;                        // panel rows (> 0)
    const int mo = m > kBW ? m - kBW : 0;        // ordinary rows (below the top block)
    const int rpc = (mo + kQrCl - 1) / kQrCl;    // per CTA (<= kQrRows)
    const int lo = rank * rpc;
    const int cnt = mo - lo < 0 ? 0 : (mo - lo < rpc ? mo - lo : rpc);
    const int nsteps = m < kBW ? m : kBW;

    if (tid == 0) {
        cx_mbar_init(mbar0, 1);
        cx_mbar_init(mbar0 + 8, 1);
        cx_fence_mbar_init();
        cx_arm(mbar0, kQrCl * kBW * (unsigned)sizeof(cplx));
        cx_arm(mbar0 + 8, kQrCl * kBW * (unsigned)sizeof(cplx));
    }
    // top block (every CTA keeps and updates its own copy, bit-identically)
    for (int e = tid; e < kBW * kBW; e += kQrThreads) {
        const int l = e % kBW, k = e / kBW;
        s_top[l * kQrP + k] = (l < m) ? a.A[(size_t)(j0 + k) * lda + g0 + l] : mk(0.0, 0.0);
        s_T[l * kQrP + k] = mk(0.0, 0.0);
    }
    if (tid < kBW) { s_tau[tid] = mk(0.0, 0.0); s_scl[tid] = mk(0.0, 0.0); }
    // ordinary rows of this CTA: thread = row (coalesced 512-byte segments per panel column), straight into registers
    cplx p[kBW];
    const int myrow = (warp - 1) * 32 + lane;
    const bool has_row = warp >= 1 && warp <= 8 && myrow < cnt;
    {
        const cplx *src = a.A + (size_t)j0 * lda + g0 + kBW + lo + (has_row ? myrow : 0);
#pragma unroll
        for (int k = 0; k < kBW; ++k) p[k] = has_row ? src[(size_t)k * lda] : mk(0.0, 0.0);
    }
    // diagonal block of this panel -> band (final: no later update touches it)
    if (rank == kQrCl - 1) {
        for (int e = tid; e < kBW * kBW; e += kQrThreads) {
            const int r = e % kBW, c = e / kBW;
            if (r >= c) a.AB[(size_t)(j0 + c) * a.ldab + (r - c)] = a.A[(size_t)(j0 + c) * lda + j0 + r];
        }
    }
    __syncthreads();
    cx_barrier();                                // every mbarrier of the cluster is initialised and armed

    const bool row_warp = warp >= 1 && warp <= 8 && (warp - 1) * 32 < cnt;      // warp-uniform

    for (int j = 0; j < nsteps; ++j) {
        const int par = j & 1;
        // ---- inner products of the raw column j with every panel column, over the rows below the diagonal row
        cplx acc = mk(0.0, 0.0);
        if (warp == 0) {
            s_row[par * kBW + lane] = s_top[j * kQrP + lane];
            if (rank == 0) acc = qr_dots(s_top, j + 1, kBW, j, lane);
        } else if (row_warp) {
            // index L of the rotated array is panel column (j + L) mod 32
            const cplx red = qr_reduce<0, kBW>(p, p[0], lane);
            acc.x = __shfl_sync(0xffffffffu, red.x, (lane - j) & (kBW - 1));
            acc.y = __shfl_sync(0xffffffffu, red.y, (lane - j) & (kBW - 1));
        }
        // (double-buffered: a warp that is through the exchange of step j may write its step j + 1 partial while a slower
        // warp of this CTA is still summing the partials of step j)
        cplx *sp = s_part + par * kQrWarps * kBW;
        sp[warp * kBW + lane] = acc;
        __syncthreads();
        if (warp < kQrCl / 2) {
            cplx tot = sp[lane];
#pragma unroll
            for (int w = 1; w < kQrWarps; ++w) tot = tot + sp[w * kBW + lane];
            const unsigned dst = cx_smem_u32(s_land + (par * kQrCl + rank) * kBW + lane);
            const unsigned mb = mbar0 + 8u * par;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int peer = 2 * warp + t;
                cx_st_async(cx_mapa(dst, peer), tot, cx_mapa(mb, peer));
            }
        }
        cx_wait(mbar0 + 8u * par, (unsigned)(j >> 1) & 1u);
        if (tid == 0) cx_arm(mbar0 + 8u * par, kQrCl * kBW * (unsigned)sizeof(cplx));      // for step j + 2
        // ---- every warp: totals (fixed order: bit-identical in all CTAs), Householder scalars, update coefficients
        cplx g = s_land[(par * kQrCl) * kBW + lane];
#pragma unroll
        for (int p = 1; p < kQrCl; ++p) g = g + s_land[(par * kQrCl + p) * kBW + lane];
        if (lane < j) g = conj_(g);              // sum conj(P[:,k]) x  for the finished columns k < j
        const double xnorm2 = __shfl_sync(0xffffffffu, g.x, j);
        const cplx rowv = s_row[par * kBW + lane];
        cplx alpha;
        alpha.x = __shfl_sync(0xffffffffu, rowv.x, j);
        alpha.y = __shfl_sync(0xffffffffu, rowv.y, j);
        double beta; cplx tau, scale;
        qr_householder(alpha, xnorm2, beta, tau, scale);
        cplx f = mk(0.0, 0.0);
        if (lane > j) f = conj_(tau) * (rowv + conj_(scale) * g);     // conj(tau) v^H P[:, lane]
        if (warp == 0) {
            if (lane > j) s_top[j * kQrP + lane] = rowv - f;
            else if (lane == j) { s_top[j * kQrP + j] = mk(beta, 0.0); s_tau[j] = tau; s_scl[j] = scale; }
            qr_update(s_top, j + 1, kBW, j, lane, f, scale);
            __syncwarp();
        } else if (row_warp) {
            // every thread needs the coefficients of ALL remaining columns: through the warp's own shared-memory line
            s_f[warp * kBW + lane] = f;
            __syncwarp();
            const cplx v = p[0] * scale;
            const cplx nv = mk(-v.x, -v.y);
#pragma unroll
            for (int k = 1; k < kBW; ++k)
                if (k <= kBW - 1 - j) cfma(p[k], s_f[warp * kBW + ((j + k) & (kBW - 1))], nv);      // columns j+1 .. 31 only
            __syncwarp();
            // rotate: the next step's column moves to p[0]; the raw column j (V = p scl_j) goes to the end
            const cplx x = p[0];
#pragma unroll
            for (int k = 0; k < kBW - 1; ++k) p[k] = p[k + 1];
            p[kBW - 1] = x;
        } else if (warp == kQrWarps - 1 && rank == 0) {
            // column j of T:  T(0:j, j) = -tau T(0:j, 0:j) (V(:, 0:j)^H v_j),  T(j, j) = tau   (zlarft, forward columnwise)
            // V[:, k] = P[:, k] scl[k] below its unit entry, so  V(:,k)^H v_j = conj(V[j,k]) + conj(scl_k) scale sum_{l>j} conj(P[l,k]) P[l,j]
            if (lane < j) {
                const cplx sk = conj_(s_scl[lane]);
                s_qw[lane] = sk * conj_(rowv) + (sk * scale) * g;
            }
            __syncwarp();
            if (lane < j) {
                cplx s = mk(0.0, 0.0);
                for (int k = lane; k < j; ++k) cfma(s, s_T[lane * kQrP + k], s_qw[k]);
                s_T[lane * kQrP + j] = mk(-tau.x, -tau.y) * s;
            } else if (lane == j) s_T[j * kQrP + j] = tau;
            __syncwarp();
        }
    }
    __syncthreads();
    // ---- results: V (unit diagonal explicit; zeros above come from the memset of V1), R -> band, tau, T
    if (has_row) {
        // ordinary rows exist only when the panel has 32 steps: 32 rotations put p[k] back on column k
        cplx *dst = a.V1 + (size_t)j0 * a.ldv + g0 + kBW + lo + myrow;
#pragma unroll
        for (int k = 0; k < kBW; ++k) dst[(size_t)k * a.ldv] = p[k] * s_scl[k];
    }
    if (rank == 0) {
        for (int e = tid; e < kBW * kBW; e += kQrThreads) {
            const int l = e % kBW, k = e / kBW;
            if (l < m) {
                if (l > k) a.V1[(size_t)(j0 + k) * a.ldv + g0 + l] = s_top[l * kQrP + k] * s_scl[k];
                else {
                    if (l == k) a.V1[(size_t)(j0 + k) * a.ldv + g0 + l] = mk(1.0, 0.0);
                    a.AB[(size_t)(j0 + k) * a.ldab + (kBW + l - k)] = s_top[l * kQrP + k];
                }
            }
            a.Tk[e] = s_T[l * kQrP + k];          // column-major b x b
        }
        if (tid < kBW) a.tau1[j0 + tid] = s_tau[tid];
    }
    cx_barrier();                                // no CTA of the cluster exits while a peer may still address its memory
}

// last diagonal block(s): no panel below them
__global__ void he2hb_tail_kernel(int n, int j0, const cplx *__restrict__ A, int lda, cplx *__restrict__ AB, int ldab) {
    const int w = n - j0;
    for (int e = threadIdx.x; e < w * w; e += blockDim.x) {
        const int r = e % w, c = e / w;
        if (r >= c) AB[(size_t)(j0 + c) * ldab + (r - c)] = A[(size_t)(j0 + c) * lda + j0 + r];
    }
}

// ---------------------------------------------------------------- trailing update
constexpr int HM_MI = 4, HM_NI = 2, HM_WM = 2, HM_WN = 2;       // 64 x 32 CTA tile, 4 warps
constexpr int HM_THREADS = HM_WM * HM_WN * 32;

struct HemmArgs {
    int m, lda, ldv, ldz, chunk;
    const cplx *A22, *V;
    cplx *Zp;
};
struct StoreEpi2 {
    cplx *C; int ld;
    __device__ __forceinline__ void operator()(int i, int j, double re, double im) const { C[(size_t)j * ld + i] = mk(re, im); }
};

// Zp[s] = A22[:, k0:k0+chunk] V[k0:k0+chunk, :]   (blockIdx.x = 64-row tile, blockIdx.y = s)
__global__ void __launch_bounds__(HM_THREADS, 2) he2hb_hemm_kernel(HemmArgs h) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int k0 = blockIdx.y * h.chunk;
    int klen = h.m - k0; if (klen > h.chunk) klen = h.chunk; if (klen < 0) klen = 0;
    GemmProblem<cplx, cplx> p;
    p.A = h.A22 + (size_t)k0 * h.lda; p.lda = h.lda;
    p.B = h.V + k0; p.ldb = h.ldv;
    p.A2 = nullptr; p.B2 = nullptr; p.lda2 = p.ldb2 = 0; p.M = h.m; p.N = kBW; p.K = klen; p.K2 = 0;
    StoreEpi2 epi{h.Zp + (size_t)blockIdx.y * h.ldz * kBW, h.ldz};
    gemm_tile_body<cplx, cplx, MNMAJ, KMAJ, false, false, HM_MI, HM_NI, HM_WM, HM_WN, false, 2>(p, blockIdx.x, 0, smem_raw, epi);
}

struct SlabArgs {
    int m, ldv, ldz, splits, nslabs;      // nslabs: number of Gram partials
    const cplx *V, *Zp, *Tk;
    cplx *Z, *Gp, *S;
    unsigned *counter;
};

// Z = sum_s Zp[s]: one element per thread, all split-K partials of the element in flight at once
// (a load -> add loop would be a chain of L2 round trips)
__global__ void __launch_bounds__(256) he2hb_zsum_kernel(SlabArgs s) {
    const int e = blockIdx.x * 256 + threadIdx.x;
    if (e >= s.m * kBW) return;
    const int r = e % s.m, c = e / s.m;
    cplx zp[kHemmSplitMax];
#pragma unroll
    for (int k = 0; k < kHemmSplitMax; ++k) zp[k] = (k < s.splits) ? s.Zp[((size_t)k * kBW + c) * s.ldz + r] : mk(0.0, 0.0);
    cplx z = mk(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < kHemmSplitMax; ++k) z = z + zp[k];
    s.Z[(size_t)c * s.ldz + r] = z;
}

// Gp[s] = V[K_s, :]^H Z[K_s, :]: split-K complex DMMA GEMM (32 x 32 output per CTA); summed in a fixed order by he2hb_s_kernel
constexpr int GR_MI = 2, GR_NI = 2, GR_WM = 2, GR_WN = 2;
__global__ void __launch_bounds__(GR_WM *GR_WN * 32) he2hb_gram_kernel(SlabArgs s, int chunk) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int k0 = blockIdx.x * chunk;
    int klen = s.m - k0; if (klen > chunk) klen = chunk; if (klen < 0) klen = 0;
    GemmProblem<cplx, cplx> p;
    p.A = s.V + k0; p.lda = s.ldv; p.B = s.Z + k0; p.ldb = s.ldz;
    p.A2 = nullptr; p.B2 = nullptr; p.lda2 = p.ldb2 = 0; p.M = kBW; p.N = kBW; p.K = klen; p.K2 = 0;
    StoreEpi2 epi{s.Gp + (size_t)blockIdx.x * kBW * kBW, kBW};
    gemm_tile_body<cplx, cplx, KMAJ, KMAJ, true, false, GR_MI, GR_NI, GR_WM, GR_WN, false>(p, 0, 0, smem_raw, epi);
}

// S = -1/2 T^H (sum of the slabs' Gram partials) T, one CTA of 1024 threads (thread = matrix element).  A kernel of its
// own: the partials come from other CTAs, and reading them inside the slab kernel needs gpu-scope loads
// (LDG.STRONG.GPU, ~170 issue cycles each: 80 us per panel, measured); across a launch boundary plain loads do.
__global__ void __launch_bounds__(kBW * kBW) he2hb_s_kernel(SlabArgs s) {
    __shared__ cplx sG[kBW][kBW], sT[kBW][kBW], sM[kBW][kBW];        // 48 KB, [row][col]
    // thread = (r, c) with c fastest: in the products below the left operand is a broadcast and the right one a
    // conflict-free row; the (column-major) global reads are coalesced and transposed on their way into shared memory
    const int e = threadIdx.x;
    {
        const int gr = e % kBW, gc = e / kBW;              // element e of a column-major b x b matrix
        cplx g = mk(0.0, 0.0);
        for (int k0 = 0; k0 < s.nslabs; k0 += 8) {          // eight independent loads per round trip, fixed summation order
            cplx gp[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) gp[k] = (k0 + k < s.nslabs) ? s.Gp[(size_t)(k0 + k) * kBW * kBW + e] : mk(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < 8; ++k) g = g + gp[k];
        }
        sG[gr][gc] = g;
        sT[gr][gc] = s.Tk[e];
    }
    __syncthreads();
    const int r = e / kBW, c = e % kBW;
    cplx acc = mk(0.0, 0.0);
    for (int k = 0; k <= c; ++k) cfma(acc, sG[r][k], sT[k][c]);             // M = G T, T upper triangular
    sM[r][c] = acc;
    __syncthreads();
    acc = mk(0.0, 0.0);
    for (int k = 0; k <= r; ++k) cfma_conj(acc, sT[k][r], sM[k][c]);        // T^H M
    s.S[r + c * kBW] = mk(-0.5 * acc.x, -0.5 * acc.y);
}

struct XArgs {
    int m, ldv, ldz;
    const cplx *Z, *V, *Tk, *S;
    cplx *X;
};
// X = Z T + V S     (blockIdx.x = 64-row tile)
__global__ void __launch_bounds__(HM_THREADS, 2) he2hb_x_kernel(XArgs x) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    GemmProblem<cplx, cplx> p;
    p.A = x.Z; p.lda = x.ldz; p.B = x.Tk; p.ldb = kBW;
    p.A2 = x.V; p.lda2 = x.ldv; p.B2 = x.S; p.ldb2 = kBW;
    p.M = x.m; p.N = kBW; p.K = kBW; p.K2 = kBW;
    StoreEpi2 epi{x.X, x.ldz};
    gemm_tile_body<cplx, cplx, MNMAJ, KMAJ, false, false, HM_MI, HM_NI, HM_WM, HM_WN, false, 2>(p, blockIdx.x, 0, smem_raw, epi);
}

// A22 -= X V^H + V X^H on the lower tiles; every updated element is mirrored into the upper triangle, so that the
// next panel's HEMM reads a plain full matrix
struct Her2kFullEpi {
    cplx *C; int ldc;
    static constexpr bool kRmw = true;
    __device__ __forceinline__ cplx load(int i, int j) const { return C[(size_t)j * ldc + i]; }
    __device__ __forceinline__ void store(int i, int j, cplx v, double re, double im) const {
        v.x -= re; v.y -= im;
        if (i == j) v.y = 0.0;
        C[(size_t)j * ldc + i] = v;
        if (i != j) C[(size_t)i * ldc + j] = conj_(v);
    }
};
constexpr int H2F_MI = 4, H2F_NI = 4, H2F_WM = 2, H2F_WN = 2;
__global__ void __launch_bounds__(H2F_WM *H2F_WN * 32, 3) he2hb_her2k_kernel(GemmProblem<cplx, cplx> p, Her2kFullEpi epi) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (blockIdx.y > blockIdx.x) return;
    gemm_tile_body<cplx, cplx, MNMAJ, MNMAJ, false, true, H2F_MI, H2F_NI, H2F_WM, H2F_WN, true, 2>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
}
__global__ void __launch_bounds__(H2F_WM *H2F_WN * 32) he2hb_her2k_small_kernel(GemmProblem<cplx, cplx> p, Her2kFullEpi epi) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (blockIdx.y > blockIdx.x) return;
    gemm_tile_body<cplx, cplx, MNMAJ, MNMAJ, false, true, 2, 2, H2F_WM, H2F_WN, true>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
}

// ---------------------------------------------------------------- host driver
static int g_ts_init_dev = -1;
static int g_ts_ok = 0;
constexpr size_t kSmemHemm = gemm_smem_bytes<cplx, cplx, MNMAJ, KMAJ, HM_MI, HM_NI, HM_WM, HM_WN, 2>();
constexpr size_t kSmemH2F = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, H2F_MI, H2F_NI, H2F_WM, H2F_WN, 2>();
constexpr size_t kSmemH2Fs = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, 2, 2, H2F_WM, H2F_WN>();
constexpr size_t kSmemGram = gemm_smem_bytes<cplx, cplx, KMAJ, KMAJ, GR_MI, GR_NI, GR_WM, GR_WN>();
constexpr int kGramSplitMax = 32;

int hb2st_init();
int backq2_init();

static void qr_launch_cfg(cudaLaunchConfig_t &cfg, cudaLaunchAttribute *at, cudaStream_t st) {
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3(kQrCl); cfg.blockDim = dim3(kQrThreads); cfg.dynamicSmemBytes = QrSmem::total; cfg.stream = st;
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = kQrCl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
}

int twostage_init() {
    int dev = 0;
    cudaGetDevice(&dev);
    if (g_ts_init_dev == dev) return 0;
    g_ts_ok = 0;
    if (cudaFuncSetAttribute(he2hb_hemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemHemm) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(he2hb_gram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemGram) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(he2hb_x_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemHemm) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(he2hb_her2k_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemH2F) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(he2hb_her2k_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemH2Fs) != cudaSuccess) return HPSD_ECUDA_;
    int rc = hb2st_init();
    if (rc) return rc;
    rc = backq2_init();
    if (rc) return rc;
    if (cudaFuncSetAttribute(he2hb_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)QrSmem::total) == cudaSuccess &&
        cudaFuncSetAttribute(he2hb_panel_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
        cudaLaunchConfig_t cfg; cudaLaunchAttribute at[1];
        qr_launch_cfg(cfg, at, nullptr);
        int nclusters = 0;
        if (cudaOccupancyMaxActiveClusters(&nclusters, he2hb_panel_kernel, &cfg) == cudaSuccess && nclusters >= 1) g_ts_ok = 1;
    }
    cudaGetLastError();            // a device without 16-CTA clusters is not an error: the one-stage path serves it
    g_ts_init_dev = dev;
    return 0;
}

int twostage_available() {
    if (twostage_init()) return 0;
    return g_ts_ok;
}

// Look-ahead: the panel QR (one cluster, ~115 us, latency-bound) of panel k+1 runs on a side stream next to the bulk of panel
// k's HER2K (all SMs, DMMA-bound): the HER2K is split into the first block column of the trailing matrix (all the next
// panel reads) and the rest.  Fork/join with events, so the whole thing stays capturable in a CUDA graph.
struct LookAhead {
    cudaStream_t st = nullptr;
    cudaEvent_t col = nullptr, qr = nullptr;
    int dev = -1;
};
static thread_local LookAhead g_la;
int g_he2hb_lookahead = 1;

static bool lookahead_ready() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    if (g_la.st && g_la.dev == dev) return true;
    if (g_la.st) { cudaStreamDestroy(g_la.st); cudaEventDestroy(g_la.col); cudaEventDestroy(g_la.qr); g_la = LookAhead(); }
    if (cudaStreamCreateWithFlags(&g_la.st, cudaStreamNonBlocking) != cudaSuccess) { g_la = LookAhead(); cudaGetLastError(); return false; }
    if (cudaEventCreateWithFlags(&g_la.col, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&g_la.qr, cudaEventDisableTiming) != cudaSuccess) {
        cudaStreamDestroy(g_la.st); g_la = LookAhead(); cudaGetLastError(); return false;
    }
    g_la.dev = dev;
    return true;
}

static int launch_panel_qr(const TwoStageWs &w, int j0, int kp, cudaStream_t st) {
    QrArgs a{w.n, w.lda, w.ldv, w.ldab, j0, w.A, w.V1, w.tau1, w.Tk + (size_t)kp * kBW * kBW, w.AB};
    cudaLaunchConfig_t cfg; cudaLaunchAttribute at[1];
    qr_launch_cfg(cfg, at, st);
    prof_begin(ST_PANEL, st);
    const cudaError_t e = cudaLaunchKernelEx(&cfg, he2hb_panel_kernel, a);
    prof_end(ST_PANEL, st);
    g_launches++;
    return e == cudaSuccess ? 0 : HPSD_ECUDA_;
}

// C (lower tiles, mirrored) -= X V^H + V X^H  for the M x N leading part of the trailing matrix at C
static int launch_her2k_part(const TwoStageWs &w, const cplx *X, const cplx *V, cplx *C, int M, int N, cudaStream_t st) {
    GemmProblem<cplx, cplx> gp;
    gp.A = X; gp.lda = w.ldz2; gp.B = V; gp.ldb = w.ldv;
    gp.A2 = V; gp.lda2 = w.ldv; gp.B2 = X; gp.ldb2 = w.ldz2;
    gp.M = M; gp.N = N; gp.K = kBW; gp.K2 = kBW;
    Her2kFullEpi epi{C, w.lda};
    if (M <= 1536 || N <= 32) {
        he2hb_her2k_small_kernel<<<dim3((M + 31) / 32, (N + 31) / 32), H2F_WM * H2F_WN * 32, kSmemH2Fs, st>>>(gp, epi);
    } else {
        he2hb_her2k_kernel<<<dim3((M + 63) / 64, (N + 63) / 64), H2F_WM * H2F_WN * 32, kSmemH2F, st>>>(gp, epi);
    }
    HPSD_LAUNCH_CHECK();
    return 0;
}

int launch_he2hb(const TwoStageWs &w, cudaStream_t st) {
    const int n = w.n;
    int rc = twostage_init();
    if (rc) return rc;
    if (!g_ts_ok) return HPSD_ECUDA_;
    if ((n - 2 * kBW + kQrCl - 1) / kQrCl > kQrRows) return HPSD_ECUDA_;      // rows of the first panel exceed the cluster's shared memory
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    HPSD_CUDA_OK(cudaMemsetAsync(w.V1, 0, sizeof(cplx) * (size_t)w.ldv * n, st));
    HPSD_CUDA_OK(cudaMemsetAsync(w.AB, 0, sizeof(cplx) * (size_t)w.ldab * n, st));
    HPSD_CUDA_OK(cudaMemsetAsync(w.tau1, 0, sizeof(cplx) * (size_t)n, st));
    const bool la = g_he2hb_lookahead && lookahead_ready();
    bool qr_on_side = false;          // the QR of the current panel was launched on the side stream by the previous iteration
    int kp = 0;
    for (int j0 = 0; j0 < n; j0 += kBW, ++kp) {
        const int m = n - j0 - kBW;
        if (m <= 0) {
            he2hb_tail_kernel<<<1, 256, 0, st>>>(n, j0, w.A, w.lda, w.AB, w.ldab);
            HPSD_LAUNCH_CHECK();
            break;
        }
        const cplx *Tk = w.Tk + (size_t)kp * kBW * kBW;
        const cplx *V = w.V1 + (size_t)j0 * w.ldv + j0 + kBW;
        cplx *A22 = w.A + (size_t)(j0 + kBW) * w.lda + j0 + kBW;
        if (qr_on_side) {
            if (cudaStreamWaitEvent(st, g_la.qr, 0) != cudaSuccess) return HPSD_ECUDA_;      // join: V, T of this panel are ready
        } else {
            rc = launch_panel_qr(w, j0, kp, st);
            if (rc) return rc;
        }
        qr_on_side = false;
        prof_begin(ST_HER2K, st);
        const int mt = (m + 63) / 64;
        int splits = (2 * sms + mt - 1) / mt;
        if (splits > kHemmSplitMax) splits = kHemmSplitMax;
        int chunk = (((m + splits - 1) / splits) + 15) & ~15;
        splits = (m + chunk - 1) / chunk;
        HemmArgs h{m, w.lda, w.ldv, w.ldz2, chunk, A22, V, w.Zp};
        he2hb_hemm_kernel<<<dim3(mt, splits), HM_THREADS, kSmemHemm, st>>>(h);
        HPSD_LAUNCH_CHECK();
        int gsplit = (m + 255) / 256; if (gsplit > kGramSplitMax) gsplit = kGramSplitMax;
        const int gchunk = (((m + gsplit - 1) / gsplit) + 15) & ~15;
        gsplit = (m + gchunk - 1) / gchunk;
        SlabArgs s{m, w.ldv, w.ldz2, splits, gsplit, V, w.Zp, Tk, w.Z, w.Gp, w.S, w.counter};
        he2hb_zsum_kernel<<<(m * kBW + 255) / 256, 256, 0, st>>>(s);
        HPSD_LAUNCH_CHECK();
        he2hb_gram_kernel<<<gsplit, GR_WM * GR_WN * 32, kSmemGram, st>>>(s, gchunk);
        HPSD_LAUNCH_CHECK();
        he2hb_s_kernel<<<1, kBW * kBW, 0, st>>>(s);
        HPSD_LAUNCH_CHECK();
        XArgs x{m, w.ldv, w.ldz2, w.Z, V, Tk, w.S, w.X};
        he2hb_x_kernel<<<mt, HM_THREADS, kSmemHemm, st>>>(x);
        HPSD_LAUNCH_CHECK();
        const int m_next = m - kBW;               // rows of the next panel
        if (la && m_next > 0 && m > 512) {
            // first block column (all the next panel's QR reads), then fork the QR, then the rest of the trailing matrix
            rc = launch_her2k_part(w, w.X, V, A22, m, kBW, st);
            if (rc) return rc;
            if (cudaEventRecord(g_la.col, st) != cudaSuccess || cudaStreamWaitEvent(g_la.st, g_la.col, 0) != cudaSuccess) return HPSD_ECUDA_;
            rc = launch_panel_qr(w, j0 + kBW, kp + 1, g_la.st);
            const bool rec = cudaEventRecord(g_la.qr, g_la.st) == cudaSuccess;
            qr_on_side = true;
            int rc2 = launch_her2k_part(w, w.X + kBW, V + kBW, A22 + (size_t)kBW * w.lda + kBW, m_next, m_next, st);
            if (rc || !rec || rc2) {              // never leave a capture forked
                cudaStreamWaitEvent(st, g_la.qr, 0);
                return rc ? rc : (rc2 ? rc2 : HPSD_ECUDA_);
            }
        } else {
            rc = launch_her2k_part(w, w.X, V, A22, m, m, st);
            if (rc) return rc;
        }
        prof_end(ST_HER2K, st);
    }
    return 0;
}

}  // namespace hpsd
