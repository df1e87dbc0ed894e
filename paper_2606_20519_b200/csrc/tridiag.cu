// tridiag.cu -- S2+S3 of SURVEY.md §8(a): Hermitian dense -> REAL symmetric tridiagonal,
// A = Q T Q^H with Q = H_0 H_1 ... H_{n-2}, H_c = I - tau_c v_c v_c^H (complex tau, real beta,
// so T's sub-diagonal is real without a separate phase pass).  "Eigendecomposition" of
// PAPER.md:1536 starts here; the paper names no kernel (library call), the design is ours.
//
// One-stage blocked reduction (see DESIGN.md for why not dense->band->tridiagonal on B200):
//   * panel of NB columns in ONE persistent cooperative kernel, two grid barriers per column.
//     Per column: Hermitian mat-vec y = A22 v over the stored lower triangle (the HBM/L2-bound
//     half of the flops), rank-2NB corrections from the panel (V, W), next-column update.
//   * trailing update A22 -= V W^H + W V^H after each panel as a DMMA HER2K (gemm.cuh).
//
// Storage: lower triangle of A (column-major, lda).  After the reduction column c holds the
// full reflector v_c in rows c+1.. (leading 1 stored explicitly at A[c+1,c]); d, e, tau are
// separate arrays.
#include <cooperative_groups.h>
#include "kernels.h"
#include "gemm.cuh"
#include "large.h"
#include "prof.h"

namespace cg = cooperative_groups;

namespace hpsd {

constexpr int kPanelThreads = 256;

struct PanelArgs {
    int n, lda, ldw, ldp, j0, nbp, ts, nblk, G;
    cplx *A, *W;            // W: ldw x NB panel workspace
    double *d, *e;
    cplx *tau;
    cplx *PR, *PC;          // nblk x ldp partial mat-vec results (row parts / column parts)
    cplx *part;             // G x (2*kNB + 1): per-CTA partials [S | gV[NB] | gW[NB]]
    cplx *tot;              // 2*kNB: cV | cW
    double *qpart;          // G
    const int2 *tiles;      // lower-triangle tile list, tile column descending
};

__device__ __forceinline__ cplx group8_sum(cplx v) {
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
    }
    return v;
}

// Householder scalars of column c from alpha = a[c+1] and xnorm2 = ||a[c+2:]||^2 (zlarfg semantics)
__device__ __forceinline__ void householder_scalars(cplx alpha, double xnorm2, double &beta, cplx &tau, cplx &scale) {
    if (xnorm2 == 0.0 && alpha.y == 0.0) {
        beta = alpha.x; tau = mk(0.0, 0.0); scale = mk(0.0, 0.0);
    } else {
        const double nrm = sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xnorm2);
        beta = -copysign(nrm, alpha.x);
        tau = mk((beta - alpha.x) / beta, -alpha.y / beta);
        const cplx den = mk(alpha.x - beta, alpha.y);
        const double d2 = abs2(den);
        scale = mk(den.x / d2, -den.y / d2);
    }
}

// Column preparation: apply the panel's first `cnt` reflector pairs (V, W) to column cn (rows >= cn),
// store it, set d[cn], and leave per-CTA partials  S = sum_{r>=cn+2}|a_r|^2,
// gV[t] = sum_{r>=cn+2} conj(V[r,t]) a_r, gW[t] likewise.  `have_new`: reflector cnt-1 lives in
// registers of the caller (v_r, w_r) -- not used here; this variant reads everything from memory and
// is only used at panel start (cnt = 0).
template <int TS>
__device__ void panel_body(const PanelArgs &p) {
    cg::grid_group grid = cg::this_grid();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // shared layout
    cplx *s_vI = reinterpret_cast<cplx *>(smem_raw);          // TS
    cplx *s_vJ = s_vI + TS;                                    // TS
    cplx *s_row = s_vJ + TS;                                   // 8 x TS
    cplx *s_col = s_row + 8 * TS;                              // TS
    cplx *s_cV = s_col + TS;                                   // kNB
    cplx *s_cW = s_cV + kNB;                                   // kNB
    cplx *s_Vc1 = s_cW + kNB;                                  // kNB : V[c+1, t]
    cplx *s_Wc1 = s_Vc1 + kNB;                                 // kNB : W[c+1, t]
    cplx *s_gV = s_Wc1 + kNB;                                  // 32 x kNB
    cplx *s_gW = s_gV + 32 * kNB;                              // 32 x kNB
    double *s_S = reinterpret_cast<double *>(s_gW + 32 * kNB); // 32
    double *s_q = s_S + 32;                                    // 8
    cplx *s_sc = reinterpret_cast<cplx *>(s_q + 8);            // scalars: [0]=tau [1]=scale [2]=(beta, alpha') [3]=w_{c+1}

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = blockIdx.x, G = p.G;
    const int n = p.n, lda = p.lda, ldw = p.ldw, ldp = p.ldp;
    cplx *A = p.A, *W = p.W;
    const int grp = tid >> 3, gl = tid & 7;          // 32 row groups of 8 lanes
    const int PSTRIDE = 2 * kNB + 1;

    // ---------------- panel start: partial norm of column j0 (already fully updated) -----
    {
        const int cn = p.j0;
        const int rows = n - cn;                     // rows cn .. n-1
        const int L = (rows + G - 1) / G;
        double S = 0.0;
        for (int rr = grp; rr < L; rr += 32) {
            const int r = cn + g * L + rr;
            if (r < n && gl == 0) {
                if (r == cn) {
                    cplx a = A[(size_t)cn * lda + r];
                    p.d[cn] = a.x;
                } else if (r >= cn + 2) {
                    S += abs2(A[(size_t)cn * lda + r]);
                }
            }
        }
        if (gl == 0) s_S[grp] = S;
        __syncthreads();
        if (tid == 0) {
            double t = 0.0;
            for (int k = 0; k < 32; ++k) t += s_S[k];
            p.part[(size_t)g * PSTRIDE] = mk(t, 0.0);
        }
    }
    grid.sync();

    for (int i = 0; i < p.nbp; ++i) {
        const int c = p.j0 + i;
        if (c >= n - 1) break;
        // ================= phase A =================
        // (a) Householder scalars, redundantly and identically in every CTA
        if (warp == 0) {
            double S = 0.0;
            for (int k = lane; k < G; k += 32) S += ldcg_(&p.part[(size_t)k * PSTRIDE].x);
            S = warp_sum(S);
            if (lane == 0) {
                const cplx alpha = ldcg_(&A[(size_t)c * lda + c + 1]);
                double beta; cplx tau, scale;
                householder_scalars(alpha, S, beta, tau, scale);
                s_sc[0] = tau; s_sc[1] = scale; s_sc[2] = mk(beta, 0.0);
                if (g == 0) { p.e[c] = beta; p.tau[c] = tau; }
            }
        }
        __syncthreads();
        const cplx tau = s_sc[0], scale = s_sc[1];

        // (b) reducer CTA: cV = V22^H v, cW = W22^H v  (rows >= c+1) from the per-CTA partials
        if (g == G - 1 && i > 0) {
            // thread -> (slice = tid/64, which = (tid/32)&1, t = tid%32)
            const int t = tid & 31, which = (tid >> 5) & 1, slice = tid >> 6;
            cplx acc = mk(0.0, 0.0);
            if (t < i) {
                for (int k = slice; k < G; k += 4) {
                    const cplx v = ldcg_(&p.part[(size_t)k * PSTRIDE + 1 + which * kNB + t]);
                    acc = acc + v;
                }
            }
            s_gV[(slice * 2 + which) * kNB + t] = acc;
            __syncthreads();
            if (tid < 64 && t < i) {
                cplx s = (s_gV[(0 * 2 + which) * kNB + t] + s_gV[(1 * 2 + which) * kNB + t]) +
                         (s_gV[(2 * 2 + which) * kNB + t] + s_gV[(3 * 2 + which) * kNB + t]);
                // row c+1 term (v = 1 there) plus scale * sum over rows >= c+2
                const cplx top = which == 0 ? ldcg_(&A[(size_t)(p.j0 + t) * lda + c + 1]) : ldcg_(&W[(size_t)t * ldw + c + 1]);
                s = conj_(top) + scale * s;
                p.tot[which * kNB + t] = s;
            }
            __syncthreads();
        }

        // (c) Hermitian mat-vec partials over the lower-triangle tiles of A[c+1:, c+1:]
        {
            const int J0 = (c + 1) / TS;
            const int nbk = p.nblk - J0;
            const int T = nbk * (nbk + 1) / 2;
            double qacc = 0.0;          // thread 0 only
            constexpr int RH = TS / 32, CPW = TS / 8;
            for (int idx = g; idx < T; idx += G) {
                const int2 ij = p.tiles[idx];
                const int I = ij.x, J = ij.y;
                const int r0 = I * TS, c0 = J * TS;
                __syncthreads();
                // vector pieces (v formed on the fly; zero outside the trailing matrix)
                for (int k = tid; k < 2 * TS; k += kPanelThreads) {
                    const int r = (k < TS) ? r0 + k : c0 + (k - TS);
                    cplx v = mk(0.0, 0.0);
                    if (r < n) {
                        if (r == c + 1) v = mk(1.0, 0.0);
                        else if (r > c + 1) v = scale * ldcg_(&A[(size_t)c * lda + r]);
                    }
                    if (k < TS) s_vI[k] = v; else s_vJ[k - TS] = v;
                }
                __syncthreads();
                cplx accR[RH];
#pragma unroll
                for (int h = 0; h < RH; ++h) accR[h] = mk(0.0, 0.0);
                const bool diag = (I == J);
                // issue all loads first (ILP), then consume
                cplx a[CPW][RH];
#pragma unroll
                for (int cc = 0; cc < CPW; ++cc) {
                    const int col = c0 + warp + 8 * cc;
#pragma unroll
                    for (int h = 0; h < RH; ++h) {
                        const int r = r0 + lane + 32 * h;
                        const bool ok = (r < n) && (col < n) && (!diag || r >= col);
                        a[cc][h] = ok ? A[(size_t)col * lda + r] : mk(0.0, 0.0);
                        if (diag && r == col) a[cc][h].y = 0.0;
                    }
                }
#pragma unroll
                for (int cc = 0; cc < CPW; ++cc) {
                    const int cl = warp + 8 * cc;
                    const cplx vj = s_vJ[cl];
                    cplx colacc = mk(0.0, 0.0);
#pragma unroll
                    for (int h = 0; h < RH; ++h) {
                        const int rl = lane + 32 * h;
                        cfma(accR[h], a[cc][h], vj);
                        // column part: conj(a) * v_I[r]; on the diagonal tile skip r == col (counted in the row part)
                        if (!(diag && rl == cl)) cfma_conj(colacc, a[cc][h], s_vI[rl]);
                    }
                    colacc = warp_sum(colacc);
                    if (lane == 0) s_col[cl] = colacc;
                }
#pragma unroll
                for (int h = 0; h < RH; ++h) s_row[warp * TS + lane + 32 * h] = accR[h];
                __syncthreads();
                if (tid < TS) {
                    cplx s = mk(0.0, 0.0);
#pragma unroll
                    for (int w = 0; w < 8; ++w) s = s + s_row[w * TS + tid];
                    double qterm;
                    if (diag) {
                        s = s + s_col[tid];
                        p.PR[(size_t)J * ldp + r0 + tid] = s;
                        qterm = s_vI[tid].x * s.x + s_vI[tid].y * s.y;
                    } else {
                        p.PR[(size_t)J * ldp + r0 + tid] = s;
                        p.PC[(size_t)I * ldp + c0 + tid] = s_col[tid];
                        qterm = 2.0 * (s_vI[tid].x * s.x + s_vI[tid].y * s.y);
                    }
                    qterm = warp_sum(qterm);
                    if (lane == 0) s_q[warp] = qterm;
                }
                __syncthreads();
                if (tid == 0) {
                    for (int w = 0; w < TS / 32; ++w) qacc += s_q[w];
                }
            }
            if (tid == 0) p.qpart[g] = qacc;
        }
        grid.sync();

        // ================= phase B =================
        {
            const bool do_next = (i + 1 < p.nbp);
            if (tid < kNB) {
                cplx cv = mk(0.0, 0.0), cw = mk(0.0, 0.0), v1 = mk(0.0, 0.0), w1 = mk(0.0, 0.0);
                if (tid < i) {
                    cv = ldcg_(&p.tot[tid]);
                    cw = ldcg_(&p.tot[kNB + tid]);
                    // row c+1 of V and W (needed for the next-column update)
                    v1 = ldcg_(&A[(size_t)(p.j0 + tid) * lda + c + 1]);
                    w1 = ldcg_(&W[(size_t)tid * ldw + c + 1]);
                }
                s_cV[tid] = cv; s_cW[tid] = cw; s_Vc1[tid] = v1; s_Wc1[tid] = w1;
            }
            if (warp == 1) {
                double q = 0.0;
                for (int k = lane; k < G; k += 32) q += ldcg_(&p.qpart[k]);
                q = warp_sum(q);
                if (lane == 0) s_q[0] = q;
            }
            __syncthreads();
            if (tid == 0) {
                double re = 0.0;   // Re(cV^H cW)
                for (int t = 0; t < i; ++t) re += s_cV[t].x * s_cW[t].x + s_cV[t].y * s_cW[t].y;
                const double vHy = s_q[0] - 2.0 * re;
                s_sc[2].y = -0.5 * abs2(tau) * vHy;   // alpha'
            }
            __syncthreads();
            const double alphap = s_sc[2].y;

            const int J0 = (c + 1) / TS;
            // y of one row from the tile partials + panel corrections; all 8 lanes get the result
            // (every lane of the warp must call this: it shuffles with a full mask; `ok` predicates loads)
            auto row_yw = [&](bool ok, int r, cplx vr, cplx (&Vr)[kNB / 8], cplx (&Wr)[kNB / 8]) -> cplx {
                const int R = r / TS;
                cplx ys = mk(0.0, 0.0);
                if (ok) {
                    for (int b = J0 + gl; b < p.nblk; b += 8) {
                        const cplx v = (b <= R) ? ldcg_(&p.PR[(size_t)b * ldp + r]) : ldcg_(&p.PC[(size_t)b * ldp + r]);
                        ys = ys + v;
                    }
                }
                cplx corr = mk(0.0, 0.0);
#pragma unroll
                for (int k = 0; k < kNB / 8; ++k) {
                    const int t = gl + 8 * k;
                    if (ok && t < i) {
                        Vr[k] = ldcg_(&A[(size_t)(p.j0 + t) * lda + r]);
                        Wr[k] = ldcg_(&W[(size_t)t * ldw + r]);
                        cfma(corr, Vr[k], s_cW[t]);
                        cfma(corr, Wr[k], s_cV[t]);
                    } else { Vr[k] = mk(0.0, 0.0); Wr[k] = mk(0.0, 0.0); }
                }
                ys = group8_sum(ys - corr);
                return tau * ys + alphap * vr;
            };

            // w_{c+1} (row c+1 of the new W column), needed by every CTA for the next-column update
            if (do_next) {
                if (warp == 0) {   // all four 8-lane groups of warp 0 compute the same value
                    cplx Vr[kNB / 8], Wr[kNB / 8];
                    const cplx w = row_yw(true, c + 1, mk(1.0, 0.0), Vr, Wr);
                    if (lane == 0) s_sc[3] = w;
                }
                __syncthreads();
            }
            const cplx wc1 = s_sc[3];

            const int rows = n - (c + 1);
            const int L = (rows + G - 1) / G;
            cplx accV[kNB / 8], accW[kNB / 8];
#pragma unroll
            for (int k = 0; k < kNB / 8; ++k) { accV[k] = mk(0.0, 0.0); accW[k] = mk(0.0, 0.0); }
            double S = 0.0;
            for (int base = 0; base < L; base += 32) {      // warp-uniform trip count
                const int rr = base + grp;
                const int r = c + 1 + g * L + rr;
                const bool ok = (rr < L) && (r < n);
                const cplx ar = ok ? ldcg_(&A[(size_t)c * lda + r]) : mk(0.0, 0.0);
                const cplx vr = (r == c + 1) ? mk(1.0, 0.0) : scale * ar;
                cplx Vr[kNB / 8], Wr[kNB / 8];
                const cplx wr = row_yw(ok, r, vr, Vr, Wr);
                if (ok && gl == 0) {
                    W[(size_t)i * ldw + r] = wr;
                    A[(size_t)c * lda + r] = vr;
                }
                if (do_next) {
                    // a'_r = A[r,c+1] - sum_{t<=i} V[r,t] conj(W[c+1,t]) + W[r,t] conj(V[c+1,t])
                    cplx upd = mk(0.0, 0.0);
#pragma unroll
                    for (int k = 0; k < kNB / 8; ++k) {
                        const int t = gl + 8 * k;
                        if (t < i) {
                            cfma(upd, Vr[k], conj_(s_Wc1[t]));
                            cfma(upd, Wr[k], conj_(s_Vc1[t]));
                        }
                    }
                    upd = group8_sum(upd);
                    cfma(upd, vr, conj_(wc1));
                    upd = upd + wr;                   // V[c+1, i] = 1
                    cplx an = (ok ? ldcg_(&A[(size_t)(c + 1) * lda + r]) : mk(0.0, 0.0)) - upd;
                    if (ok && r == c + 1) { an.y = 0.0; if (gl == 0) p.d[c + 1] = an.x; }
                    if (ok && gl == 0) A[(size_t)(c + 1) * lda + r] = an;
                    if (ok && r >= c + 3) {
                        if (gl == 0) S += abs2(an);
#pragma unroll
                        for (int k = 0; k < kNB / 8; ++k) {
                            const int t = gl + 8 * k;
                            if (t < i) { cfma_conj(accV[k], Vr[k], an); cfma_conj(accW[k], Wr[k], an); }
                            else if (t == i) { cfma_conj(accV[k], vr, an); cfma_conj(accW[k], wr, an); }
                        }
                    }
                }
            }
            if (do_next) {
#pragma unroll
                for (int k = 0; k < kNB / 8; ++k) {
                    s_gV[grp * kNB + gl + 8 * k] = accV[k];
                    s_gW[grp * kNB + gl + 8 * k] = accW[k];
                }
                if (gl == 0) s_S[grp] = S;
                __syncthreads();
                if (tid < 2 * kNB) {
                    const int t = tid % kNB;
                    const cplx *src = (tid < kNB) ? s_gV : s_gW;
                    cplx s = mk(0.0, 0.0);
                    for (int k = 0; k < 32; ++k) s = s + src[k * kNB + t];
                    p.part[(size_t)g * PSTRIDE + 1 + tid] = s;
                } else if (tid == 2 * kNB) {
                    double t = 0.0;
                    for (int k = 0; k < 32; ++k) t += s_S[k];
                    p.part[(size_t)g * PSTRIDE] = mk(t, 0.0);
                }
            }
        }
        if (i + 1 < p.nbp) grid.sync();
    }
}

template <int TS>
__global__ void __launch_bounds__(kPanelThreads, 1) tridiag_panel_kernel(PanelArgs p) { panel_body<TS>(p); }

static size_t panel_smem_bytes(int ts) {
    return sizeof(cplx) * (size_t)(2 * ts + 8 * ts + ts + 4 * kNB + 64 * kNB + 4) + sizeof(double) * 40;
}

// ---------------------------------------------------------------- HER2K (DMMA)
struct Her2kEpi {
    cplx *C; int ldc;
    __device__ __forceinline__ void operator()(int i, int j, double re, double im) const {
        cplx *c = C + (size_t)j * ldc + i;
        cplx v = *c;
        v.x -= re; v.y -= im;
        if (i == j) v.y = 0.0;
        *c = v;
    }
};

constexpr int H2_MI = 4, H2_NI = 4, H2_WM = 2, H2_WN = 2;   // 64 x 64 CTA tile, 4 warps

__global__ void __launch_bounds__(H2_WM *H2_WN * 32) her2k_kernel(GemmProblem<cplx, cplx> p, Her2kEpi epi) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (blockIdx.y > blockIdx.x) return;   // lower triangle of tiles only
    gemm_tile_body<cplx, cplx, MNMAJ, MNMAJ, false, true, H2_MI, H2_NI, H2_WM, H2_WN, true>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
}

// After the reduction: zero the (unused) diagonal and upper part so that V blocks are plain dense
// sub-matrices for the back-transformation (S5).
__global__ void clean_v_kernel(int n, cplx *A, int lda) {
    const int j = blockIdx.y;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= j && i < n; i += gridDim.x * blockDim.x) A[(size_t)j * lda + i] = mk(0.0, 0.0);
}

// ---------------------------------------------------------------- host driver
static int g_panel_init_dev = -1;

int tridiag_init() {
    int dev = 0;
    cudaGetDevice(&dev);
    if (g_panel_init_dev == dev) return 0;
    if (cudaFuncSetAttribute(tridiag_panel_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)panel_smem_bytes(32)) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(tridiag_panel_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)panel_smem_bytes(64)) != cudaSuccess) return HPSD_ECUDA_;
    constexpr size_t h2 = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, H2_MI, H2_NI, H2_WM, H2_WN>();
    if (cudaFuncSetAttribute(her2k_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h2) != cudaSuccess) return HPSD_ECUDA_;
    g_panel_init_dev = dev;
    return 0;
}

int tridiag_tile_size(int n) { return n >= 1536 ? 64 : 32; }

size_t tridiag_tile_count(int n) {
    const int ts = tridiag_tile_size(n);
    const int nblk = (n + ts - 1) / ts;
    return (size_t)nblk * (nblk + 1) / 2;
}

void tridiag_fill_tiles(int n, int2 *tiles) {
    const int ts = tridiag_tile_size(n);
    const int nblk = (n + ts - 1) / ts;
    size_t k = 0;
    for (int J = nblk - 1; J >= 0; --J)
        for (int I = J; I < nblk; ++I) tiles[k++] = make_int2(I, J);
}

int launch_tridiag(const TridiagWs &w, cudaStream_t st) {
    const int n = w.n;
    if (n <= 0) return 0;
    int rc = tridiag_init();
    if (rc) return rc;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int ts = tridiag_tile_size(n);
    PanelArgs p;
    p.n = n; p.lda = w.lda; p.ldw = w.ldw; p.ts = ts; p.nblk = (n + ts - 1) / ts; p.G = sms;
    p.A = w.A; p.W = w.W; p.d = w.d; p.e = w.e; p.tau = w.tau;
    p.ldp = w.ldp; p.PR = w.PR; p.PC = w.PC; p.part = w.part; p.tot = w.tot; p.qpart = w.qpart; p.tiles = w.tiles;
    if (n == 1) {
        // d[0] = Re A[0,0]; handled by a 1-column panel (sets d in the prologue)
    }
    for (int j0 = 0; j0 < n; j0 += kNB) {
        p.j0 = j0;
        p.nbp = (n - j0 < kNB) ? (n - j0) : kNB;
        void *args[] = {&p};
        const size_t smem = panel_smem_bytes(ts);
        cudaError_t e;
        prof_begin(ST_PANEL, st);
        if (ts == 64) e = cudaLaunchCooperativeKernel((void *)tridiag_panel_kernel<64>, dim3(p.G), dim3(kPanelThreads), args, smem, st);
        else e = cudaLaunchCooperativeKernel((void *)tridiag_panel_kernel<32>, dim3(p.G), dim3(kPanelThreads), args, smem, st);
        prof_end(ST_PANEL, st);
        g_launches++;
        if (e != cudaSuccess) return HPSD_ECUDA_;
        const int m2 = n - (j0 + kNB);
        if (m2 > 0) {
            GemmProblem<cplx, cplx> gp;
            const cplx *V = w.A + (size_t)j0 * w.lda + (j0 + kNB);
            const cplx *Wp = w.W + (j0 + kNB);
            gp.A = V; gp.lda = w.lda; gp.B = Wp; gp.ldb = w.ldw;
            gp.A2 = Wp; gp.lda2 = w.ldw; gp.B2 = V; gp.ldb2 = w.lda;
            gp.M = m2; gp.N = m2; gp.K = kNB; gp.K2 = kNB;
            Her2kEpi epi{w.A + (size_t)(j0 + kNB) * w.lda + (j0 + kNB), w.lda};
            const int nt = (m2 + 63) / 64;
            constexpr size_t h2 = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, H2_MI, H2_NI, H2_WM, H2_WN>();
            prof_begin(ST_HER2K, st);
            her2k_kernel<<<dim3(nt, nt), H2_WM * H2_WN * 32, h2, st>>>(gp, epi);
            prof_end(ST_HER2K, st);
            HPSD_LAUNCH_CHECK();
        }
    }
    if (n > 1) {
        clean_v_kernel<<<dim3((n + 255) / 256, n), 256, 0, st>>>(n, w.A, w.lda);
        HPSD_LAUNCH_CHECK();
    }
    return 0;
}

}  // namespace hpsd
