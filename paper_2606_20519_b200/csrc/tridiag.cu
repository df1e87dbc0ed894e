// tridiag.cu -- S2+S3 of SURVEY.md §8(a): Hermitian dense -> REAL symmetric tridiagonal,
// A = Q T Q^H with Q = H_0 H_1 ... H_{n-2}, H_c = I - tau_c v_c v_c^H (complex tau, real beta,
// so T's sub-diagonal is real without a separate phase pass).  "Eigendecomposition" of
// PAPER.md:1536 starts here; the paper names no kernel (library call), the design is ours.
//
// One-stage blocked reduction (DESIGN.md §7 for why not dense->band->tridiagonal on B200):
//   * panel of NB = 32 columns in ONE persistent cooperative kernel, two grid barriers per column.
//     The trailing matrix is NOT modified inside a panel, so its 32 x 32 tiles are distributed over
//     the shared memory of all SMs ONCE per panel (12 slots of 16.5 KB per CTA: 28 MB over 148 SMs,
//     i.e. trailing sizes up to ~1880 stay resident; larger ones stream through the same slots:
//     each pair of warps runs a ring of three slots filled by 512-byte bulk copies (TMA engine, one
//     mbarrier per slot) that keeps its last tiles across the grid barrier).
//     Phase A (per column): every warp multiplies its own tiles by the Householder vector
//       (y = A22 v, row parts and column parts of the stored lower triangle), no block-level sync.
//     Phase B: rows are spread over the CTAs; y is assembled from the tile partials, w is formed,
//       the next column is updated and its norm / V^H a, W^H a partials are left for phase A.
//     Each phase has ONE dependent L2 round trip.
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
constexpr int kTS = 32;                  // tile edge of the distributed trailing matrix
constexpr int kTP = kTS + 1;             // shared-memory pitch (elements): row- and column-wise reads conflict free
constexpr int kSlots = 12;               // tile slots per CTA
constexpr int kSlotElems = kTS * kTP;
static_assert(kNB == kTS, "panel width and tile edge must agree (tile set is fixed per panel)");

struct PanelArgs {
    int n, lda, ldw, ldp, j0, nbp, nblk, G;
    int T;                  // tiles of this panel's trailing matrix (prefix of `tiles`)
    int q;                  // tiles per CTA = ceil(T / G)
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

// Loads of data another CTA wrote before the last grid barrier.  The barrier's fence invalidates this SM's L1
// (CCTL.IVALL, which is how grid.sync makes ordinary loads safe), so plain loads are correct here, and they are
// much cheaper to issue than ld.global.cg, which ptxas turns into LDG.STRONG.GPU (~170 cycles of issue each).
__device__ __forceinline__ double ldx_(const double *p) { return *p; }
__device__ __forceinline__ cplx ldx_(const cplx *p) { return *p; }

// Householder scalars of column c from alpha = a[c+1] and xnorm2 = ||a[c+2:]||^2 (zlarfg semantics)
__device__ __forceinline__ void householder_scalars(cplx alpha, double xnorm2, double &beta, cplx &tau, cplx &scale) {
    if (xnorm2 == 0.0 && alpha.y == 0.0) {
        beta = alpha.x; tau = mk(0.0, 0.0); scale = mk(0.0, 0.0);
    } else {
        // one reciprocal square root (refined by a Newton step to full accuracy) and one reciprocal on the dependent chain
        // instead of DSQRT + two DDIV (100 + 2 x 132 cycles): warp 0 of EVERY CTA runs this at the head of every column,
        // with all other warps waiting at the block barrier behind it
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

// Phase-B row distribution: 31 rows per CTA (one per 8-lane group; group 31 is the helper), more
// only when the rows outnumber 31 G.  Few producers keep the cross-CTA reductions small.
// (runtime integer divisions are ~100 cycles on the critical path: only taken when the rows outnumber 31 G)
__device__ __forceinline__ int rows_per_cta(int rows, int G) { return rows <= 31 * G ? 31 : (rows + G - 1) / G; }
__device__ __forceinline__ int producers(int rows, int G) {
    const int l = rows_per_cta(rows, G);
    return l == 31 ? (rows + 30) / 31 : (rows + l - 1) / l;
}

// ---- mbarrier / bulk-copy helpers (each tile slot has an mbarrier that one load completes one phase of)
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned mbar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned mbar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned mbar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned mbar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(mbar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}

// One warp copies tile (I, J) of A into a shared-memory slot and completes one phase of the slot's mbarrier.
// Full tiles: one 512-byte bulk copy (TMA engine) per column, issued by lane = column; the LSU path (cp.async, 16 bytes
// per thread) caps the bytes an SM keeps in flight, which is what bounded the streaming regime.  Edge tiles (zero fill
// outside the matrix): cp.async, waited for here.
__device__ __forceinline__ void warp_load_tile(cplx *slot, unsigned mbar, const cplx *__restrict__ A, int lda, int n, int2 ij, int lane) {
    const int r0 = ij.x * kTS, c0 = ij.y * kTS;
    if (r0 + kTS <= n && c0 + kTS <= n) {                  // warp-uniform
        if (lane == 0) mbar_arrive_expect_tx(mbar, kTS * kTS * (unsigned)sizeof(cplx));
        __syncwarp();
        bulk_g2s(smem_u32(slot + lane * kTP), A + (size_t)(c0 + lane) * lda + r0, kTS * (unsigned)sizeof(cplx), mbar);
        return;
    }
    const int r = r0 + lane;
    const bool rok = r < n;
#pragma unroll 8
    for (int cc = 0; cc < kTS; ++cc) {
        const bool ok = rok && (c0 + cc < n);
        cp_async_16(slot + cc * kTP + lane, ok ? A + (size_t)(c0 + cc) * lda + r : A, ok);
    }
    cp_async_commit();
    cp_async_wait<0>();
    __syncwarp();
    if (lane == 0) mbar_arrive(mbar);
}

__global__ void __launch_bounds__(kPanelThreads, 1) tridiag_panel_kernel(PanelArgs p) {
    cg::grid_group grid = cg::this_grid();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *s_slots = reinterpret_cast<cplx *>(smem_raw);        // kSlots x kSlotElems
    cplx *s_v = s_slots + kSlots * kSlotElems;                 // 8 warps x 2 x kTS : v pieces of the tile in flight
    cplx *s_cV = s_v + 8 * 2 * kTS;                            // kNB
    cplx *s_cW = s_cV + kNB;                                   // kNB
    cplx *s_Vc1 = s_cW + kNB;                                  // kNB : V[c+1, t]
    cplx *s_Wc1 = s_Vc1 + kNB;                                 // kNB : W[c+1, t]
    cplx *s_gV = s_Wc1 + kNB;                                  // 8 x kNB
    cplx *s_gW = s_gV + 8 * kNB;                               // 8 x kNB
    cplx *s_sc = s_gW + 8 * kNB;                               // [0]=tau [1]=scale [2]=w_{c+1}
    double *s_S = reinterpret_cast<double *>(s_sc + 4);        // 8
    double *s_q = s_S + 8;                                     // 8 (+1: total)
    const unsigned mbar0 = smem_u32(s_q + 12);                 // kSlots mbarriers (8 bytes each), one per tile slot

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = blockIdx.x, G = p.G;
    const int n = p.n, lda = p.lda, ldw = p.ldw, ldp = p.ldp;
    cplx *A = p.A, *W = p.W;
    constexpr int PSTRIDE = 2 * kNB + 1;
    const int T = p.T, q = p.q;
    const bool streaming = q > kSlots;
    const bool wide = q <= 2;                       // block-uniform

    // ---------------- tile slots: warps p and p + 4 (a pair) share the slots p, p + 4, p + 8 as a ring of three ---------
    // tile k of this CTA is tiles[g + k G]; the pair's tiles are t = 0, 1, 2, ... with k(t) = (t / 3) kSlots + p + 4 (t % 3),
    // tile t lives in slot p + 4 (t % 3).  In pass order (forwards on even, backwards on odd columns) the two warps take
    // alternate positions P = 2 jj + m; whoever finishes position P refills its slot with the tile of position P + 3,
    // which the OTHER warp consumes.  So all eight warps carry the same number of tiles and every load has a whole tile
    // time to arrive (before: warps 0..3 owned two slots and did two thirds of the tiles, warps 4..7 one slot, no prefetch).
    const int pr_p = warp & 3, pr_m = warp >> 2;
    auto kpair = [&](int t) { return (t / 3) * kSlots + pr_p + 4 * (t % 3); };
    volatile int *s_iss = reinterpret_cast<volatile int *>(s_q + 12 + kSlots);     // loads issued so far into each slot
    if (threadIdx.x < kSlots) { mbar_init(mbar0 + 8u * threadIdx.x, 1); s_iss[threadIdx.x] = 1; }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async;" ::: "memory");
    __syncthreads();
    int pcnt = 0;                           // tiles of this pair
    for (int t = 0;; ++t) {
        const int k = kpair(t);
        if (k >= q || g + k * G >= T) break;
        pcnt = t + 1;
    }
    const int cnt = (pcnt + 1 - pr_m) / 2;  // positions of this warp in a pass
    // coordinates of the pair's first three tiles (all of them in the resident regimes), read once
    int2 ijc[3] = {make_int2(0, 0), make_int2(0, 0), make_int2(0, 0)};
    if (wide) { if ((warp >> 2) < q && g + (warp >> 2) * G < T) ijc[0] = p.tiles[g + (warp >> 2) * G]; }
    else {
#pragma unroll
        for (int t = 0; t < 3; ++t) if (t < pcnt) ijc[t] = p.tiles[g + kpair(t) * G];
    }
    if (wide) {           // slots 0 and 1 (tiles 0 and 1), loaded by warps 0 and 1, read by four warps each
        if (warp < 2 && warp < q && g + warp * G < T) warp_load_tile(s_slots + (size_t)warp * kSlotElems, mbar0 + 8u * warp, A, lda, n, p.tiles[g + warp * G], lane);
    } else {
#pragma unroll
        for (int t = 0; t < 3; ++t)
            if (t < pcnt && (t & 1) == pr_m)
                warp_load_tile(s_slots + (size_t)(pr_p + 4 * t) * kSlotElems, mbar0 + 8u * (pr_p + 4 * t), A, lda, n, ijc[t], lane);
    }
    unsigned base0 = 1u, base1 = 1u, base2 = 1u;     // loads issued into the pair's three slots before the current pass

    // ---------------- panel start: d[j0] and the partial norm of column j0 (already fully updated) -----
    {
        const int cn = p.j0;
        const int rows = n - cn;
        const int L = rows_per_cta(rows, G);
        double S = 0.0;
        for (int rr = tid; rr < L; rr += kPanelThreads) {
            const int r = cn + g * L + rr;
            if (r < n) {
                if (r == cn) p.d[cn] = A[(size_t)cn * lda + r].x;
                else if (r >= cn + 2) S += abs2(A[(size_t)cn * lda + r]);
            }
        }
        S = warp_sum(S);
        if (lane == 0) s_S[warp] = S;
        __syncthreads();
        if (tid == 0) {
            double t = 0.0;
            for (int k = 0; k < 8; ++k) t += s_S[k];
            p.part[(size_t)g * PSTRIDE] = mk(t, 0.0);
        }
    }
    // wide mode: the slots are read by other warps; every reader waits for its slot's (only) load itself
    if (wide && (warp >> 2) < q && g + (warp >> 2) * G < T) mbar_wait(mbar0 + 8u * (warp >> 2), 0u);
    grid.sync();

    for (int i = 0; i < p.nbp; ++i) {
        const int c = p.j0 + i;
        if (c >= n - 1) break;
        // ================= phase A: y = A22 v over this CTA's tiles (no block-level sync) =================
        // raw pieces of column c for this warp's first tiles: issued before anything that waits
        // Tiles are walked forwards on even columns and backwards on odd ones: when they stream, the tail
        // of one pass is the head of the next, so it is still in the slots / in L2.
        const bool fwd = (i & 1) == 0;
        // wide mode (at most two tiles per CTA): four warps share a tile, eight columns each
        const int wtile = warp >> 2, wq = warp & 3;
        const bool wvalid = wide && wtile < q && g + wtile * G < T;
        // coordinates of this warp's tile number jj of the pass (pass order: forwards or backwards through its sequence)
        auto pos_tile = [&](int P) -> int2 {          // tile of the pair at position P of this pass
            const int t = fwd ? P : pcnt - 1 - P;
            return (t == 0) ? ijc[0] : (t == 1) ? ijc[1] : (t == 2) ? ijc[2] : p.tiles[g + kpair(t) * G];
        };
        auto tile_of = [&](int jj) -> int2 { return pos_tile(2 * jj + pr_m); };
        cplx rawI[2], rawJ[2];
        int2 ijq[3] = {make_int2(0, 0), make_int2(0, 0), make_int2(0, 0)};     // coordinates of tiles jj, jj + 1, jj + 2
#pragma unroll
        for (int jj = 0; jj < 2; ++jj) {
            rawI[jj] = mk(0.0, 0.0); rawJ[jj] = mk(0.0, 0.0);
            if (wide) {
                if (jj == 0 && wvalid) {
                    const int2 ij = ijc[0];
                    const int rI = ij.x * kTS + lane, rJ = ij.y * kTS + lane;
                    if (rI < n && rI > c + 1) rawI[0] = ldx_(&A[(size_t)c * lda + rI]);
                    if (ij.x != ij.y && rJ < n && rJ > c + 1) rawJ[0] = ldx_(&A[(size_t)c * lda + rJ]);
                }
            } else if (jj < cnt) {
                const int2 ij = tile_of(jj);
                ijq[jj] = ij;
                const int rI = ij.x * kTS + lane, rJ = ij.y * kTS + lane;
                if (rI < n && rI > c + 1) rawI[jj] = ldx_(&A[(size_t)c * lda + rI]);
                if (ij.x != ij.y && rJ < n && rJ > c + 1) rawJ[jj] = ldx_(&A[(size_t)c * lda + rJ]);
            }
        }
        if (!wide && cnt > 2) ijq[2] = tile_of(2);
        int2 ijr = make_int2(0, 0);                 // coordinates of the tile this warp loads after its next tile
        if (streaming && pr_m + 3 < pcnt) ijr = pos_tile(pr_m + 3);
        const int nprod = producers(n - c, G);          // CTAs that left partials for this column
        // warp 0: Householder scalars from the partial norms
        if (warp == 0) {
            // five independent loads in flight (a load -> add -> load loop costs one L2 round trip per 32 producers)
            double Sp[5];
#pragma unroll
            for (int u = 0; u < 5; ++u) { const int k = lane + 32 * u; Sp[u] = (k < nprod) ? ldx_(&p.part[(size_t)k * PSTRIDE].x) : 0.0; }
            const cplx alpha = ldx_(&A[(size_t)c * lda + c + 1]);
            double S = ((Sp[0] + Sp[1]) + (Sp[2] + Sp[3])) + Sp[4];
            for (int k = lane + 160; k < nprod; k += 32) S += ldx_(&p.part[(size_t)k * PSTRIDE].x);
            S = warp_sum(S);
            double beta; cplx tau0, scale0;
            householder_scalars(alpha, S, beta, tau0, scale0);
            if (lane == 0) {
                s_sc[0] = tau0; s_sc[1] = scale0;
                if (g == 0) { p.e[c] = beta; p.tau[c] = tau0; }
            }
        }
        // warp 7 of CTA idx < 64: reducers cV[t] = (V22^H v)_t, cW[t] = (W22^H v)_t (rows >= c+1)
        cplx red_s = mk(0.0, 0.0), red_top = mk(0.0, 0.0);
        const bool reducer = (warp == 7 && i > 0 && g < 2 * kNB && (g % kNB) < i);
        if (reducer) {
            const int t = g % kNB, which = g / kNB;
            cplx rp[5];
#pragma unroll
            for (int u = 0; u < 5; ++u) { const int k = lane + 32 * u; rp[u] = (k < nprod) ? ldx_(&p.part[(size_t)k * PSTRIDE + 1 + which * kNB + t]) : mk(0.0, 0.0); }
            red_top = which == 0 ? ldx_(&A[(size_t)(p.j0 + t) * lda + c + 1]) : ldx_(&W[(size_t)t * ldw + c + 1]);
            red_s = ((rp[0] + rp[1]) + (rp[2] + rp[3])) + rp[4];
            for (int k = lane + 160; k < nprod; k += 32) red_s = red_s + ldx_(&p.part[(size_t)k * PSTRIDE + 1 + which * kNB + t]);
            red_s = warp_sum(red_s);
        }
        __syncthreads();
        const cplx tau = s_sc[0], scale = s_sc[1];
        if (reducer && lane == 0)     // row c+1 term (v = 1 there) plus scale * sum over rows >= c+2
            p.tot[(g / kNB) * kNB + (g % kNB)] = conj_(red_top) + scale * red_s;
        double qacc = 0.0;
        if (wide) {
            cplx *vI = s_v + warp * 2 * kTS, *vJ = vI + kTS;
            cplx accR = mk(0.0, 0.0), accC = mk(0.0, 0.0);
            int2 ij = make_int2(0, 0);
            if (wvalid) {
                ij = ijc[0];
                const bool diag = (ij.x == ij.y);
                const int rI = ij.x * kTS + lane, rJ = ij.y * kTS + lane;
                const cplx a = (rI == c + 1) ? mk(1.0, 0.0) : scale * rawI[0];
                const cplx b = diag ? a : ((rJ == c + 1) ? mk(1.0, 0.0) : scale * rawJ[0]);
                vI[lane] = a; vJ[lane] = b;
                __syncwarp();
                const cplx *sl = s_slots + (size_t)wtile * kSlotElems;
                if (!diag) {
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int cc = wq * 8 + u;
                        cfma(accR, sl[cc * kTP + lane], vJ[cc]);
                        cfma_conj(accC, sl[lane * kTP + cc], vI[cc]);
                    }
                } else {
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int cc = wq * 8 + u;
                        cplx x = sl[cc * kTP + lane];
                        x.x = (lane >= cc) ? x.x : 0.0;
                        x.y = (lane > cc) ? x.y : 0.0;
                        cfma(accR, x, vJ[cc]);
                        cplx y = sl[lane * kTP + cc];
                        y.x = (cc > lane) ? y.x : 0.0;
                        y.y = (cc > lane) ? y.y : 0.0;
                        cfma_conj(accC, y, vI[cc]);
                    }
                }
            }
            s_gV[warp * 32 + lane] = accR;
            s_gW[warp * 32 + lane] = accC;
            __syncthreads();
            if (wvalid && wq == 0) {
#pragma unroll
                for (int u = 1; u < 4; ++u) { accR = accR + s_gV[(warp + u) * 32 + lane]; accC = accC + s_gW[(warp + u) * 32 + lane]; }
                double qterm;
                if (ij.x == ij.y) {
                    const cplx sdiag = accR + accC;
                    p.PR[(size_t)ij.y * ldp + ij.x * kTS + lane] = sdiag;
                    qterm = vI[lane].x * sdiag.x + vI[lane].y * sdiag.y;
                } else {
                    p.PR[(size_t)ij.y * ldp + ij.x * kTS + lane] = accR;
                    p.PC[(size_t)ij.x * ldp + ij.y * kTS + lane] = accC;
                    qterm = 2.0 * (vI[lane].x * accR.x + vI[lane].y * accR.y);
                }
                qacc = warp_sum(qterm);
            }
        } else {
            cplx *vI = s_v + warp * 2 * kTS, *vJ = vI + kTS;
            {
                // the tile coordinates run three tiles and the pieces of column c two tiles ahead of the tile in work: a
                // tile used to start with two dependent L2 round trips (coordinates, then the column pieces)
                for (int jj = 0; jj < cnt; ++jj) {
                    const int P = 2 * jj + pr_m;
                    const int s3 = (fwd ? P : pcnt - 1 - P) % 3;
                    const int slot = pr_p + 4 * s3;
                    const unsigned expected = ((s3 == 0) ? base0 : (s3 == 1) ? base1 : base2) + (unsigned)(P / 3);
                    const int2 ij = ijq[0];
                    const int r0 = ij.x * kTS, c0 = ij.y * kTS;
                    const bool diag = (ij.x == ij.y);
                    int2 ij3 = make_int2(0, 0);
                    if (jj + 3 < cnt) ij3 = tile_of(jj + 3);
                    cplx nxtI = mk(0.0, 0.0), nxtJ = mk(0.0, 0.0);
                    if (jj + 2 < cnt) {
                        const int rI = ijq[2].x * kTS + lane, rJ = ijq[2].y * kTS + lane;
                        if (rI < n && rI > c + 1) nxtI = ldx_(&A[(size_t)c * lda + rI]);
                        if (ijq[2].x != ijq[2].y && rJ < n && rJ > c + 1) nxtJ = ldx_(&A[(size_t)c * lda + rJ]);
                    }
                    int2 ijr_n = make_int2(0, 0);
                    if (streaming && P + 5 < pcnt) ijr_n = pos_tile(P + 5);
                    // v pieces (formed on the fly; zero outside the trailing matrix)
                    {
                        const int rI = r0 + lane, rJ = c0 + lane;
                        cplx a = rawI[0], b = rawJ[0];
                        rawI[0] = rawI[1]; rawJ[0] = rawJ[1]; rawI[1] = nxtI; rawJ[1] = nxtJ;
                        ijq[0] = ijq[1]; ijq[1] = ijq[2]; ijq[2] = ij3;
                        a = (rI == c + 1) ? mk(1.0, 0.0) : scale * a;
                        b = diag ? a : ((rJ == c + 1) ? mk(1.0, 0.0) : scale * b);
                        __syncwarp();
                        vI[lane] = a; vJ[lane] = b;
                    }
                    // the load of this tile is the `expected`-th into its slot; it may not have been issued yet (the other warp
                    // of the pair issues it after its own tile): wait for the issue count first, a parity alone could be a
                    // whole phase behind
                    if (streaming) { while ((unsigned)s_iss[slot] < expected) {} }
                    mbar_wait(mbar0 + 8u * slot, (expected - 1u) & 1u);
                    __syncwarp();
                    const cplx *sl = s_slots + (size_t)slot * kSlotElems;
                    // two independent accumulator sets (even / odd columns) halve the dependent DFMA chains
                    cplx accR = mk(0.0, 0.0), accC = mk(0.0, 0.0), accR1 = mk(0.0, 0.0), accC1 = mk(0.0, 0.0);
                    if (!diag) {
#pragma unroll 8
                        for (int cc = 0; cc < kTS; cc += 2) {
                            cfma(accR, sl[cc * kTP + lane], vJ[cc]);              // lane = row
                            cfma(accR1, sl[(cc + 1) * kTP + lane], vJ[cc + 1]);
                            cfma_conj(accC, sl[lane * kTP + cc], vI[cc]);         // lane = column, cc = row
                            cfma_conj(accC1, sl[lane * kTP + cc + 1], vI[cc + 1]);
                        }
                    } else {
#pragma unroll 8
                        for (int cc = 0; cc < kTS; ++cc) {
                            cplx a = sl[cc * kTP + lane];                      // row = lane, col = cc
                            a.x = (lane >= cc) ? a.x : 0.0;
                            a.y = (lane > cc) ? a.y : 0.0;                     // real diagonal, nothing above it
                            cfma(accR, a, vJ[cc]);
                            cplx b = sl[lane * kTP + cc];                      // col = lane, row = cc
                            b.x = (cc > lane) ? b.x : 0.0;
                            b.y = (cc > lane) ? b.y : 0.0;
                            cfma_conj(accC1, b, vI[cc]);
                        }
                    }
                    accR = accR + accR1; accC = accC + accC1;
                    double qterm;
                    if (diag) {
                        const cplx s = accR + accC;
                        p.PR[(size_t)ij.y * ldp + r0 + lane] = s;
                        qterm = vI[lane].x * s.x + vI[lane].y * s.y;
                    } else {
                        p.PR[(size_t)ij.y * ldp + r0 + lane] = accR;
                        p.PC[(size_t)ij.x * ldp + c0 + lane] = accC;
                        qterm = 2.0 * (vI[lane].x * accR.x + vI[lane].y * accR.y);
                    }
                    qacc += qterm;                    // per lane; one warp reduction after the pass
                    if (streaming) {
                        // refill this slot with the tile that uses it next in this pass (position P + 3, the other warp's);
                        // at the end of a pass the slots keep their tiles, the first ones the reversed next pass needs
                        if (P + 3 < pcnt) {
                            __syncwarp();
                            warp_load_tile(s_slots + (size_t)slot * kSlotElems, mbar0 + 8u * slot, A, lda, n, ijr, lane);
                            if (lane == 0) { __threadfence_block(); s_iss[slot] = (int)(expected + 1u); }
                        }
                        ijr = ijr_n;
                    }
                }
                if (streaming) {
                    // loads of this pass per slot: positions 3 <= P' < pcnt; positions of one residue mod 3 share a slot
#pragma unroll
                    for (int r = 0; r < 3; ++r) {
                        if (pcnt - 1 >= r) {
                            const int s3r = (fwd ? r : pcnt - 1 - r) % 3;
                            const unsigned add = (unsigned)((pcnt - 1 - r) / 3);
                            if (s3r == 0) base0 += add; else if (s3r == 1) base1 += add; else base2 += add;
                        }
                    }
                }
            }
        }
        if (!wide) qacc = warp_sum(qacc);
        if (lane == 0) s_q[warp] = qacc;
        __syncthreads();
        if (tid == 0 && g < T) {
            double t = 0.0;
            for (int k = 0; k < 8; ++k) t += s_q[k];
            p.qpart[g] = t;
        }
        grid.sync();

        // ================= phase B: rows spread over the CTAs; one dependent L2 round trip =================
        // lane = row (31 consecutive rows per CTA; lane 31 is the helper row c+1, whose w every CTA needs
        // for the next-column update); warp w serves tile columns b = J0 + w (mod 8) of the partials and
        // panel columns t = w (mod 8) of V and W: every global load is a coalesced 512-byte row segment.
        {
            const bool do_next = (i + 1 < p.nbp);
            const int J0 = (c + 1) / kTS;
            const int rows = n - (c + 1);
            const int L = rows_per_cta(rows, G);
            const bool active = g * L < rows;                    // block-uniform: this CTA owns rows
            cplx *s_p1 = s_gV, *s_p2 = s_gW;                     // 8 x 32 each
            double *s_re = s_S;                                  // 8
            cplx accV[kNB / 8], accW[kNB / 8];
#pragma unroll
            for (int k = 0; k < kNB / 8; ++k) { accV[k] = mk(0.0, 0.0); accW[k] = mk(0.0, 0.0); }
            double S = 0.0;
            for (int base = 0; active && base < L; base += 31) {          // block-uniform trip count
                const bool helper = (lane == 31);
                const int rr = base + lane;
                const int r = helper ? c + 1 : c + 1 + g * L + rr;
                const bool ok = helper ? do_next : (rr < L && r < n);
                const bool okr = ok && !helper;
                // ---- every global load of the pass is issued before the first shared-memory write
                const cplx ar = okr ? ldx_(&A[(size_t)c * lda + r]) : mk(0.0, 0.0);
                const cplx anx = (okr && do_next) ? ldx_(&A[(size_t)(c + 1) * lda + r]) : mk(0.0, 0.0);
                // warp 1 also gathers the v^H y partials of phase A; issued here so that they share the round trip
                double qv = 0.0, qv0 = 0.0, qv1 = 0.0, qv2 = 0.0, qv3 = 0.0, qv4 = 0.0;
                if (warp == 1) {
                    const int nq = T < G ? T : G;
                    if (lane < nq) qv0 = ldx_(&p.qpart[lane]);
                    if (lane + 32 < nq) qv1 = ldx_(&p.qpart[lane + 32]);
                    if (lane + 64 < nq) qv2 = ldx_(&p.qpart[lane + 64]);
                    if (lane + 96 < nq) qv3 = ldx_(&p.qpart[lane + 96]);
                    for (int k = lane + 128; k < nq; k += 32) qv4 += ldx_(&p.qpart[k]);
                }
                // cV, cW are the same 2 x 32 values for every warp of every CTA: one warp fetches them with two coalesced
                // loads and hands them over in shared memory (a load per warp and value made these 8 lines the hottest
                // in L2: ~1000 requests per line per column at n = 4096, queued for microseconds)
                cplx totV = mk(0.0, 0.0), totW = mk(0.0, 0.0);
                if (warp == 2 && lane < i) { totV = ldx_(&p.tot[lane]); totW = ldx_(&p.tot[kNB + lane]); }
                cplx Vr[kNB / 8], Wr[kNB / 8];
#pragma unroll
                for (int k = 0; k < kNB / 8; ++k) {
                    const int t = warp + 8 * k;
                    Vr[k] = mk(0.0, 0.0); Wr[k] = mk(0.0, 0.0);
                    if (t < i && ok) {
                        Vr[k] = ldx_(&A[(size_t)(p.j0 + t) * lda + r]);
                        Wr[k] = ldx_(&W[(size_t)t * ldw + r]);
                    }
                }
                cplx p1 = mk(0.0, 0.0);
                if (ok) {
                    const int R = r / kTS;
                    // eight independent loads in flight per group (no load -> add -> load chains)
                    for (int b0 = J0 + warp; b0 < p.nblk; b0 += 64) {
                        cplx v[8];
#pragma unroll
                        for (int u = 0; u < 8; ++u) {
                            const int bb = b0 + 8 * u;
                            v[u] = mk(0.0, 0.0);
                            if (bb < p.nblk) v[u] = (bb <= R) ? ldx_(&p.PR[(size_t)bb * ldp + r]) : ldx_(&p.PC[(size_t)bb * ldp + r]);
                        }
                        p1 = p1 + (((v[0] + v[1]) + (v[2] + v[3])) + ((v[4] + v[5]) + (v[6] + v[7])));
                    }
                }
                if (warp == 1) qv = warp_sum((qv0 + qv1) + (qv2 + qv3) + qv4);
                if (warp == 2) { s_cV[lane] = totV; s_cW[lane] = totW; }
                __syncthreads();                                  // cV, cW visible; previous pass / previous column readers done
                // ---- partial sums of this warp: y - V cW - W cV,  V conj(W[c+1,:]) + W conj(V[c+1,:]),  Re(cV^H cW)
                cplx p2 = mk(0.0, 0.0);
                double re = 0.0;
#pragma unroll
                for (int k = 0; k < kNB / 8; ++k) {
                    if (warp + 8 * k >= i) continue;             // warp-uniform
                    const cplx cvk = s_cV[warp + 8 * k], cwk = s_cW[warp + 8 * k];
                    // rows c+1 of V and W sit in the helper lane
                    const cplx v1 = mk(__shfl_sync(0xffffffffu, Vr[k].x, 31), __shfl_sync(0xffffffffu, Vr[k].y, 31));
                    const cplx w1 = mk(__shfl_sync(0xffffffffu, Wr[k].x, 31), __shfl_sync(0xffffffffu, Wr[k].y, 31));
                    cplx corr = mk(0.0, 0.0);
                    cfma(corr, Vr[k], cwk); cfma(corr, Wr[k], cvk);
                    p1 = p1 - corr;
                    cfma(p2, Vr[k], conj_(w1)); cfma(p2, Wr[k], conj_(v1));
                    re += cvk.x * cwk.x + cvk.y * cwk.y;
                }
                s_p1[warp * 32 + lane] = p1;
                s_p2[warp * 32 + lane] = p2;
                if (lane == 0) s_re[warp] = re;
                if (warp == 1 && lane == 0) s_q[8] = qv;
                __syncthreads();
                cplx ys = mk(0.0, 0.0), upd = mk(0.0, 0.0);
                double ret = 0.0;
#pragma unroll
                for (int w8 = 0; w8 < 8; ++w8) { ys = ys + s_p1[w8 * 32 + lane]; upd = upd + s_p2[w8 * 32 + lane]; ret += s_re[w8]; }
                // alpha' = -1/2 |tau|^2 (v^H y), v^H y = q - 2 Re(cV^H cW);  w_r = tau (y_r - V_r cW - W_r cV) + alpha' v_r
                const double alphap = -0.5 * abs2(tau) * (s_q[8] - 2.0 * ret);
                const cplx vr = (r == c + 1) ? mk(1.0, 0.0) : scale * ar;
                const cplx wr = tau * ys + alphap * vr;
                if (okr && warp == 0) W[(size_t)i * ldw + r] = wr;
                if (okr && warp == 1) A[(size_t)c * lda + r] = vr;
                if (!do_next) continue;                           // block-uniform
                const cplx wc1 = mk(__shfl_sync(0xffffffffu, wr.x, 31), __shfl_sync(0xffffffffu, wr.y, 31));
                // a'_r = A[r,c+1] - sum_{t<=i} V[r,t] conj(W[c+1,t]) + W[r,t] conj(V[c+1,t])
                cfma(upd, vr, conj_(wc1));
                upd = upd + wr;                                   // V[c+1, i] = 1
                cplx an = anx - upd;
                if (okr && r == c + 1) { an.y = 0.0; if (warp == 2) p.d[c + 1] = an.x; }
                if (okr && warp == 2) A[(size_t)(c + 1) * lda + r] = an;
                if (!(okr && r >= c + 3)) an = mk(0.0, 0.0);       // rows that enter the next column's partials
                if (warp == 3) S += abs2(an);
#pragma unroll
                for (int k = 0; k < kNB / 8; ++k) {
                    const int t = warp + 8 * k;
                    if (t < i) { cfma_conj(accV[k], Vr[k], an); cfma_conj(accW[k], Wr[k], an); }
                    else if (t == i) { cfma_conj(accV[k], vr, an); cfma_conj(accW[k], wr, an); }
                }
            }
            if (do_next && active) {
                // partials of the next column: sums over this CTA's rows (lanes), written straight to global
#pragma unroll
                for (int k = 0; k < kNB / 8; ++k) {
                    const int t = warp + 8 * k;
                    if (t <= i) {                                  // warp-uniform
                        const cplx sv = warp_sum(accV[k]), sw = warp_sum(accW[k]);
                        if (lane == 0) {
                            p.part[(size_t)g * PSTRIDE + 1 + t] = sv;
                            p.part[(size_t)g * PSTRIDE + 1 + kNB + t] = sw;
                        }
                    }
                }
                if (warp == 3) {
                    S = warp_sum(S);
                    if (lane == 0) p.part[(size_t)g * PSTRIDE] = mk(S, 0.0);
                }
            }
        }
        if (i + 1 < p.nbp) grid.sync();
    }
    // no bulk copy may be in flight when the CTA exits (a one-column last panel never reads its tiles)
    if (wide) { if (warp < 2 && warp < q && g + warp * G < T) mbar_wait(mbar0 + 8u * warp, 0u); }
    else {
        if (0 < pcnt) mbar_wait(mbar0 + 8u * (pr_p + 0), (base0 - 1u) & 1u);
        if (1 < pcnt) mbar_wait(mbar0 + 8u * (pr_p + 4), (base1 - 1u) & 1u);
        if (2 < pcnt) mbar_wait(mbar0 + 8u * (pr_p + 8), (base2 - 1u) & 1u);
    }
}

static size_t panel_smem_bytes() {
    return sizeof(cplx) * (size_t)(kSlots * kSlotElems + 8 * 2 * kTS + 4 * kNB + 16 * kNB + 4) + sizeof(double) * (20 + kSlots + (kSlots + 1) / 2);
}

// ---------------------------------------------------------------- HER2K (DMMA)
struct Her2kEpi {
    cplx *C; int ldc;
    static constexpr bool kRmw = true;
    __device__ __forceinline__ cplx load(int i, int j) const { return C[(size_t)j * ldc + i]; }
    __device__ __forceinline__ void store(int i, int j, cplx v, double re, double im) const {
        v.x -= re; v.y -= im;
        if (i == j) v.y = 0.0;
        C[(size_t)j * ldc + i] = v;
    }
};

constexpr int H2_MI = 4, H2_NI = 4, H2_WM = 2, H2_WN = 2;   // 64 x 64 CTA tile, 4 warps

// K is only 64 per output tile, so prologue and epilogue weigh as much as the main loop: two stages and
// three CTAs per SM let one CTA's loads and read-modify-write overlap another's DMMAs
__global__ void __launch_bounds__(H2_WM *H2_WN * 32, 3) her2k_kernel(GemmProblem<cplx, cplx> p, Her2kEpi epi) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (blockIdx.y > blockIdx.x) return;   // lower triangle of tiles only
    gemm_tile_body<cplx, cplx, MNMAJ, MNMAJ, false, true, H2_MI, H2_NI, H2_WM, H2_WN, true, 2>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
}

// small trailing matrices: 32 x 32 CTA tiles, so that the grid still covers the SMs and each CTA is short
__global__ void __launch_bounds__(H2_WM *H2_WN * 32) her2k_small_kernel(GemmProblem<cplx, cplx> p, Her2kEpi epi) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (blockIdx.y > blockIdx.x) return;
    gemm_tile_body<cplx, cplx, MNMAJ, MNMAJ, false, true, 2, 2, H2_WM, H2_WN, true>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
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
    if (cudaFuncSetAttribute(tridiag_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)panel_smem_bytes()) != cudaSuccess) return HPSD_ECUDA_;
    constexpr size_t h2 = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, H2_MI, H2_NI, H2_WM, H2_WN, 2>();
    if (cudaFuncSetAttribute(her2k_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h2) != cudaSuccess) return HPSD_ECUDA_;
    constexpr size_t h2s = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, 2, 2, H2_WM, H2_WN>();
    if (cudaFuncSetAttribute(her2k_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h2s) != cudaSuccess) return HPSD_ECUDA_;
    g_panel_init_dev = dev;
    return 0;
}


int tridiag_tile_size(int) { return kTS; }

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
    p.n = n; p.lda = w.lda; p.ldw = w.ldw; p.nblk = (n + ts - 1) / ts; p.G = sms < kMaxPanelCtas ? sms : kMaxPanelCtas;
    if (p.G < 2 * kNB) return HPSD_ECUDA_;   // the reducers of phase A need 64 CTAs
    p.A = w.A; p.W = w.W; p.d = w.d; p.e = w.e; p.tau = w.tau;
    p.ldp = w.ldp; p.PR = w.PR; p.PC = w.PC; p.part = w.part; p.tot = w.tot; p.qpart = w.qpart; p.tiles = w.tiles;
    if (n == 1) {
        // d[0] = Re A[0,0]; handled by a 1-column panel (sets d in the prologue)
    }
    const int G_full = p.G;
    const int G_cap = (w.max_ctas >= 2 * kNB && w.max_ctas < G_full) ? w.max_ctas : G_full;
    if (w.wide_done && w.wide_panels <= 0 && cudaEventRecord(w.wide_done, st) != cudaSuccess) return HPSD_ECUDA_;
    for (int j0 = 0; j0 < n; j0 += kNB) {
        // panel lanes: the first wide_panels panels on every SM, the rest next to the other lane's kernel
        p.G = (j0 / kNB >= w.wide_panels) ? G_cap : G_full;
        if (w.wide_done && w.wide_panels > 0 && j0 / kNB == w.wide_panels && cudaEventRecord(w.wide_done, st) != cudaSuccess) return HPSD_ECUDA_;
        p.j0 = j0;
        p.nbp = (n - j0 < kNB) ? (n - j0) : kNB;
        const int nbk = p.nblk - j0 / kTS;              // tile rows/columns of this panel's trailing matrix
        p.T = nbk * (nbk + 1) / 2;
        p.q = (p.T + p.G - 1) / p.G;
        void *args[] = {&p};
        const size_t smem = panel_smem_bytes();
        cudaError_t e;
        prof_begin(ST_PANEL, st);
        e = cudaLaunchCooperativeKernel((void *)tridiag_panel_kernel, dim3(p.G), dim3(kPanelThreads), args, smem, st);
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
            constexpr size_t h2 = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, H2_MI, H2_NI, H2_WM, H2_WN, 2>();
            constexpr size_t h2s = gemm_smem_bytes<cplx, cplx, MNMAJ, MNMAJ, 2, 2, H2_WM, H2_WN>();
            prof_begin(ST_HER2K, st);
            if (m2 <= 1536) {
                const int nt = (m2 + 31) / 32;
                her2k_small_kernel<<<dim3(nt, nt), H2_WM * H2_WN * 32, h2s, st>>>(gp, epi);
            } else {
                const int nt = (m2 + 63) / 64;
                her2k_kernel<<<dim3(nt, nt), H2_WM * H2_WN * 32, h2, st>>>(gp, epi);
            }
            prof_end(ST_HER2K, st);
            HPSD_LAUNCH_CHECK();
        }
    }
    if (w.wide_done && w.wide_panels > 0 && (long long)w.wide_panels * kNB >= n && cudaEventRecord(w.wide_done, st) != cudaSuccess) return HPSD_ECUDA_;
    if (n > 1) {
        clean_v_kernel<<<dim3((n + 255) / 256, n), 256, 0, st>>>(n, w.A, w.lda);
        HPSD_LAUNCH_CHECK();
    }
    return 0;
}

}  // namespace hpsd
