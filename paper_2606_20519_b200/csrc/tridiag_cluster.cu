// tridiag_cluster.cu -- S1 + S2 + S3 of SURVEY.md §8(a) for blocks whose lower triangle fits in the
// shared memory of ONE 16-CTA thread-block cluster (n <= ~631: the paper's d = 5, n = 625 block).
// svec -> REAL symmetric tridiagonal (d, e) + reflectors V, tau, same conventions as tridiag.cu:
// A = Q T Q^H, Q = H_0 ... H_{n-2}, H_c = I - tau_c v_c v_c^H (zlarfg: complex tau, real beta).
// "Eigendecomposition" of PAPER.md:1536 starts here; the design is ours (the paper calls a library).
//
// Why: at n = 625 the grid-wide panel kernel is bound by two grid barriers per column (1.1-1.5 us
// each on B200).  Exchanges inside a cluster are cheaper, and 16 x 227 KB of distributed
// shared memory hold the whole packed lower triangle (3.1 MB at n = 625), so the matrix is read from
// HBM exactly once (straight from the svec: S1 is fused) and every column step runs out of shared memory.
//
// Layout: column j belongs to CTA j mod 16 and is stored packed (rows j..n-1, contiguous).
// Rows are owned by threads: three 32-row chunks per warp (cl_chunk: a light, a middle and a heavy one); each thread
// keeps v_i, w_i, u_i of its rows in registers.
//
// Step c (unblocked, LAPACK zhetd2 arithmetic, one fused pass per column):
//   [A] every CTA (redundantly, bit-identically) forms column c of the current matrix from the raw
//       column the owner exported, a' = raw - v conj(w_c) - w, its Householder vector u = v_c, tau, beta;
//   [B] one pass over the CTA's own columns j >= c+1: A_ij -= v_i conj(w_j) + w_i conj(v_j) (the
//       rank-2 update of step c-1, applied late) and, in the same sweep, z_i += A_ij u_j,
//       t_j += conj(A_ij) u_i (the Hermitian mat-vec of step c from the stored half);
//   [C] contributions z_i (+ t_i) are pushed through DSMEM to the CTA that sums row i (rows are dealt to the
//       16 CTAs in contiguous slices); the partial v^H y goes to everybody with phase 2 (needed only with w);
//   [D] that CTA sums the 16 contributions of its rows and broadcasts tau y_i;
//       w_i = tau y_i - 1/2 |tau|^2 (v^H y) u_i is completed by every receiver.
// Both exchanges are st.async stores that complete transaction bytes on the RECEIVER's mbarrier: data and
// signal travel together (one DSMEM trip), there is no cluster-wide barrier inside the loop (the hardware
// cluster barrier costs 0.55-0.7 us with 16 CTAs, measured).  The raw next column travels through a
// two-entry ring in global memory (L2): the CTA that stores column c+1 brings it up to date and exports it BEFORE
// its pass, fences after the pass and sends one 8-byte token per warp to every CTA on the phase-1 mbarrier, so
// nobody reads the ring before the export is visible and the fence is off the critical path.
// Buffer and mbarrier-phase reuse is safe by construction, not by timing: phase tokens and the late
// push of v^H y order the steps between CTAs, every thread reads before it sends, and nothing a peer may write early
// shares memory with anything read late (the t_j partials once did: a race that eight concurrent clusters exposed).
//
// Measured on B200 (round 1), S1+S2+S3 alone: n = 200 0.70 ms (grid-wide panel kernel 1.31), n = 400 1.97 (2.70),
// n = 625 3.93 (4.37).  Every warp walks a serial chain of ~10 trips of ~1500 cycles per column step (t_j warp
// reductions and the issue overhead around the 16 DFMA per element), so the FP64 pipe of the 16 SMs is 17 % busy at n = 625 (ncu, profiles/r1_cluster_ncu_full.md).
#include <cooperative_groups.h>
#include "kernels.h"
#include "large.h"
#include "prof.h"

namespace cg = cooperative_groups;

namespace hpsd {

constexpr int kCl = 16;            // CTAs per cluster (non-portable size)
constexpr int kClThreads = 256;
constexpr int kClWarps = kClThreads / 32;
constexpr int kClR = 3;            // row slots per thread: n <= 768
constexpr int kClMaxN = 32 * kClWarps * kClR;
constexpr int kKT = 4;             // own columns per trip of the pass
constexpr int kRedN = 0, kRedQ = kClWarps, kRedS = 2 * kClWarps;   // s_red: norm partials | dot partials | alpha.x, alpha.y, d_c
// 32-row chunk of (slot, warp): odd slots run backwards so that every warp gets a light and a heavy chunk
__device__ __forceinline__ int cl_chunk(int s, int wp) { return kClWarps * s + ((s & 1) ? kClWarps - 1 - wp : wp); }
// ---- data + signal in one DSMEM trip: st.async stores complete transaction bytes on the receiver's mbarrier ----
__device__ __forceinline__ unsigned cl_mapa(unsigned addr, int rank) {
    unsigned remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(addr), "r"(rank));
    return remote;
}
__device__ __forceinline__ void cl_st_async(unsigned raddr, cplx v, unsigned rmbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(raddr), "d"(v.x), "d"(v.y), "r"(rmbar) : "memory");
}
__device__ __forceinline__ void cl_st_async(unsigned raddr, double v, unsigned rmbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(raddr), "d"(v), "r"(rmbar) : "memory");
}
// one pending arrival per phase (this arm) + the bytes the phase will receive
__device__ __forceinline__ void cl_arm(unsigned mbar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cl_wait(unsigned mbar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "CL_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra CL_DONE_%=;\n\t"
        "bra CL_WAIT_%=;\n\t"
        "CL_DONE_%=:\n\t}" ::"r"(mbar), "r"(parity) : "memory");
}
__device__ __forceinline__ void cl_barrier() {
    // release/acquire at CLUSTER scope (cooperative_groups' cluster.sync() fences at gpu scope: MEMBAR.ALL.GPU)
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

struct ClusterArgs {
    int n, lda;
    const double *in, *sub;        // svec (and the ADMM subtrahend, or null)
    cplx *A;                       // lda x n: reflectors out (zero on and above the diagonal)
    cplx *raw;                     // 2 x lda ring of exported raw columns
    double *d, *e;
    cplx *tau;
    int *nf;                       // device flag: non-finite input seen
    int f32;                       // svec stored as FP32 (common.cuh)
};

__host__ __device__ inline int cl_ncols(int n, int r) { return r < n ? (n - r + kCl - 1) / kCl : 0; }
__host__ __device__ inline size_t cl_col_off(int n, int r, int jl) { return (size_t)jl * (n - r) - (size_t)8 * jl * (jl - 1); }

struct ClusterSmem {
    size_t mbar, tok, colv, q, red, rbuf, wbuf, tpart, stor, total;
};
__host__ __device__ inline ClusterSmem cl_smem(int n, int r) {
    ClusterSmem s;
    const int nc = cl_ncols(n, 0);                 // widest CTA
    const int rs = (n + kCl - 1) / kCl;
    size_t off = 0;
    s.mbar = off; off += 16;                      // two mbarriers
    s.tok = off; off += 8 * (kClWarps + kCl);     // landing slots of the export tokens and of the phase tokens
    s.colv = off; off += sizeof(cplx) * 3 * nc;
    s.q = off; off += sizeof(double) * 2 * kCl;    // v^H y partials, double-buffered by step parity
    s.red = off; off += sizeof(double) * (2 * kClWarps + 4);   // block-reduction scratch + alpha, d_c
    s.rbuf = off; off += sizeof(cplx) * kCl * (rs | 1);
    s.wbuf = off; off += sizeof(cplx) * n;
    // the t_j partials must NOT share memory with wbuf: a reducer may broadcast tau y (into wbuf) as soon as IT has the
    // contributions of its own rows, while another thread of this CTA is still reading t_j partials for a different row
    s.tpart = off; off += sizeof(cplx) * kClWarps * nc;
    s.stor = off;
    off += sizeof(cplx) * cl_col_off(n, r, cl_ncols(n, r));
    s.total = off;
    return s;
}

__device__ __forceinline__ void cl_householder(cplx alpha, double xnorm2, double &beta, cplx &tau, cplx &scale) {
    if (xnorm2 == 0.0 && alpha.y == 0.0) {
        beta = alpha.x; tau = mk(0.0, 0.0); scale = mk(0.0, 0.0);
    } else {
        // zlarfg scalars with one reciprocal square root and one reciprocal on the dependent chain (every CTA runs this
        // redundantly once per column): 1/beta comes from rsqrt, refined by one Newton step to full accuracy
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

// element (i, j), i >= j, of the input matrix from the svec (Eq. D10 inverted; same arithmetic as unpack_kernel)
// non-finite entries are replaced by zero and *nf is set (common.cuh: the output block becomes NaN)
__device__ __forceinline__ cplx cl_load_svec(const double *__restrict__ sv, const double *__restrict__ sub, int n, int i, int j, int *nf, int f32) {
    const size_t o = svec_col_off(n, j);
    cplx v;
    if (i == j) v = mk(sub ? sv_ld(sv, o, f32) - sv_ld(sub, o, f32) : sv_ld(sv, o, f32), 0.0);
    else {
        const size_t k = o + 1 + 2 * (size_t)(i - j - 1);
        double re = sv_ld(sv, k, f32), im = sv_ld(sv, k + 1, f32);
        if (sub) { re -= sv_ld(sub, k, f32); im -= sv_ld(sub, k + 1, f32); }
        v = mk(re / kSqrt2, im / kSqrt2);
    }
    if (nonfinite(v.x) || nonfinite(v.y)) { v = mk(0.0, 0.0); if (nf) *nf = 1; }
    return v;
}


// One row chunk x kKT own columns of the fused pass.  x holds A(i, j_k) (zero where the element does not exist), m says
// where it exists.  Branch-free: masks are selects (a predicate-free variant behind a warp-uniform branch was slower).
__device__ __forceinline__ void cl_elems(cplx (&x)[kKT], const bool (&m)[kKT], int i, int j0, cplx *const (&col)[kKT], int i0,
                                         cplx v, cplx w, cplx u, const cplx (&cv)[kKT], const cplx (&cw)[kKT], const cplx (&cu)[kKT],
                                         cplx &z, cplx (&tj)[kKT]) {
#pragma unroll
    for (int k = 0; k < kKT; ++k) {
        cplx xx = x[k];
        // xx -= v_i conj(w_j) + w_i conj(v_j)
        xx.x = fma(-v.x, cw[k].x, xx.x); xx.x = fma(-v.y, cw[k].y, xx.x);
        xx.x = fma(-w.x, cv[k].x, xx.x); xx.x = fma(-w.y, cv[k].y, xx.x);
        xx.y = fma(-v.y, cw[k].x, xx.y); xx.y = fma(v.x, cw[k].y, xx.y);
        xx.y = fma(-w.y, cv[k].x, xx.y); xx.y = fma(w.x, cv[k].y, xx.y);
        cplx ut = u;
        const int j = j0 + kCl * k;
        if (!m[k]) xx = mk(0.0, 0.0);
        if (i == j) xx.y = 0.0;                                   // the diagonal stays real
        if (i <= j) ut = mk(0.0, 0.0);                            // t_j sums the rows strictly below the diagonal
        if (m[k]) col[k][i0] = xx;
        cfma(z, xx, cu[k]);
        cfma_conj(tj[k], xx, ut);
    }
}

__global__ void __launch_bounds__(kClThreads, 1) tridiag_cluster_kernel(ClusterArgs p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cg::cluster_group cluster = cg::this_cluster();
    const int r = (int)cluster.block_rank();
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    const int n = p.n, lda = p.lda;
    const ClusterSmem L = cl_smem(n, r);
    cplx *colv_v = reinterpret_cast<cplx *>(smem_raw + L.colv);
    const int ncw = cl_ncols(n, 0);
    cplx *colv_w = colv_v + ncw, *colv_u = colv_w + ncw;
    double *s_q = reinterpret_cast<double *>(smem_raw + L.q);
    double *s_red = reinterpret_cast<double *>(smem_raw + L.red);   // kRedN.. norm, kRedQ.. dot, kRedS.. alpha, d_c
    cplx *rbuf = reinterpret_cast<cplx *>(smem_raw + L.rbuf);                 // [sender][RSP]
    const int RS = (n + kCl - 1) / kCl, RSP = RS | 1;
    cplx *wbuf = reinterpret_cast<cplx *>(smem_raw + L.wbuf);
    cplx *tpart = reinterpret_cast<cplx *>(smem_raw + L.tpart);       // [warp][ncw]
    cplx *stor = reinterpret_cast<cplx *>(smem_raw + L.stor);
    const int nc = cl_ncols(n, r);

    // ---- S1 fused: own columns straight from the svec into shared memory (one warp per column)
    for (int jl = wp; jl < nc; jl += kClWarps) {
        const int j = r + kCl * jl;
        cplx *col = stor + cl_col_off(n, r, jl);
        for (int i = j + lane; i < n; i += 32) col[i - j] = cl_load_svec(p.in, p.sub, n, i, j, p.nf, p.f32);
    }
    int row[kClR], dest[kClR], dslot[kClR];
    cplx v[kClR], w[kClR], u[kClR], z[kClR], raw[kClR];
#pragma unroll
    for (int s = 0; s < kClR; ++s) {
        row[s] = 32 * cl_chunk(s, wp) + lane;
        dest[s] = row[s] / RS; dslot[s] = row[s] - dest[s] * RS;       // reducer CTA of the row and its slot there
        v[s] = w[s] = u[s] = z[s] = mk(0.0, 0.0);
        raw[s] = row[s] < n ? cl_load_svec(p.in, p.sub, n, row[s], 0, p.nf, p.f32) : mk(0.0, 0.0);
    }
    cplx wc = mk(0.0, 0.0);
    const unsigned mbar1 = (unsigned)__cvta_generic_to_shared(smem_raw + L.mbar), mbar2 = mbar1 + 8;
    const unsigned rbuf_a = (unsigned)__cvta_generic_to_shared(rbuf), wbuf_a = (unsigned)__cvta_generic_to_shared(wbuf);
    const unsigned sq_a = (unsigned)__cvta_generic_to_shared(s_q), tok_a = (unsigned)__cvta_generic_to_shared(smem_raw + L.tok);
    // bytes phase c of each mbarrier receives: 16 senders x (my active rows + the v^H y partial); all active rows of w
    auto bytes_r = [&](int c) -> unsigned {
        int lo = r * RS, hi = lo + RS;
        if (lo < c + 1) lo = c + 1;
        if (hi > n) hi = n;
        const int act = hi > lo ? hi - lo : 0;
        // + the export tokens of the owner of column c+1 + (from step 1 on) one phase token per CTA
        return (unsigned)(kCl * act * 16 + kClWarps * 8 + (c > 0 ? kCl * 8 : 0));
    };
    auto bytes_w = [&](int c) -> unsigned { return (unsigned)((n - c - 1) * 16 + kCl * 8); };
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar1), "r"(1));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar2), "r"(1));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        cl_arm(mbar1, bytes_r(0));
        cl_arm(mbar2, bytes_w(0));
    }
    cl_barrier();       // every CTA of the cluster is resident before the first DSMEM access

    for (int c = 0; c < n; ++c) {
        // ================= [A] column c of the current matrix, Householder vector =================
        cplx a[kClR];
        double xn = 0.0;
#pragma unroll
        for (int s = 0; s < kClR; ++s) {
            const int i = row[s];
            cplx t = mk(0.0, 0.0);
            if (i >= c && i < n) {
                t = raw[s] - w[s];
                t.x -= v[s].x * wc.x + v[s].y * wc.y;       // v conj(wc)
                t.y -= v[s].y * wc.x - v[s].x * wc.y;
            }
            a[s] = t;
            if (i == c) s_red[kRedS + 2] = t.x;
            if (i == c + 1) { s_red[kRedS] = t.x; s_red[kRedS + 1] = t.y; }
            if (i >= c + 2) xn += abs2(t);
        }
        xn = warp_sum(xn);
        if (lane == 0) s_red[kRedN + wp] = xn;
        __syncthreads();
        const double dc = s_red[kRedS + 2];
        if (c == n - 1) {
            if (r == (c & (kCl - 1))) {
                if (tid == 0) { p.d[c] = dc; p.e[c] = 0.0; p.tau[c] = mk(0.0, 0.0); }
#pragma unroll
                for (int s = 0; s < kClR; ++s) if (row[s] < n) p.A[(size_t)c * lda + row[s]] = mk(0.0, 0.0);
            }
            break;
        }
        double xnorm2 = 0.0;
#pragma unroll
        for (int k = 0; k < kClWarps; ++k) xnorm2 += s_red[kRedN + k];
        const cplx alpha = mk(s_red[kRedS], s_red[kRedS + 1]);
        double beta; cplx tau, scale;
        cl_householder(alpha, xnorm2, beta, tau, scale);
#pragma unroll
        for (int s = 0; s < kClR; ++s) {
            const int i = row[s];
            u[s] = (i == c + 1) ? mk(1.0, 0.0) : ((i > c + 1 && i < n) ? scale * a[s] : mk(0.0, 0.0));
            if (i < n && (i & (kCl - 1)) == r && i >= c + 1) {
                const int jl = i >> 4;
                colv_v[jl] = v[s]; colv_w[jl] = w[s]; colv_u[jl] = u[s];
            }
        }
        if (r == (c & (kCl - 1))) {
            if (tid == 0) { p.d[c] = dc; p.e[c] = beta; p.tau[c] = tau; }
#pragma unroll
            for (int s = 0; s < kClR; ++s) if (row[s] < n) p.A[(size_t)c * lda + row[s]] = u[s];   // zero for rows <= c
        }
        __syncthreads();

        // ================= [B] fused rank-2 update (step c-1) + Hermitian mat-vec (step c) =================
        // Four own columns per trip: twelve independent element chains per thread hide the shared-memory
        // and DFMA latencies; the four t_j are reduced over the warp by one halving butterfly.
#pragma unroll
        for (int s = 0; s < kClR; ++s) z[s] = mk(0.0, 0.0);
        const int jl0 = (c + 1 > r) ? (c + 1 - r + kCl - 1) / kCl : 0;
        cplx *rawn = p.raw + (size_t)((c + 1) & 1) * lda;
        const bool owner = (jl0 < nc && r + kCl * jl0 == c + 1);  // this CTA stores column c+1
        if (owner) {
            // bring column c+1 to its final state first and export it for step c+1 (L2); every thread updates the
            // rows it also handles in the pass, so no synchronisation is needed; the pass then skips its update
            const cplx cvo = colv_v[jl0], cwo = colv_w[jl0];
            cplx *colx = stor + cl_col_off(n, r, jl0) - (c + 1);
#pragma unroll
            for (int s = 0; s < kClR; ++s) {
                const int i = row[s];
                if (i >= c + 1 && i < n) {
                    cplx x = colx[i];
                    x.x = fma(-v[s].x, cwo.x, x.x); x.x = fma(-v[s].y, cwo.y, x.x);
                    x.x = fma(-w[s].x, cvo.x, x.x); x.x = fma(-w[s].y, cvo.y, x.x);
                    x.y = fma(-v[s].y, cwo.x, x.y); x.y = fma(v[s].x, cwo.y, x.y);
                    x.y = fma(-w[s].y, cvo.x, x.y); x.y = fma(w[s].x, cvo.y, x.y);
                    if (i == c + 1) x.y = 0.0;
                    colx[i] = x;
                    rawn[i] = x;
                }
            }
        }
        // rows of this warp end at top_end: once the trip's first column lies beyond them the warp is done
        int top_end = 0;
#pragma unroll
        for (int s = 0; s < kClR; ++s) { const int e = 32 * cl_chunk(s, wp) + 32; if (e - 32 < n && e > top_end) top_end = e; }
        if (top_end > n) top_end = n;
        int jl = jl0;
        for (; jl < nc; jl += kKT) {
            const int j0 = r + kCl * jl;
            if (j0 >= top_end) break;                              // warp-uniform
            cplx cv[kKT], cw[kKT], cu[kKT], tj[kKT];
            cplx *col[kKT];
#pragma unroll
            for (int k = 0; k < kKT; ++k) {
                const bool okc = jl + k < nc;
                const int jk = okc ? jl + k : jl;
                cv[k] = colv_v[jk]; cw[k] = colv_w[jk];
                if (owner && jk == jl0) cv[k] = cw[k] = mk(0.0, 0.0);           // column c+1 is already up to date
                cu[k] = okc ? colv_u[jk] : mk(0.0, 0.0);
                col[k] = stor + cl_col_off(n, r, jk) - (r + kCl * jk) + lane;   // col[k][i0] = A(i0 + lane, j_k)
                tj[k] = mk(0.0, 0.0);
            }
            const int ncol = nc - jl;                             // valid columns of this trip (>= kKT except in the last one)
            cplx x[kClR][kKT];
            bool m[kClR][kKT];
#pragma unroll
            for (int s = 0; s < kClR; ++s) {
                const int i0 = 32 * cl_chunk(s, wp), i = i0 + lane;
#pragma unroll
                for (int k = 0; k < kKT; ++k) {
                    m[s][k] = (k < ncol) && i >= j0 + kCl * k && i < n;
                    x[s][k] = mk(0.0, 0.0);
                    if (m[s][k]) x[s][k] = col[k][i0];
                }
            }
#pragma unroll
            for (int s = 0; s < kClR; ++s) {
                const int i0 = 32 * cl_chunk(s, wp), i = i0 + lane;
                if (i0 + 31 < j0 || i0 >= n) continue;            // warp-uniform: nothing of this chunk in the trip
                // (a predicate-free variant for chunks entirely below the diagonals was measured and dropped: the extra
                // warp-uniform branch costs more than the ~11 select/compare instructions per element it saves)
                cl_elems(x[s], m[s], i, j0, col, i0, v[s], w[s], u[s], cv, cw, cu, z[s], tj);
            }
            // halving butterfly: kKT values x 32 lanes -> lane 32 q / kKT holds the total of column q
            {
                cplx kp;
                if constexpr (kKT == 4) {
                    const bool hi = (lane & 16) != 0, b8 = (lane & 8) != 0;
                    const cplx s0 = hi ? tj[0] : tj[2], s1 = hi ? tj[1] : tj[3];
                    cplx k0 = hi ? tj[2] : tj[0], k1 = hi ? tj[3] : tj[1];
                    k0.x += __shfl_xor_sync(0xffffffffu, s0.x, 16); k0.y += __shfl_xor_sync(0xffffffffu, s0.y, 16);
                    k1.x += __shfl_xor_sync(0xffffffffu, s1.x, 16); k1.y += __shfl_xor_sync(0xffffffffu, s1.y, 16);
                    const cplx snd = b8 ? k0 : k1;
                    kp = b8 ? k1 : k0;
                    kp.x += __shfl_xor_sync(0xffffffffu, snd.x, 8); kp.y += __shfl_xor_sync(0xffffffffu, snd.y, 8);
                } else {
                    static_assert(kKT == 2 || kKT == 4, "butterfly written for 2 or 4 columns per trip");
                    const bool hi = (lane & 16) != 0;
                    const cplx snd = hi ? tj[0] : tj[kKT - 1];
                    kp = hi ? tj[kKT - 1] : tj[0];
                    kp.x += __shfl_xor_sync(0xffffffffu, snd.x, 16); kp.y += __shfl_xor_sync(0xffffffffu, snd.y, 16);
                    kp.x += __shfl_xor_sync(0xffffffffu, kp.x, 8); kp.y += __shfl_xor_sync(0xffffffffu, kp.y, 8);
                }
#pragma unroll
                for (int o = 4; o > 0; o >>= 1) {
                    kp.x += __shfl_xor_sync(0xffffffffu, kp.x, o); kp.y += __shfl_xor_sync(0xffffffffu, kp.y, o);
                }
                const int idx = lane / (32 / kKT);
                if ((lane & (32 / kKT - 1)) == 0 && jl + idx < nc) tpart[wp * ncw + jl + idx] = kp;
            }
        }
        for (int q = jl + lane; q < nc; q += 32) tpart[wp * ncw + q] = mk(0.0, 0.0);   // columns beyond this warp's rows
        if (owner) {
            // the export stores were issued before the pass: the fence is cheap by now.  One token per warp and
            // receiver on phase 1: nobody reads the ring before every exporting warp has fenced.
            __threadfence();
            __syncwarp();
            if (lane < kCl) cl_st_async(cl_mapa(tok_a + 8u * (unsigned)wp, lane), 1.0, cl_mapa(mbar1, lane));
        }
        __syncthreads();

        // ================= [C] contributions to y = A v: reduce-scatter through DSMEM =================
        // Rows [rho RS, (rho+1) RS) are summed by CTA rho, so a warp's 32 consecutive rows go to at most two
        // destinations as contiguous segments (scattered 16-byte remote stores cost ~6 cycles each).
        double qp = 0.0;
#pragma unroll
        for (int s = 0; s < kClR; ++s) {
            const int i = row[s];
            if (i >= c + 1 && i < n) {
                cplx y = z[s];
                if ((i & (kCl - 1)) == r) {
                    const int slot = i >> 4;
#pragma unroll
                    for (int k = 0; k < kClWarps; ++k) y = y + tpart[k * ncw + slot];
                }
                qp += u[s].x * y.x + u[s].y * y.y;               // Re(conj(u_i) y_i): v^H A v is real
                cl_st_async(cl_mapa(rbuf_a + 16u * (unsigned)(r * RSP + dslot[s]), dest[s]), y, cl_mapa(mbar1, dest[s]));
            }
        }
        qp = warp_sum(qp);
        if (lane == 0) s_red[kRedQ + wp] = qp;
        __syncthreads();
        cl_wait(mbar1, c & 1);                                    // every contribution to my rows has landed
        if (tid == 0) cl_arm(mbar1, bytes_r(c + 1));
        if (tid < kCl) {
            // the partial v^H y is needed only with w, so it rides on phase 2; it is sent AFTER this CTA completed
            // phase 1, which makes "a peer completed phase 2 of step c" imply "I completed phase 1 of step c":
            // nothing of step c+1 can reach an mbarrier that is still in step c (see also the tokens below)
            double q = 0.0;
#pragma unroll
            for (int k = 0; k < kClWarps; ++k) q += s_red[kRedQ + k];
            cl_st_async(cl_mapa(sq_a + 8u * (unsigned)((c & 1) * kCl + r), tid), q, cl_mapa(mbar2, tid));
        }

        // ================= [D] sum the contributions of my rows, broadcast tau y =================
        const cplx *rawc = p.raw + (size_t)((c + 1) & 1) * lda;
#pragma unroll
        for (int s = 0; s < kClR; ++s) raw[s] = (row[s] >= c + 1 && row[s] < n) ? ldcg_(&rawc[row[s]]) : mk(0.0, 0.0);   // L2: the ring is rewritten every other step
        {
            // slot t = tid / 4 (row i = r RS + t); the four threads of a slot sum four contributions each and
            // send tau y_i to four of the 16 CTAs each
            const int t = tid >> 2, part = tid & 3;
            const int i = r * RS + t;
            const bool on = (t < RS && i >= c + 1 && i < n);      // uniform over the four threads of a slot
            cplx y = mk(0.0, 0.0);
            if (on) {
#pragma unroll
                for (int k = 0; k < 4; ++k) y = y + rbuf[(4 * part + k) * RSP + t];
            }
            y.x += __shfl_xor_sync(0xffffffffu, y.x, 1); y.y += __shfl_xor_sync(0xffffffffu, y.y, 1);
            y.x += __shfl_xor_sync(0xffffffffu, y.x, 2); y.y += __shfl_xor_sync(0xffffffffu, y.y, 2);
            if (on) {
                const cplx ty = tau * y;
#pragma unroll
                for (int k = 0; k < 4; ++k) cl_st_async(cl_mapa(wbuf_a + 16u * (unsigned)i, 4 * part + k), ty, cl_mapa(mbar2, 4 * part + k));
            }
        }
        cl_wait(mbar2, c & 1);                                    // all of tau y has landed
        // one 8-byte token to every CTA on phase 1 of the NEXT step: a peer completes that phase only after I have
        // completed phase 2 of this step, so its phase-2 traffic of step c+1 cannot arrive here early
        if (tid < kCl && c + 1 < n - 1) cl_st_async(cl_mapa(tok_a + 8u * (unsigned)(kClWarps + r), tid), 1.0, cl_mapa(mbar1, tid));
        double q = 0.0;
#pragma unroll
        for (int k = 0; k < kCl; ++k) q += s_q[(c & 1) * kCl + k];
        const double alphap = -0.5 * abs2(tau) * q;
        if (tid == 0) cl_arm(mbar2, bytes_w(c + 1));
#pragma unroll
        for (int s = 0; s < kClR; ++s) {
            const int i = row[s];
            v[s] = u[s];
            w[s] = (i >= c + 1 && i < n) ? wbuf[i] + alphap * u[s] : mk(0.0, 0.0);
        }
        wc = wbuf[c + 1] + alphap * mk(1.0, 0.0);
    }
}

// ---------------------------------------------------------------- host side
int g_cluster_tridiag = 1;
static int g_cl_init_dev = -1;
static int g_cl_ok = 0;            // 1: 16-CTA clusters with the maximum shared memory are launchable on this device

static size_t cl_smem_max(int n) {
    size_t m = 0;
    for (int r = 0; r < kCl; ++r) { const size_t t = cl_smem(n, r).total; if (t > m) m = t; }
    return m;
}

int tridiag_cluster_init() {
    int dev = 0;
    cudaGetDevice(&dev);
    if (g_cl_init_dev == dev) return 0;
    g_cl_ok = 0;
    int maxsm = 0;
    cudaDeviceGetAttribute(&maxsm, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (cudaFuncSetAttribute(tridiag_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, maxsm) == cudaSuccess &&
        cudaFuncSetAttribute(tridiag_cluster_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(kCl); cfg.blockDim = dim3(kClThreads); cfg.dynamicSmemBytes = (size_t)maxsm;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = kCl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int nclusters = 0;
        if (cudaOccupancyMaxActiveClusters(&nclusters, tridiag_cluster_kernel, &cfg) == cudaSuccess && nclusters >= 1) g_cl_ok = 1;
    }
    cudaGetLastError();            // a device without 16-CTA clusters is not an error: the grid-wide path serves it
    g_cl_init_dev = dev;
    return 0;
}

// device-independent: the packed lower triangle of an n x n block fits in 16 x 227 KB (hpsd_workspace_size's bound)
int tridiag_cluster_size_ok(int n) { return n >= kCl && n <= kClMaxN && cl_smem_max(n) <= (size_t)232448; }

// 1 when a block of size n is served by the cluster kernel on this device
int tridiag_cluster_fits(int n) {
    tridiag_cluster_init();
    if (!g_cl_ok || n < kCl || n > kClMaxN) return 0;
    int dev = 0, maxsm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&maxsm, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    return cl_smem_max(n) <= (size_t)maxsm;
}

// S1 + S2 + S3 in one launch.  w.W (ldw x kNB) hosts the raw-column ring.
int launch_tridiag_cluster(const TridiagWs &w, const double *in, const double *sub, cudaStream_t st, int *nf, int f32) {
    ClusterArgs a;
    a.n = w.n; a.lda = w.lda; a.in = in; a.sub = sub; a.A = w.A; a.raw = w.W; a.d = w.d; a.e = w.e; a.tau = w.tau; a.nf = nf; a.f32 = f32;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(kCl); cfg.blockDim = dim3(kClThreads); cfg.dynamicSmemBytes = cl_smem_max(w.n); cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = kCl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    prof_begin(ST_PANEL, st);
    const cudaError_t e = cudaLaunchKernelEx(&cfg, tridiag_cluster_kernel, a);
    prof_end(ST_PANEL, st);
    g_launches++;
    return e == cudaSuccess ? 0 : HPSD_ECUDA_;
}

}  // namespace hpsd
