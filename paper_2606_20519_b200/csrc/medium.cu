// medium.cu -- S10 of SURVEY.md §8(a): medium blocks (jacobi_max_n < n <= kMediumMaxN), batched.
// One CTA per matrix, the whole matrix in shared memory, one kernel from svec to svec:
//   S1 unpack -> Householder tridiagonalisation (unblocked, rank-2 updates) -> Q formed IN PLACE over the
//   reflectors -> implicit QL with Wilkinson shift on (d, e), the real rotations applied to the complex
//   columns of Q -> S6 clamp/scale -> S7 W W^H -> S8 pack.
// Operation defined at PAPER.md:1536; layout Eq. (D10) PAPER.md:1220-1222.
//
// The serial part of QL (the rotation parameters, ~1.7 n^2/2 of them, each a dependent chain of about
// 150 cycles) is produced by ONE thread running ahead through a ring buffer in shared memory; the other
// warps apply the rotations to the rows of Q as the batches become ready.  The generator depends only on
// (d, e), never on Q, so the two never wait on each other except through the ring.
//
// Only one n x n complex array is needed (105 KB at n = 81: two CTAs per SM, so 256 matrices are one wave).
#include "kernels.h"
#include "large.h"

namespace hpsd {

constexpr int kMedThreads = 256;
constexpr int kRing = 128;                 // rotations in flight between generator and appliers
constexpr int kMedMaxIter = 60;            // QL iterations per eigenvalue before giving up

struct MedSmem {
    cplx *A;            // n x ld: matrix -> reflectors -> Q
    cplx *tau;          // n
    cplx *x;            // n : Householder vector / work row
    cplx *y;            // n : A v, then w
    cplx *x2, *y2;      // n each: second parity of (v, w) in the fused tridiagonalisation
    double *d, *e;      // n each
    double *rc, *rs;    // kRing each
    int *ri;            // kRing : column index i of the rotation (acts on columns i, i+1)
    double *red;        // 32
    volatile int *ctl;  // [0] produced, [1] done flag, [2] info, [3] consumed (min over appliers, lazily)
};

__host__ __device__ inline int med_ld(int n) { return n | 1; }

__host__ __device__ inline size_t med_smem_bytes(int n) {
    const size_t ld = med_ld(n);
    return sizeof(cplx) * ((size_t)n * ld + 5 * (size_t)n) + sizeof(double) * (2 * (size_t)n + 2 * kRing + 32) +
           sizeof(int) * (kRing + 16) + 64;
}

__device__ __forceinline__ MedSmem med_carve(unsigned char *base, int n) {
    MedSmem sm;
    const int ld = med_ld(n);
    sm.A = reinterpret_cast<cplx *>(base);
    sm.tau = sm.A + (size_t)n * ld;
    sm.x = sm.tau + n;
    sm.y = sm.x + n;
    sm.x2 = sm.y + n;
    sm.y2 = sm.x2 + n;
    sm.d = reinterpret_cast<double *>(sm.y2 + n);
    sm.e = sm.d + n;
    sm.rc = sm.e + n;
    sm.rs = sm.rc + kRing;
    sm.red = sm.rs + kRing;
    sm.ri = reinterpret_cast<int *>(sm.red + 32);
    sm.ctl = sm.ri + kRing;
    return sm;
}

// block-wide sum of one double (every thread gets the result); red has >= 9 entries
__device__ __forceinline__ double block_sum(double v, double *red) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < kMedThreads / 32; ++w) t += red[w];
    return t;
}
__device__ __forceinline__ cplx block_sum(cplx v, double *red) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5] = v.x; red[8 + (threadIdx.x >> 5)] = v.y; }
    __syncthreads();
    cplx t = mk(0.0, 0.0);
#pragma unroll
    for (int w = 0; w < kMedThreads / 32; ++w) { t.x += red[w]; t.y += red[8 + w]; }
    return t;
}

// zlarfg semantics (same conventions as tridiag.cu): H^H (alpha; x) = (beta; 0), H = I - tau v v^H, v = (1; scale x)
__device__ __forceinline__ void med_householder(cplx alpha, double xnorm2, double &beta, cplx &tau, cplx &scale) {
    if (xnorm2 == 0.0 && alpha.y == 0.0) {
        beta = alpha.x; tau = mk(0.0, 0.0); scale = mk(0.0, 0.0);
    } else {
        // rsqrt + one Newton step and one reciprocal instead of DSQRT + two DDIV on the per-column dependent chain
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

// ---- phase 1: A (full Hermitian, shared memory) -> real tridiagonal (d, e), reflectors in the lower part
// One pass over the trailing block per column: the rank-2 update of step c-1 is applied to an element right before the
// element is used in the mat-vec of step c (as in tridiag_cluster.cu), so the block is read once and written once per
// column instead of read twice and written once, with four block barriers per column instead of five.  (v, w) of two
// consecutive steps live in two parities of shared-memory vectors; column c itself is brought up to date on the fly.
__device__ void med_tridiagonalize(const MedSmem &sm, int n, int ld) {
    cplx *A = sm.A;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int r = tid; r < n; r += kMedThreads) { sm.x[r] = sm.y[r] = sm.x2[r] = sm.y2[r] = mk(0.0, 0.0); }
    __syncthreads();
    for (int c = 0; c < n - 1; ++c) {
        cplx *X = (c & 1) ? sm.x2 : sm.x, *W = (c & 1) ? sm.y2 : sm.y;                  // v_c, w_c
        const cplx *Vp = (c & 1) ? sm.x : sm.x2, *Wp = (c & 1) ? sm.y : sm.y2;          // v_{c-1}, w_{c-1} (zero at c = 0)
        // [1] column c of the current matrix (one row per thread: n <= 116), its norm, alpha and d_c through ONE barrier
        cplx a = mk(0.0, 0.0);
        const int rc = c + tid;
        if (rc < n) {
            a = A[(size_t)c * ld + rc];
            const cplx vr = Vp[rc], wr = Wp[rc], vc = Vp[c], wc = Wp[c];
            a.x -= vr.x * wc.x + vr.y * wc.y + wr.x * vc.x + wr.y * vc.y;
            a.y -= vr.y * wc.x - vr.x * wc.y + wr.y * vc.x - wr.x * vc.y;
        }
        double S = (rc >= c + 2 && rc < n) ? abs2(a) : 0.0;
        S = warp_sum(S);
        if (lane == 0) sm.red[warp] = S;
        if (tid == 1) { sm.red[16] = a.x; sm.red[17] = a.y; }
        if (tid == 0) sm.red[18] = a.x;
        __syncthreads();
        S = 0.0;
#pragma unroll
        for (int k = 0; k < kMedThreads / 32; ++k) S += sm.red[k];
        const cplx alpha = mk(sm.red[16], sm.red[17]);
        double beta; cplx tau, scale;
        med_householder(alpha, S, beta, tau, scale);
        if (tid == 0) { sm.d[c] = sm.red[18]; sm.e[c] = beta; sm.tau[c] = tau; }
        // [2] v_c into its vector and over column c (the reflector the back-transformation reads)
        if (rc >= c + 1 && rc < n) {
            const cplx v = (rc == c + 1) ? mk(1.0, 0.0) : scale * a;
            X[rc] = v;
            A[(size_t)c * ld + rc] = v;
        }
        __syncthreads();
        // [3] fused pass over the trailing block: A22 -= v' w'^H + w' v'^H (step c-1), y = A22 v (step c).
        // 64 rows per round (8 per warp), 4 column classes per row (lane >> 3), reduced by shuffles
        cplx q = mk(0.0, 0.0);
        for (int base = 0; base < n; base += 64) {
            const int r = base + (lane & 7) + 8 * warp;
            if (base + 63 < c + 1) continue;                                            // block-uniform
            const bool rok = (r >= c + 1 && r < n);
            cplx acc = mk(0.0, 0.0);
            if (rok) {
                const cplx vr = Vp[r], wr = Wp[r];
                for (int j = c + 1 + (lane >> 3); j < n; j += 4) {
                    const cplx vj = Vp[j], wj = Wp[j];
                    cplx e = A[(size_t)j * ld + r];
                    e.x -= vr.x * wj.x + vr.y * wj.y + wr.x * vj.x + wr.y * vj.y;
                    e.y -= vr.y * wj.x - vr.x * wj.y + wr.y * vj.x - wr.x * vj.y;
                    if (r == j) e.y = 0.0;
                    A[(size_t)j * ld + r] = e;
                    cfma(acc, e, X[j]);
                }
            }
            acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 8);  acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 8);
            acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 16); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 16);
            if (rok && lane < 8) {
                W[r] = acc;                                     // y_r for now
                cfma_conj(q, X[r], acc);                        // conj(v_r) y_r
            }
        }
        // v^H y (real): partials in red[8..15], one barrier, which also publishes y
        {
            const double qs = warp_sum(q.x);
            if (lane == 0) sm.red[8 + warp] = qs;
        }
        __syncthreads();
        // [4] w = tau y - 1/2 |tau|^2 (v^H y) v
        double qsum = 0.0;
#pragma unroll
        for (int k = 0; k < kMedThreads / 32; ++k) qsum += sm.red[8 + k];
        const double alphap = -0.5 * abs2(tau) * qsum;      // v^H A v is real
        if (rc >= c + 1 && rc < n) W[rc] = tau * W[rc] + alphap * X[rc];
        __syncthreads();
    }
    // the update of the last step on the last diagonal entry: v_{n-1} = 1 there
    if (tid == 0) {
        double dl = A[(size_t)(n - 1) * ld + n - 1].x;
        if (n >= 2) { const cplx *Wl = ((n - 2) & 1) ? sm.y2 : sm.y; dl -= 2.0 * Wl[n - 1].x; }
        sm.d[n - 1] = dl; sm.e[n - 1] = 0.0; sm.tau[n - 1] = mk(0.0, 0.0);
    }
    __syncthreads();
}

// ---- phase 2: Q = H_0 H_1 ... H_{n-2} formed in place over the reflectors (backward accumulation)
__device__ void med_form_q(const MedSmem &sm, int n, int ld) {
    cplx *A = sm.A;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int k = n - 2; k >= 0; --k) {
        const cplx tau = sm.tau[k];
        const int m2 = n - k - 2;                           // size of the already formed block B = A[k+2:, k+2:]
        // z_j = sum_{r >= k+2} conj(x_r) B[r, j],  x = A[k+2:, k]
        for (int base = 0; base < m2; base += 64) {
            const int j = k + 2 + base + (lane & 7) + 8 * warp;
            cplx acc = mk(0.0, 0.0);
            if (j < n)
                for (int r = k + 2 + (lane >> 3); r < n; r += 4) cfma_conj(acc, A[(size_t)k * ld + r], A[(size_t)j * ld + r]);
            acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 8);  acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 8);
            acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 16); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 16);
            if (j < n && lane < 8) sm.y[j] = acc;
        }
        __syncthreads();
        const cplx mtau = mk(-tau.x, -tau.y);
        const int m1 = m2 + 1;                              // block C = A[k+1:, k+1:]
        for (int e = tid; e < m1 * m1; e += kMedThreads) {
            const int rr = e % m1, jj = e / m1;
            const int r = k + 1 + rr, j = k + 1 + jj;
            cplx v;
            if (rr == 0 && jj == 0) v = mk(1.0 - tau.x, -tau.y);
            else if (rr == 0) v = mtau * sm.y[j];
            else if (jj == 0) v = mtau * A[(size_t)k * ld + r];
            else v = A[(size_t)j * ld + r] + (mtau * A[(size_t)k * ld + r]) * sm.y[j];
            A[(size_t)j * ld + r] = v;
        }
        __syncthreads();
    }
    for (int e = tid; e < n; e += kMedThreads) {
        A[(size_t)e * ld] = mk(e == 0 ? 1.0 : 0.0, 0.0);    // row 0
        A[e] = mk(e == 0 ? 1.0 : 0.0, 0.0);                 // column 0
    }
    __syncthreads();
}

// ---- phase 3: implicit QL (tql2 scheme).  Thread 0 generates the rotations, warps 1.. apply them to Q.
// ctl[0] = rotations produced, ctl[1] = generator finished, ctl[2] = failure flag, ctl[4 + w] = consumed by warp w
__device__ void med_ql_generate(const MedSmem &sm, int n) {
    double *d = sm.d, *e = sm.e;
    volatile int *ctl = sm.ctl;
    int produced = 0, safe = kRing;         // slots below `safe` may be written without asking the appliers
    double an = 0.0;
    for (int k = 0; k < n; ++k) an = fmax(an, fabs(d[k]) + fabs(e[k]));
    bool fail = false;
    for (int l = 0; l < n && !fail; ++l) {
        int iter = 0;
        for (;;) {
            int mm;
            for (mm = l; mm < n - 1; ++mm) {
                const double s = fabs(d[mm]) + fabs(d[mm + 1]);
                if (fabs(e[mm]) <= kEps * s || fabs(e[mm]) <= kEps * an) break;
            }
            if (mm == l) break;
            if (++iter > kMedMaxIter) { fail = true; break; }
            double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
            double r = sqrt(g * g + 1.0);
            if (!(fabs(g) < 1e150)) r = fabs(g);
            g = d[mm] - d[l] + e[l] / (g + copysign(r, g));
            double s = 1.0, c = 1.0, p = 0.0;
            int i;
            bool under = false;
            // d[i+1] at step i is the (unchanged) d[i] read at step i+1: carried in a register;
            // e[i], d[i] of the next step are loaded before the dependent chain of this one
            double dnext = d[mm];
            double ei = e[mm - 1], di = d[mm - 1];
            for (i = mm - 1; i >= l; --i) {
                const double f = s * ei, b = c * ei;
                const double dcur = di;
                if (i > l) { ei = e[i - 1]; di = d[i - 1]; }
                const double h2 = fma(f, f, g * g);
                double r, ir;
                if (h2 > 1e-280 && h2 < 1e280) {
                    ir = rsqrt(h2);
                    ir = ir * fma(-0.5 * h2 * ir, ir, 1.5);     // one Newton step: 1/sqrt(h2) to working precision
                    r = h2 * ir;
                } else {
                    r = hypot(f, g);
                    if (r == 0.0) { e[i + 1] = 0.0; d[i + 1] = dnext - p; e[mm] = 0.0; under = true; break; }
                    ir = 1.0 / r;
                }
                e[i + 1] = r;
                s = f * ir; c = g * ir;
                g = dnext - p;
                r = (dcur - g) * s + 2.0 * c * b;
                p = s * r;
                d[i + 1] = g + p;
                g = c * r - b;
                dnext = dcur;
                // emit rotation (i, c, s)
                if (produced >= safe) {
                    __threadfence_block();
                    ctl[0] = produced;                     // let the appliers drain everything produced so far
                    int mn;
                    do {
                        mn = ctl[4 + 1];
                        for (int w = 2; w < kMedThreads / 32; ++w) mn = min(mn, ctl[4 + w]);
                    } while (produced - mn >= kRing);
                    safe = mn + kRing;
                }
                const int slot = produced & (kRing - 1);
                sm.ri[slot] = i; sm.rc[slot] = c; sm.rs[slot] = s;
                ++produced;
                if ((produced & 15) == 0) { __threadfence_block(); ctl[0] = produced; }
            }
            if (!under) { d[l] -= p; e[l] = g; e[mm] = 0.0; }
            __threadfence_block();
            ctl[0] = produced;
        }
    }
    __threadfence_block();
    ctl[0] = produced;
    if (fail) ctl[2] = 1;
    __threadfence_block();
    ctl[1] = 1;
}

__device__ void med_ql_apply(const MedSmem &sm, int n, int ld) {
    volatile int *ctl = sm.ctl;
    const int warp = threadIdx.x >> 5;
    const int a = threadIdx.x - 32;                   // applier index: (row, component) pairs, 2n of them
    const int na = kMedThreads - 32;
    double *Z = reinterpret_cast<double *>(sm.A);
    int consumed = 0;
    const int lane = threadIdx.x & 31;
    for (;;) {
        int done = 0, avail = 0;
        if (lane == 0) { done = ctl[1]; avail = ctl[0]; }   // done first: if it is set, avail is final
        done = __shfl_sync(0xffffffffu, done, 0);
        avail = __shfl_sync(0xffffffffu, avail, 0);
        if (avail == consumed) {
            if (done) break;
            continue;
        }
        __threadfence_block();
        for (; consumed < avail; ++consumed) {
            const int slot = consumed & (kRing - 1);
            const int i = sm.ri[slot];
            const double c = sm.rc[slot], s = sm.rs[slot];
            for (int t = a; t < 2 * n; t += na) {
                double *z0 = Z + 2 * (size_t)i * ld + t, *z1 = z0 + 2 * (size_t)ld;
                const double q = *z0, f = *z1;
                *z1 = s * q + c * f;
                *z0 = c * q - s * f;
            }
        }
        __syncwarp();
        if (lane == 0) ctl[4 + warp] = consumed;
    }
}


__global__ void __launch_bounds__(kMedThreads) hhql_project_kernel(int n, const long long *__restrict__ offs,
                                                                   SvecIo io,
                                                                   int *__restrict__ info, const int *__restrict__ info_idx) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ld = med_ld(n);
    MedSmem sm = med_carve(smem_raw, n);
    cplx *A = sm.A;
    const int tid = threadIdx.x;
    const size_t base = (size_t)offs[blockIdx.x];

    // ---- S1: unpack into shared memory, both triangles
    int bad = 0;
    for (int t = tid; t < n * n; t += kMedThreads) {
        const int j = t / n, i = t % n;
        if (i < j) continue;
        const size_t c = base + svec_col_off(n, j);
        if (i == j) { const double d = io_load(io, c); bad |= nonfinite(d); A[(size_t)j * ld + i] = mk(d, 0.0); }
        else {
            const int k = i - j - 1;
            const cplx v = mk(io_load(io, c + 1 + 2 * k) / kSqrt2, io_load(io, c + 2 + 2 * k) / kSqrt2);
            bad |= nonfinite(v.x) | nonfinite(v.y);
            A[(size_t)j * ld + i] = v;
            A[(size_t)i * ld + j] = conj_(v);
        }
    }
    if (tid < 16) sm.ctl[tid] = 0;
    if (__syncthreads_or(bad)) {               // NaN / Inf in the block: all-NaN output, info = 2
        io_fill_nan(io, base, n, tid, kMedThreads);
        if (info != nullptr && tid == 0) info[info_idx[blockIdx.x]] = kInfoNonFinite;
        return;
    }

    med_tridiagonalize(sm, n, ld);
    med_form_q(sm, n, ld);

    if (tid == 0) med_ql_generate(sm, n);
    else if (tid >= 32) med_ql_apply(sm, n, ld);
    __syncthreads();
    if (info != nullptr && tid == 0) info[info_idx[blockIdx.x]] = sm.ctl[2] ? 4 : 0;

    // ---- S6: clamp, W = Q_+ diag(sqrt(lambda_+)); the positive columns are scaled in place
    int *poslist = reinterpret_cast<int *>(sm.x);            // x, y are dead now (n cplx >= n ints)
    if (tid == 0) {
        int k = 0;
        for (int l = 0; l < n; ++l)
            if (sm.d[l] > 0.0) poslist[k++] = l;
        sm.ctl[3] = k;
    }
    __syncthreads();
    const int kpos = sm.ctl[3];
    for (int t = tid; t < kpos * n; t += kMedThreads) {
        const int l = poslist[t / n], i = t % n;
        A[(size_t)l * ld + i] = sqrt(sm.d[l]) * A[(size_t)l * ld + i];
    }
    __syncthreads();
    // ---- S7 + S8: lower triangle of W W^H straight into the svec
    for (int t = tid; t < n * n; t += kMedThreads) {
        const int j = t / n, i = t % n;
        if (i < j) continue;
        cplx acc = mk(0.0, 0.0);
        for (int k = 0; k < kpos; ++k) {
            const int l = poslist[k];
            const cplx a = A[(size_t)l * ld + i], b = A[(size_t)l * ld + j];
            acc.x = fma(a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
            acc.y = fma(a.y, b.x, acc.y); acc.y = fma(-a.x, b.y, acc.y);
        }
        const size_t c = base + svec_col_off(n, j);
        if (i == j) io_store(io, c, acc.x);
        else {
            const int k = i - j - 1;
            io_store(io, c + 1 + 2 * k, kSqrt2 * acc.x);
            io_store(io, c + 2 + 2 * k, kSqrt2 * acc.y);
        }
    }
}

// =====================================================================================================
// Batched divide-and-conquer variant of S10 (n <= kMedDcMaxN): the serial QL generator above costs ~480 cycles
// per rotation; here the tridiagonal eigenproblems of a whole group of equal-size blocks are solved by the
// device-side D&C of stedc.cu, the group being ONE virtual tridiagonal of size blk 2^d0 whose top d0 levels are
// never merged.  Kernel A: unpack + Householder tridiagonalisation per CTA (reflectors, tau, d, e to global);
// stedc; kernel C: W = Q Z_+ diag(sqrt(lambda_+)) by applying the reflectors to the kept columns in shared
// memory, then HERK + pack.
// =====================================================================================================
struct MedDcWs {
    int n, count, B, ld;          // block size, blocks, padded batch (power of two), leading dimension of the reflectors
    cplx *Ar;                     // count x (n x ld): reflectors (column c rows c+1.. = v_c)
    cplx *tau;                    // B n
    double *d, *e;                // B n
    int *info;                    // 1: D&C failure flag of the group
    StedcWs s;
};

__global__ void __launch_bounds__(kMedThreads) meddc_tridiag_kernel(int n, const long long *__restrict__ offs, SvecIo io, MedDcWs w) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ld = med_ld(n);
    MedSmem sm = med_carve(smem_raw, n);
    cplx *A = sm.A;
    const int tid = threadIdx.x, t = blockIdx.x;
    const size_t base = (size_t)offs[t];
    int bad = 0;
    for (int q = tid; q < n * n; q += kMedThreads) {
        const int j = q / n, i = q % n;
        if (i < j) continue;
        const size_t c = base + svec_col_off(n, j);
        if (i == j) { const double d = io_load(io, c); bad |= nonfinite(d); A[(size_t)j * ld + i] = mk(d, 0.0); }
        else {
            const int k = i - j - 1;
            const cplx v = mk(io_load(io, c + 1 + 2 * k) / kSqrt2, io_load(io, c + 2 + 2 * k) / kSqrt2);
            bad |= nonfinite(v.x) | nonfinite(v.y);
            A[(size_t)j * ld + i] = v;
            A[(size_t)i * ld + j] = conj_(v);
        }
    }
    cplx *Ag = w.Ar + (size_t)t * n * w.ld;
    if (__syncthreads_or(bad)) {
        // NaN / Inf in the block: the group's divide & conquer gets a zero tridiagonal for it; tau[n-1] (always zero
        // otherwise) carries the flag to meddc_back_kernel, which writes the all-NaN output
        for (int q = tid; q < n * n; q += kMedThreads) { const int j = q / n, i = q % n; if (i > j) Ag[(size_t)j * w.ld + i] = mk(0.0, 0.0); }
        for (int i = tid; i < n; i += kMedThreads) {
            w.tau[(size_t)t * n + i] = (i == n - 1) ? mk(nan_(), 0.0) : mk(0.0, 0.0);
            w.d[(size_t)t * n + i] = 0.0;
            w.e[(size_t)t * n + i] = 0.0;
        }
        return;
    }
    med_tridiagonalize(sm, n, ld);
    for (int q = tid; q < n * n; q += kMedThreads) {
        const int j = q / n, i = q % n;
        if (i > j) Ag[(size_t)j * w.ld + i] = A[(size_t)j * ld + i];
    }
    for (int i = tid; i < n; i += kMedThreads) {
        w.tau[(size_t)t * n + i] = sm.tau[i];
        w.d[(size_t)t * n + i] = sm.d[i];
        w.e[(size_t)t * n + i] = sm.e[i];
    }
}

__global__ void __launch_bounds__(kMedThreads) meddc_back_kernel(int n, const long long *__restrict__ offs, SvecIo io, MedDcWs w,
                                                                 const double *__restrict__ lam, const double *__restrict__ Z, int ldz,
                                                                 int *__restrict__ info, const int *__restrict__ info_idx) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ld = med_ld(n);
    // Only the kept eigenvectors live in shared memory; the reflectors stream from L2 (52 KB per matrix, each column read
    // once), two at a time, one pair ahead in registers.  Half the shared memory of the first version (which also held
    // the n x n reflector block): two CTAs per SM, so the 256 matrices of config 2 are resident at once instead of in two waves.
    cplx *Wm = reinterpret_cast<cplx *>(smem_raw);              // n x ld kept eigenvectors
    cplx *vb = Wm + (size_t)n * ld;                              // 2 x n : the two reflectors in work
    cplx *tau = vb + 2 * n;                                      // n
    cplx *sv = tau + n;                                          // 2 x n : x_k, x_{k-1}
    double *lm = reinterpret_cast<double *>(sv + 2 * n) + 16;    // n (behind the 16 reduction slots)
    __shared__ int s_p0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, t = blockIdx.x;
    const cplx *Ag = w.Ar + (size_t)t * n * w.ld;
    for (int i = tid; i < n; i += kMedThreads) { tau[i] = w.tau[(size_t)t * n + i]; lm[i] = lam[(size_t)t * n + i]; }
    __syncthreads();
    if (tau[n - 1].x != tau[n - 1].x) {        // flag of meddc_tridiag_kernel: non-finite input (block-uniform)
        io_fill_nan(io, (size_t)offs[t], n, tid, kMedThreads);
        if (info != nullptr && tid == 0) info[info_idx[t]] = kInfoNonFinite;
        return;
    }
    if (tid == 0) {
        int lo = 0, hi = n;                                      // eigenvalues ascending: first index with lam > 0
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (lm[mid] > 0.0) hi = mid; else lo = mid + 1; }
        s_p0 = lo;
        if (info != nullptr) info[info_idx[t]] = (w.info != nullptr && *w.info) ? *w.info : 0;
    }
    __syncthreads();
    const int p0 = s_p0, kpos = n - p0;
    // S6: W = Z_+ diag(sqrt(lambda_+)), real -> complex
    const double *Zt = Z + (size_t)t * n * ldz;
    for (int j = warp; j < kpos; j += kMedThreads / 32) {
        const double sq = sqrt(lm[p0 + j]);
        for (int r = lane; r < n; r += 32) Wm[(size_t)j * ld + r] = mk(sq * Zt[(size_t)(p0 + j) * ldz + r], 0.0);
    }
    __syncthreads();
    // S5: W <- H_0 H_1 ... H_{n-2} W, last reflector first, TWO reflectors per pass over W:
    //   H_{k-1} H_k W = W - v_k x_k - v_{k-1} x_{k-1},  x_k = tau_k v_k^H W,  x_{k-1} = tau_{k-1} (v_{k-1}^H W - (v_{k-1}^H v_k) x_k),
    // so W is read twice and written once per PAIR (the kernel is bound by shared-memory bandwidth) with three block
    // barriers per pair.  The next pair is on its way from L2 (one row per thread, in registers) while this one is applied.
    cplx *v0 = vb, *v1 = vb + n;                                 // v_k, v_{k-1}: rows >= k, zero where the reflector has no entry
    double *red = reinterpret_cast<double *>(sv + 2 * n);        // 16 : partials of v_{k-1}^H v_k
    auto fetch = [&](int k, cplx &a, cplx &b) {                  // row tid of reflectors k and k-1
        a = mk(0.0, 0.0); b = mk(0.0, 0.0);
        if (tid < n && k >= 0) {
            if (tid >= k + 1) a = Ag[(size_t)k * w.ld + tid];
            if (k >= 1 && tid >= k) b = Ag[(size_t)(k - 1) * w.ld + tid];
        }
    };
    cplx pa, pb;
    fetch(n - 2, pa, pb);
    for (int k = n - 2; k >= 0; k -= 2) {
        const cplx tk = tau[k], tk1 = (k >= 1) ? tau[k - 1] : mk(0.0, 0.0);
        // [a] the pair into shared memory, v_{k-1}^H v_k, and the next pair's loads issued
        if (tid < n) { v0[tid] = pa; v1[tid] = pb; }
        {
            cplx gp = mk(0.0, 0.0);
            cfma_conj(gp, pb, pa);
            gp = warp_sum(gp);
            if (lane == 0) { red[2 * warp] = gp.x; red[2 * warp + 1] = gp.y; }
        }
        fetch(k - 2, pa, pb);
        __syncthreads();
        cplx g = mk(0.0, 0.0);
#pragma unroll
        for (int q = 0; q < kMedThreads / 32; ++q) { g.x += red[2 * q]; g.y += red[2 * q + 1]; }
        // [b] s_k = v_k^H W, s_{k-1} = v_{k-1}^H W per kept column: 8 columns per warp, 4 row classes per column
        for (int base = 0; base < kpos; base += 64) {
            const int j = base + (lane & 7) + 8 * warp;
            cplx a0 = mk(0.0, 0.0), a1 = mk(0.0, 0.0);
            if (j < kpos)
                for (int r = k + (lane >> 3); r < n; r += 4) {
                    const cplx x = Wm[(size_t)j * ld + r];
                    cfma_conj(a0, v0[r], x);
                    cfma_conj(a1, v1[r], x);
                }
            a0.x += __shfl_xor_sync(0xffffffffu, a0.x, 8);  a0.y += __shfl_xor_sync(0xffffffffu, a0.y, 8);
            a1.x += __shfl_xor_sync(0xffffffffu, a1.x, 8);  a1.y += __shfl_xor_sync(0xffffffffu, a1.y, 8);
            a0.x += __shfl_xor_sync(0xffffffffu, a0.x, 16); a0.y += __shfl_xor_sync(0xffffffffu, a0.y, 16);
            a1.x += __shfl_xor_sync(0xffffffffu, a1.x, 16); a1.y += __shfl_xor_sync(0xffffffffu, a1.y, 16);
            if (j < kpos && lane < 8) {
                const cplx xk = tk * a0;
                sv[j] = xk;
                sv[n + j] = tk1 * (a1 - g * xk);
            }
        }
        __syncthreads();
        // [c] W[r, j] -= v_k[r] x_k[j] + v_{k-1}[r] x_{k-1}[j] : lane = row, warp = column class
        for (int rb = k; rb < n; rb += 32) {
            const int r = rb + lane;
            if (r < n) {
                const cplx va = v0[r], vc = v1[r];
                for (int j = warp; j < kpos; j += kMedThreads / 32) {
                    const cplx xa = sv[j], xb = sv[n + j];
                    cplx x = Wm[(size_t)j * ld + r];
                    x.x -= va.x * xa.x - va.y * xa.y + vc.x * xb.x - vc.y * xb.y;
                    x.y -= va.x * xa.y + va.y * xa.x + vc.x * xb.y + vc.y * xb.x;
                    Wm[(size_t)j * ld + r] = x;
                }
            }
        }
        __syncthreads();
    }
    // S7 + S8
    const size_t obase = (size_t)offs[t];
    for (int q = tid; q < n * n; q += kMedThreads) {
        const int j = q / n, i = q % n;
        if (i < j) continue;
        cplx acc = mk(0.0, 0.0);
        for (int l = 0; l < kpos; ++l) {
            const cplx a = Wm[(size_t)l * ld + i], b = Wm[(size_t)l * ld + j];
            acc.x = fma(a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
            acc.y = fma(a.y, b.x, acc.y); acc.y = fma(-a.x, b.y, acc.y);
        }
        const size_t c = obase + svec_col_off(n, j);
        if (i == j) io_store(io, c, acc.x);
        else {
            const int k = i - j - 1;
            io_store(io, c + 1 + 2 * k, kSqrt2 * acc.x);
            io_store(io, c + 2 + 2 * k, kSqrt2 * acc.y);
        }
    }
}

static size_t meddc_back_smem(int n) {
    return sizeof(cplx) * ((size_t)n * med_ld(n) + 5 * (size_t)n) + sizeof(double) * (n + 16) + 64;
}

static int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }

// Carve the scratch of one group (base may be nullptr: size query).
static size_t meddc_carve(int n, int count, unsigned char *base, MedDcWs &w) {
    size_t off = 0;
    auto take = [&](size_t bytes) -> unsigned char * { unsigned char *p = base ? base + off : nullptr; off += align_up(bytes, 256); return p; };
    auto dbl = [&](size_t c) { return reinterpret_cast<double *>(take(sizeof(double) * c)); };
    auto itg = [&](size_t c) { return reinterpret_cast<int *>(take(sizeof(int) * c)); };
    const int B = next_pow2(count);
    int d0 = 0; while ((1 << d0) < B) ++d0;
    const size_t N = (size_t)B * n;
    const int ldz = (int)align_up((size_t)n, 8);
    w.n = n; w.count = count; w.B = B; w.ld = n;
    w.Ar = reinterpret_cast<cplx *>(take(sizeof(cplx) * (size_t)count * n * n));
    w.tau = reinterpret_cast<cplx *>(take(sizeof(cplx) * N));
    w.d = dbl(N); w.e = dbl(N);
    w.info = itg(4);
    StedcWs &s = w.s;
    s.n = (int)N; s.ldz = ldz; s.blk = n; s.d0 = d0; s.depth = d0 + stedc_depth(n);
    s.Za = dbl((size_t)ldz * N); s.Zb = dbl((size_t)ldz * N); s.Qw = dbl((size_t)ldz * N); s.U = dbl((size_t)ldz * N);
    s.lamA = dbl(N); s.lamB = dbl(N); s.dmod = dbl(N); s.es = dbl(N); s.scal = dbl(2 * (size_t)B);
    s.dt = dbl(N); s.zt = dbl(N); s.mu = dbl(N); s.lamroot = dbl(N); s.zhat = dbl(N); s.dval = dbl(N); s.rc = dbl(N); s.rs = dbl(N);
    s.org = itg(N); s.grow = itg(N); s.gsrc = itg(N); s.dcol = itg(N);
    s.dest_root = itg(N); s.dest_defl = itg(N); s.rp = itg(N); s.rq = itg(N);
    const size_t maxnodes = (size_t)1 << (s.depth > 0 ? s.depth - 1 : 0);
    s.nodeinfo = itg(8 * maxnodes);
    s.rho = dbl(maxnodes);
    s.info = w.info;
    return off;
}

size_t meddc_ws_bytes(int n, int count) { MedDcWs w; return meddc_carve(n, count, nullptr, w); }

int launch_meddc_project(int n, int count, const long long *offs_dev, const SvecIo &io, unsigned char *scratch,
                         int *info_dev, const int *info_idx_dev, cudaStream_t st) {
    if (count <= 0) return 0;
    if (n < 2 || n > kMedDcMaxN || (long long)next_pow2(count) * n > kMaxLargeN * 64LL) return -1;
    MedDcWs w;
    meddc_carve(n, count, scratch, w);
    const size_t N = (size_t)w.B * n;
    if (cudaMemsetAsync(w.d, 0, sizeof(double) * N, st) != cudaSuccess) return HPSD_ECUDA_;   // padding blocks: zero matrices
    if (cudaMemsetAsync(w.e, 0, sizeof(double) * N, st) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaMemsetAsync(w.info, 0, sizeof(int) * 4, st) != cudaSuccess) return HPSD_ECUDA_;
    meddc_tridiag_kernel<<<count, kMedThreads, med_smem_bytes(n), st>>>(n, offs_dev, io, w);
    HPSD_LAUNCH_CHECK();
    double *lam, *Z;
    int rc = launch_stedc(w.s, w.d, w.e, &lam, &Z, st);
    if (rc) return rc;
    meddc_back_kernel<<<count, kMedThreads, meddc_back_smem(n), st>>>(n, offs_dev, io, w, lam, Z, w.s.ldz, info_dev, info_idx_dev);
    HPSD_LAUNCH_CHECK();
    return 0;
}

int medium_init() {
    const int maxb = (int)med_smem_bytes(kMediumMaxN);
    if (cudaFuncSetAttribute(hhql_project_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, maxb) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(meddc_tridiag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)med_smem_bytes(kMedDcMaxN)) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(meddc_back_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)meddc_back_smem(kMedDcMaxN)) != cudaSuccess) return HPSD_ECUDA_;
    return 0;
}

int launch_hhql_project(int n, int count, const long long *offs_dev, const SvecIo &io,
                        int *info_dev, const int *info_idx_dev, cudaStream_t st) {
    if (count <= 0) return 0;
    if (n < 2 || n > kMediumMaxN) return -1;
    hhql_project_kernel<<<count, kMedThreads, med_smem_bytes(n), st>>>(n, offs_dev, io, info_dev, info_idx_dev);
    HPSD_LAUNCH_CHECK();
    return 0;
}

}  // namespace hpsd
