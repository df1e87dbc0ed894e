// hb2st.cu -- S3 of SURVEY.md §8(a): Hermitian band (width b = kBW) -> REAL symmetric tridiagonal by bulge chasing,
// B = Q2 T Q2^H.  Second half of the two-stage reduction behind the "eigendecomposition" of PAPER.md:1536
// (BASELINE.json north star (c): "band to tridiagonal by ... bulge chasing").
//
// Sweep s (s = 0 .. n-2) annihilates column s below the sub-diagonal with a reflector of length <= b (hop 0) and
// chases the bulge it creates down the band, one b x b block pair per hop:
//   hop 0:  H_0 from A[s+1 : s+1+b, s];  D_0 <- H_0^H D_0 H_0                 (D_k = A[r_k, r_k], r_k = s+1+kb .. +b)
//   hop k:  B_k = A[r_k, r_{k-1}] <- B_k H_{k-1};  H_k from column 0 of B_k;  B_k <- H_k^H B_k;  D_k <- H_k^H D_k H_k
// Every reflector comes from zlarfg (complex tau, REAL beta), so the final sub-diagonal is real without a phase pass.
//
// Dependencies: (s, k) needs (s, k-1) and (s-1, k+1): consecutive sweeps run two hops apart and the whole stage is a
// chain of ~2n hops, i.e. latency-bound.  One CTA runs one sweep at a time (sweep s on CTA s mod G)
// and publishes its progress with a release store that the next sweep's CTA polls.  Inside a CTA two warp groups
// split a hop, so that only the B_k work is on the sweep's own chain:
//   group B (warps 0-3): B_k right update, reflector H_k, left update; hands v_k to group D through shared memory
//   group D (warps 4-7): D_k two-sided update (at most two hops behind), then the release of hop k
// Every thread keeps its 8 block elements in registers (loaded straight from the band in L2, stored straight back).
// The band lives in L2 (16 * 2b * n bytes: 4.2 MB at n = 4096).  The reflectors are kept for the back-transformation
// (backq2.cu): (s, k) at V2[(k n + s) b], tau2[k n + s].
#include "kernels.h"
#include "twostage.h"
#include "prof.h"

namespace hpsd {

constexpr int kBcGroup = 128;                 // threads per warp group
constexpr int kBcThreads = 2 * kBcGroup;
constexpr int kBcP = kBW + 2;                 // pitch of the transposed staging of B_k (row index contiguous)
constexpr int kBcDone = 1 << 30;
static_assert(kBW == 32 && kBcGroup == 128, "thread tiling of the bulge-chasing kernel: 4 threads per block row");

// named barriers (0 is left to __syncthreads).  VREADY: B arrives, D waits.  VFREE: D arrives, B waits (two hops later).
// BSTORED: B arrives, D waits.  The [slot] variants alternate with the hop counter.
enum { BAR_B = 1, BAR_D = 2, BAR_VREADY = 3, BAR_VFREE = 5, BAR_BSTORED = 7 };
__device__ __forceinline__ void bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

struct BcArgs {
    int n, ldab;
    cplx *AB;
    cplx *V2, *tau2;
    double *d, *e;
    int *prog;
};

__device__ __forceinline__ int bc_ld_acquire(const int *p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void bc_st_release(int *p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// zlarfg scalars with one reciprocal square root and one reciprocal on the dependent chain
__device__ __forceinline__ void bc_householder(cplx alpha, double xnorm2, double &beta, cplx &tau, cplx &scale) {
    if (xnorm2 == 0.0 && alpha.y == 0.0) {
        beta = alpha.x; tau = mk(0.0, 0.0); scale = mk(0.0, 0.0);
    } else {
        const double s = alpha.x * alpha.x + alpha.y * alpha.y + xnorm2;
        double rinv = rsqrt(s);
        rinv = fma(0.5 * rinv, fma(-s * rinv, rinv, 1.0), rinv);      // one Newton step: full accuracy
        const double nrm = s * rinv;
        beta = -copysign(nrm, alpha.x);
        const double ib = -copysign(rinv, alpha.x);
        tau = mk((beta - alpha.x) * ib, -alpha.y * ib);
        const cplx den = mk(alpha.x - beta, alpha.y);
        const double id2 = __drcp_rn(abs2(den));
        scale = mk(den.x * id2, -den.y * id2);
    }
}

// sum over the 4 lanes of a row group
__device__ __forceinline__ cplx quad_sum(cplx v) {
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
    }
    return v;
}
// sum over the 8 row groups of a warp (lanes with equal lane % 4)
__device__ __forceinline__ double oct_sum(double v) {
#pragma unroll
    for (int o = 4; o <= 16; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

struct BcSmem {
    cplx Bt[kBW * kBcP];           // B_k transposed staging for the left update: Bt[c][r]
    cplx v[2][kBW];                // reflector ring (slot = hop counter & 1)
    cplx w[kBW];
    cplx tau[2];
    double redB[4], redD[4];
    cplx alpha;
};

__global__ void __launch_bounds__(kBcThreads, 1) hb2st_kernel(BcArgs a) {
    extern __shared__ __align__(16) unsigned char bc_smem[];
    BcSmem &S = *reinterpret_cast<BcSmem *>(bc_smem);
    const int tid = threadIdx.x;
    const bool isB = tid < kBcGroup;
    const int gt = tid & (kBcGroup - 1), lane = tid & 31, gw = gt >> 5;     // thread / warp inside the group
    const int r = gt >> 2, q = gt & 3;                                      // block row, column residue (columns q + 4t)
    const int n = a.n, ldab = a.ldab;
    unsigned h = 0;                                                         // hop counter of this CTA (both groups count alike)

    for (int s = blockIdx.x; s < n - 1; s += gridDim.x) {
        const int nhops = (n - 1 - s + kBW - 1) / kBW;
        cplx tau_prev = mk(0.0, 0.0);
        for (int k = 0; k < nhops; ++k, ++h) {
            const int slot = h & 1;
            const int r0 = s + 1 + k * kBW;
            const int len = (n - r0 < kBW) ? n - r0 : kBW;
            // ---- wait for sweep s-1 to be two hops ahead (each group polls for itself, then loads its own block;
            //      the acquire invalidates this SM's L1, so the plain loads below see what the other SM published)
            if (s > 0) {
                if (gt == 0) {
                    const int *pp = a.prog + (s - 1);
                    while (bc_ld_acquire(pp) < k + 2) { }
                }
                bar_sync(isB ? BAR_B : BAR_D, kBcGroup);
            }
            if (isB) {
                // =========================== group B: reflector of this hop ===========================
                double beta = 0.0; cplx tau = mk(0.0, 0.0), scale = mk(0.0, 0.0);
                cplx b8[8];
                cplx x0 = mk(0.0, 0.0);                              // hop 0, warp 0: column s below the diagonal
                if (k == 0) {
                    if (gw == 0) {
                        if (lane < len) x0 = a.AB[(size_t)s * ldab + 1 + lane];
                        double p2 = (lane >= 1) ? abs2(x0) : 0.0;
                        p2 = warp_sum(p2);
                        cplx alpha;
                        alpha.x = __shfl_sync(0xffffffffu, x0.x, 0);
                        alpha.y = __shfl_sync(0xffffffffu, x0.y, 0);
                        bc_householder(alpha, p2, beta, tau, scale);
                    }
                } else {
                    const int p0 = r0 - kBW;
                    // B_k = A[r0 : r0+len, p0 : p0+b]: element (r, c) at band offset b + r - c of column p0 + c
#pragma unroll
                    for (int t = 0; t < 8; ++t) {
                        const int c = q + 4 * t;
                        b8[t] = (r < len) ? a.AB[(size_t)(p0 + c) * ldab + (kBW + r - c)] : mk(0.0, 0.0);
                    }
                    // right: B <- B (I - tau_p vp vp^H)
                    const cplx *vp = S.v[slot ^ 1];
                    cplx vpc[8];
                    cplx wv = mk(0.0, 0.0);
#pragma unroll
                    for (int t = 0; t < 8; ++t) { vpc[t] = vp[q + 4 * t]; cfma(wv, b8[t], vpc[t]); }
                    wv = quad_sum(wv);
                    const cplx tw = tau_prev * wv;
#pragma unroll
                    for (int t = 0; t < 8; ++t) cfma(b8[t], mk(-tw.x, -tw.y), conj_(vpc[t]));
                    // new reflector from column 0 (threads with q == 0 hold it in b8[0])
                    double p2 = (q == 0 && r >= 1) ? abs2(b8[0]) : 0.0;
                    p2 = oct_sum(p2);
                    if (lane == 0) S.redB[gw] = p2;
                    if (gt == 0) S.alpha = b8[0];
                    bar_sync(BAR_B, kBcGroup);
                    const double xn2 = (S.redB[0] + S.redB[1]) + (S.redB[2] + S.redB[3]);
                    bc_householder(S.alpha, xn2, beta, tau, scale);
                }
                // the slot of the reflector ring is free once group D is through hop h - 2
                if (h >= 2) bar_sync(BAR_VFREE + slot, kBcThreads);
                // ---- publish v_k, tau_k (and B_k, transposed, for the left update)
                if (k == 0) {
                    if (gw == 0) {
                        S.v[slot][lane] = (lane == 0) ? mk(1.0, 0.0) : (lane < len ? x0 * scale : mk(0.0, 0.0));
                        if (lane == 0) {
                            S.tau[slot] = tau;
                            a.d[s] = a.AB[(size_t)s * ldab].x;
                            a.e[s] = beta;
                        }
                    }
                } else {
                    if (q == 0) {
                        S.v[slot][r] = (r == 0) ? mk(1.0, 0.0) : (r < len ? b8[0] * scale : mk(0.0, 0.0));
                        b8[0] = (r == 0) ? mk(beta, 0.0) : mk(0.0, 0.0);
                        if (r == 0) S.tau[slot] = tau;
                    }
#pragma unroll
                    for (int t = 0; t < 8; ++t) S.Bt[(q + 4 * t) * kBcP + r] = b8[t];
                }
                bar_sync(BAR_B, kBcGroup);
                tau = S.tau[slot];
                bar_arrive(BAR_VREADY + slot, kBcThreads);          // group D may start on D_k
                if (gt < kBW) a.V2[((size_t)k * n + s) * kBW + gt] = S.v[slot][gt];
                if (gt == 0) a.tau2[(size_t)k * n + s] = tau;
                if (k > 0) {
                    // left: columns 1 .. b-1:  B <- B - conj(tau) v (v^H B)     (thread = column c, rows q + 4t)
                    const int p0 = r0 - kBW;
                    const int c = gt >> 2;
                    cplx col[8], vv[8];
                    cplx z = mk(0.0, 0.0);
#pragma unroll
                    for (int t = 0; t < 8; ++t) { col[t] = S.Bt[c * kBcP + q + 4 * t]; vv[t] = S.v[slot][q + 4 * t]; cfma_conj(z, vv[t], col[t]); }
                    z = quad_sum(z);
                    const cplx ctz = conj_(tau) * z;
                    cplx *dst = a.AB + (size_t)(p0 + c) * ldab + (kBW - c);
#pragma unroll
                    for (int t = 0; t < 8; ++t) {
                        const int rr = q + 4 * t;
                        if (c >= 1) cfma(col[t], mk(-ctz.x, -ctz.y), vv[t]);
                        if (rr < len) dst[rr] = col[t];
                    }
                }
                tau_prev = tau;
                bar_arrive(BAR_BSTORED + slot, kBcThreads);         // B_k is on its way to L2
            } else {
                // =========================== group D: two-sided update of D_k ===========================
                cplx d8[8];
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    const int c = q + 4 * t;
                    // stored lower: (r, c) with r < c is the conjugate of (c, r); one load either way, no branch
                    const int lo = r < c ? r : c, df = r < c ? c - r : r - c;
                    cplx val = (r < len && c < len) ? a.AB[(size_t)(r0 + lo) * ldab + df] : mk(0.0, 0.0);
                    if (r < c) val.y = -val.y;
                    d8[t] = val;
                }
                bar_sync(BAR_VREADY + slot, kBcThreads);            // v_k, tau_k are in the ring
                const cplx *v = S.v[slot];
                const cplx tau = S.tau[slot];
                cplx vc[8];
                cplx y = mk(0.0, 0.0);
#pragma unroll
                for (int t = 0; t < 8; ++t) { vc[t] = v[q + 4 * t]; cfma(y, d8[t], vc[t]); }
                y = quad_sum(y);
                const cplx vr = v[r];
                // dot = v^H y (real for Hermitian D; the imaginary rounding residue is dropped)
                double part = (q == 0) ? (vr.x * y.x + vr.y * y.y) : 0.0;
                part = oct_sum(part);
                if (lane == 0) S.redD[gw] = part;
                if (q == 0) S.w[r] = y;                              // y, not w: every thread finishes w_c itself (one exchange)
                bar_sync(BAR_D, kBcGroup);
                const double dot = (S.redD[0] + S.redD[1]) + (S.redD[2] + S.redD[3]);
                // w_r = tau y_r - 1/2 |tau|^2 dot v_r     (zhetd2: x = tau D v, w = x - 1/2 tau (x^H v) v)
                const double cc = 0.5 * abs2(tau) * dot;
                const cplx ty = tau * y;
                const cplx wr = mk(ty.x - cc * vr.x, ty.y - cc * vr.y);
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    const int c = q + 4 * t;
                    const cplx tyc = tau * S.w[c];
                    const cplx wc = mk(tyc.x - cc * vc[t].x, -(tyc.y - cc * vc[t].y));      // conj(w_c)
                    cfma(d8[t], mk(-vr.x, -vr.y), wc);
                    cfma(d8[t], mk(-wr.x, -wr.y), conj_(vc[t]));
                    if (r == c) d8[t].y = 0.0;
                    if (r >= c && r < len) a.AB[(size_t)(r0 + c) * ldab + (r - c)] = d8[t];
                }
                if (s == n - 2 && gt == 0) a.d[n - 1] = d8[0].x;   // the 1 x 1 block of the last sweep
                bar_sync(BAR_BSTORED + slot, kBcThreads);           // group B's stores of this hop are issued as well
                // release at gpu scope is cumulative over the stores the barriers ordered before it
                if (gt == 0) bc_st_release(a.prog + s, (k == nhops - 1) ? kBcDone : k + 1);
                bar_arrive(BAR_VFREE + slot, kBcThreads);           // ring slot and S.w are free again
            }
        }
    }
}

__global__ void hb2st_n1_kernel(const cplx *AB, double *d) { d[0] = AB[0].x; }

static int g_bc_init_dev = -1;
int hb2st_init() {
    int dev = 0;
    cudaGetDevice(&dev);
    if (g_bc_init_dev == dev) return 0;
    if (cudaFuncSetAttribute(hb2st_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BcSmem)) != cudaSuccess) return HPSD_ECUDA_;
    g_bc_init_dev = dev;
    return 0;
}

size_t twostage_hops(int n) { return n > 1 ? (size_t)(n - 1 + kBW - 1) / kBW : 1; }

int launch_hb2st(const TwoStageWs &w, cudaStream_t st) {
    const int n = w.n;
    if (n <= 0) return 0;
    int rc = hb2st_init();
    if (rc) return rc;
    prof_begin(ST_BULGE, st);
    if (n == 1) {
        hb2st_n1_kernel<<<1, 1, 0, st>>>(w.AB, w.d);
        HPSD_LAUNCH_CHECK();
        prof_end(ST_BULGE, st);
        return 0;
    }
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    HPSD_CUDA_OK(cudaMemsetAsync(w.prog, 0, sizeof(int) * (size_t)n, st));
    BcArgs a{n, w.ldab, w.AB, w.V2, w.tau2, w.d, w.e, w.prog};
    int G = sms < n - 1 ? sms : n - 1;
    void *args[] = {&a};
    // cooperative launch: every CTA must be resident, a sweep's CTA spins on the previous sweep's CTA
    const cudaError_t e = cudaLaunchCooperativeKernel((void *)hb2st_kernel, dim3(G), dim3(kBcThreads), args, sizeof(BcSmem), st);
    g_launches++;
    prof_end(ST_BULGE, st);
    return e == cudaSuccess ? 0 : HPSD_ECUDA_;
}

}  // namespace hpsd
