// hb2st.cu -- S3 of SURVEY.md §8(a): Hermitian band (width b = kBW) -> REAL symmetric tridiagonal by bulge chasing,
// B = Q2 T Q2^H.  Second half of the two-stage reduction behind the "eigendecomposition" of PAPER.md:1536
// (BASELINE.json north star (c): "band to tridiagonal by ... bulge chasing").
//
// Sweep s (s = 0 .. n-2) annihilates column s below the sub-diagonal with a reflector of length <= b (hop 0) and
// chases the bulge it creates down the band, one b x b block pair per hop:
//   hop 0:  H_0 from A[s+1 : s+1+b, s];  D_0 <- H_0^H D_0 H_0                 (D_k = A[r_k, r_k], r_k = s+1+kb .. +b)
//   hop k:  B_k = A[r_k, r_{k-1}] <- B_k H_{k-1};  H_k from column 0 of B_k;  B_k <- H_k^H B_k;  D_k <- H_k^H D_k H_k
// Every reflector comes from zlarfg (complex tau, REAL beta), so the final sub-diagonal is real without a phase pass.
// Dependencies: (s, k) needs (s, k-1) and (s-1, k+1).  One CTA runs one sweep at a time (sweep s on CTA s mod G) and
// publishes its progress with a release store; the next sweep's CTA polls it with acquire loads, so the sweeps run as
// a pipeline two hops apart over the SMs.  The band lives in L2 (16 * 2b * n bytes: 4.2 MB at n = 4096).
// The reflectors are kept for the back-transformation (backq2.cu): (s, k) at V2[(k n + s) b], tau2[k n + s].
#include <cooperative_groups.h>
#include "kernels.h"
#include "twostage.h"
#include "prof.h"

namespace hpsd {

constexpr int kBcThreads = 128;
constexpr int kBcP = kBW + 4;            // shared-memory pitch of the blocks (elements): thread tiles (row, 4 lanes) conflict free
constexpr int kBcDone = 1 << 30;
static_assert(kBW == 32 && kBcThreads == 128, "thread tiling of the bulge-chasing kernel");

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

__device__ __forceinline__ void bc_householder(cplx alpha, double xnorm2, double &beta, cplx &tau, cplx &scale) {
    if (xnorm2 == 0.0 && alpha.y == 0.0) {
        beta = alpha.x; tau = mk(0.0, 0.0); scale = mk(0.0, 0.0);
    } else {
        const double nrm = sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xnorm2);
        beta = -copysign(nrm, alpha.x);
        const double ib = 1.0 / beta;
        tau = mk((beta - alpha.x) * ib, -alpha.y * ib);
        const cplx den = mk(alpha.x - beta, alpha.y);
        const double id2 = 1.0 / abs2(den);
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
    cplx Bk[kBW * kBcP];
    cplx D[kBW * kBcP];
    cplx v[kBW], vp[kBW], w[kBW];
    double red[8];
    cplx alpha;
    int flag;
};

// D (len x len, full in shared memory) <- H^H D H with H = I - tau v v^H (zhetd2 arithmetic): x = tau D v,
// w = x - 1/2 tau (x^H v) v,  D -= v w^H + w v^H.  The lower triangle goes back to the band.
__device__ __forceinline__ void bc_two_sided(BcSmem &S, cplx *AB, int ldab, int r0, int len, cplx tau, int tid) {
    const int r = tid >> 2, q = tid & 3, lane = tid & 31, warp = tid >> 5;
    cplx y = mk(0.0, 0.0);
#pragma unroll
    for (int t = 0; t < 8; ++t) cfma(y, S.D[r * kBcP + q + 4 * t], S.v[q + 4 * t]);
    y = quad_sum(y);
    // dot = v^H y (real for Hermitian D; the imaginary rounding residue is dropped)
    double part = (q == 0) ? (S.v[r].x * y.x + S.v[r].y * y.y) : 0.0;
    part = oct_sum(part);
    if (lane == 0) S.red[warp] = part;
    __syncthreads();
    const double dot = (S.red[0] + S.red[1]) + (S.red[2] + S.red[3]);
    // w_r = tau y_r - 1/2 |tau|^2 dot v_r
    if (q == 0) {
        const double c = 0.5 * abs2(tau) * dot;
        const cplx vr = S.v[r];
        const cplx ty = tau * y;
        S.w[r] = mk(ty.x - c * vr.x, ty.y - c * vr.y);
    }
    __syncthreads();
    {
        const cplx vr = S.v[r], wr = S.w[r];
#pragma unroll
        for (int t = 0; t < 8; ++t) {
            const int c = q + 4 * t;
            cplx dv = S.D[r * kBcP + c];
            const cplx vc = conj_(S.v[c]), wc = conj_(S.w[c]);
            cfma(dv, mk(-vr.x, -vr.y), wc);
            cfma(dv, mk(-wr.x, -wr.y), vc);
            if (r == c) dv.y = 0.0;
            S.D[r * kBcP + c] = dv;
        }
    }
    __syncthreads();
    // lower triangle -> band: column c = tid / 4, rows part of 8
    {
        const int c = tid >> 2, p8 = (tid & 3) * 8;
        if (c < len) {
            cplx *dst = AB + (size_t)(r0 + c) * ldab;
#pragma unroll
            for (int t = 0; t < 8; ++t) {
                const int rr = p8 + t;
                if (rr >= c && rr < len) dst[rr - c] = S.D[rr * kBcP + c];
            }
        }
    }
}

// load D = A[r0 : r0+len, r0 : r0+len] from the band (lower stored) as a full Hermitian block, zero padded to b x b
__device__ __forceinline__ void bc_load_diag(BcSmem &S, const cplx *AB, int ldab, int r0, int len, int tid) {
    const int c = tid >> 2, p8 = (tid & 3) * 8;
    const cplx *src = AB + (size_t)(r0 + c) * ldab;
    cplx val[8];
#pragma unroll
    for (int t = 0; t < 8; ++t) {             // eight independent loads in flight per thread
        const int rr = p8 + t;
        val[t] = (rr >= c && rr < len && c < len) ? src[rr - c] : mk(0.0, 0.0);
    }
#pragma unroll
    for (int t = 0; t < 8; ++t) {
        const int rr = p8 + t;
        if (rr >= c) {
            S.D[rr * kBcP + c] = val[t];
            if (rr > c) S.D[c * kBcP + rr] = conj_(val[t]);
        }
    }
}

__global__ void __launch_bounds__(kBcThreads) hb2st_kernel(BcArgs a) {
    extern __shared__ __align__(16) unsigned char bc_smem[];
    BcSmem &S = *reinterpret_cast<BcSmem *>(bc_smem);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = a.n, ldab = a.ldab;
    const int r = tid >> 2, q = tid & 3;

    for (int s = blockIdx.x; s < n - 1; s += gridDim.x) {
        const int nhops = (n - 1 - s + kBW - 1) / kBW;
        cplx tau_prev = mk(0.0, 0.0);
        for (int k = 0; k < nhops; ++k) {
            // ---- wait for sweep s-1 to be two hops ahead
            if (s > 0) {
                if (tid == 0) {
                    const int *pp = a.prog + (s - 1);
                    while (bc_ld_acquire(pp) < k + 2) { }
                }
                __syncthreads();
            }
            const int r0 = s + 1 + k * kBW;
            const int len = (n - r0 < kBW) ? n - r0 : kBW;
            double beta; cplx tau, scale;
            if (k == 0) {
                // column s below the diagonal
                cplx x = mk(0.0, 0.0);
                if (tid < kBW && tid < len) x = a.AB[(size_t)s * ldab + 1 + tid];
                bc_load_diag(S, a.AB, ldab, r0, len, tid);
                if (warp == 0) {
                    double p2 = (lane >= 1) ? abs2(x) : 0.0;
                    p2 = warp_sum(p2);
                    cplx alpha;
                    alpha.x = __shfl_sync(0xffffffffu, x.x, 0);
                    alpha.y = __shfl_sync(0xffffffffu, x.y, 0);
                    bc_householder(alpha, p2, beta, tau, scale);
                    S.v[lane] = (lane == 0) ? mk(1.0, 0.0) : (lane < len ? x * scale : mk(0.0, 0.0));
                    if (lane == 0) {
                        S.alpha = tau; S.red[4] = beta;
                        a.d[s] = a.AB[(size_t)s * ldab].x;
                        a.e[s] = beta;
                    }
                }
                __syncthreads();
                tau = S.alpha;
            } else {
                const int p0 = r0 - kBW;
                // ---- load B_k = A[r0 : r0+len, p0 : p0+b] (column c: band offsets b - c ..) and D_k
                {
                    const int c = tid >> 2, p8 = (tid & 3) * 8;
                    const cplx *src = a.AB + (size_t)(p0 + c) * ldab + (kBW - c);
                    cplx val[8];
#pragma unroll
                    for (int t = 0; t < 8; ++t) val[t] = (p8 + t < len) ? src[p8 + t] : mk(0.0, 0.0);
                    bc_load_diag(S, a.AB, ldab, r0, len, tid);
#pragma unroll
                    for (int t = 0; t < 8; ++t) S.Bk[(p8 + t) * kBcP + c] = val[t];
                }
                __syncthreads();
                // ---- right: B <- B (I - tau_p vp vp^H)
                cplx b8[8];
                {
                    cplx wv = mk(0.0, 0.0);
#pragma unroll
                    for (int t = 0; t < 8; ++t) { b8[t] = S.Bk[r * kBcP + q + 4 * t]; cfma(wv, b8[t], S.vp[q + 4 * t]); }
                    wv = quad_sum(wv);
                    const cplx tw = tau_prev * wv;
#pragma unroll
                    for (int t = 0; t < 8; ++t) cfma(b8[t], mk(-tw.x, -tw.y), conj_(S.vp[q + 4 * t]));
                }
                // ---- new reflector from column 0 (threads with q == 0 hold it in b8[0])
                {
                    double p2 = (q == 0 && r >= 1) ? abs2(b8[0]) : 0.0;
                    p2 = oct_sum(p2);
                    if (lane == 0) S.red[warp] = p2;
                    if (tid == 0) S.alpha = b8[0];
                }
                __syncthreads();
                {
                    const double xn2 = (S.red[0] + S.red[1]) + (S.red[2] + S.red[3]);
                    bc_householder(S.alpha, xn2, beta, tau, scale);
                    if (q == 0) {
                        S.v[r] = (r == 0) ? mk(1.0, 0.0) : (r < len ? b8[0] * scale : mk(0.0, 0.0));
                        b8[0] = (r == 0) ? mk(beta, 0.0) : mk(0.0, 0.0);
                    }
#pragma unroll
                    for (int t = 0; t < 8; ++t) S.Bk[r * kBcP + q + 4 * t] = b8[t];
                }
                __syncthreads();
                // ---- left: columns 1 .. b-1:  B <- B - conj(tau) v (v^H B)     (thread = column c, rows q + 4t)
                {
                    const int c = tid >> 2;
                    cplx col[8];
                    cplx z = mk(0.0, 0.0);
#pragma unroll
                    for (int t = 0; t < 8; ++t) { col[t] = S.Bk[(q + 4 * t) * kBcP + c]; cfma_conj(z, S.v[q + 4 * t], col[t]); }
                    z = quad_sum(z);
                    const cplx ctz = conj_(tau) * z;
                    cplx *dst = a.AB + (size_t)(p0 + c) * ldab + (kBW - c);
#pragma unroll
                    for (int t = 0; t < 8; ++t) {
                        const int rr = q + 4 * t;
                        if (c >= 1) cfma(col[t], mk(-ctz.x, -ctz.y), S.v[rr]);
                        if (rr < len) dst[rr] = col[t];
                    }
                }
            }
            // ---- D_k <- H_k^H D_k H_k, reflector out
            bc_two_sided(S, a.AB, ldab, r0, len, tau, tid);
            if (tid < kBW) {
                a.V2[((size_t)k * n + s) * kBW + tid] = S.v[tid];
                S.vp[tid] = S.v[tid];
            }
            if (tid == 0) a.tau2[(size_t)k * n + s] = tau;
            tau_prev = tau;
            __syncthreads();                         // all stores of this hop are issued; vp is in place
            // release at gpu scope is cumulative over the stores the block barrier ordered before it: no separate fence
            if (tid == 0) bc_st_release(a.prog + s, (k == nhops - 1) ? kBcDone : k + 1);
        }
        if (s == n - 2 && tid == 0) a.d[n - 1] = S.D[0].x;      // the 1 x 1 block of the last hop
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
