// jacobi.cu -- S9/S10 of SURVEY.md §8(a): small and medium blocks (2 <= n <= 84).
// One CTA per matrix, everything in shared memory, one kernel from svec to svec:
//   S1 unpack -> two-sided cyclic Jacobi on the complex Hermitian matrix with the
//   eigenvectors accumulated -> S6 clamp/scale -> S7 W W^H -> S8 pack.
// Operation defined at PAPER.md:1536; layout Eq. (D10) PAPER.md:1220-1222.
//
// Parallel ordering: round-robin ("circle") tournament on m = n rounded up to even:
// m-1 rounds per sweep, m/2 disjoint index pairs per round.  In a round every 2x2
// sub-block A[{p_i,q_i},{p_j,q_j}] is updated as J_i^H B J_j by one thread, so A is
// read and written once per round and no sync is needed between the row and the
// column halves of the similarity transform.
//
// Rotation for the pair (p,q) with alpha=a_pp, gamma=a_qq, beta=a_pq=|beta|e^{i phi}:
//   tau=(gamma-alpha)/(2|beta|), t=sgn(tau)/(|tau|+sqrt(1+tau^2)), c=1/sqrt(1+t^2), s=tc,
//   J = [[c, s], [-s e^{-i phi}, c e^{-i phi}]]   (acts on coordinates p,q),  A <- J^H A J.
#include "kernels.h"

namespace hpsd {

constexpr int kJacobiMaxSweeps = 40;

struct JacobiSmem {
    cplx *A, *V, *eph;
    double *c, *s, *red;
    int *p, *q, *poslist;
};

__device__ __forceinline__ JacobiSmem carve(unsigned char *base, int m) {
    JacobiSmem sm;
    sm.A = reinterpret_cast<cplx *>(base);
    sm.V = sm.A + (size_t)m * m;
    sm.eph = sm.V + (size_t)m * m;
    sm.c = reinterpret_cast<double *>(sm.eph + m / 2);
    sm.s = sm.c + m / 2;
    sm.red = sm.s + m / 2;            // 32 doubles
    sm.p = reinterpret_cast<int *>(sm.red + 32);
    sm.q = sm.p + m / 2;
    sm.poslist = sm.q + m / 2;        // m ints
    return sm;
}

static size_t jacobi_smem_bytes(int m) {
    return (size_t)2 * m * m * sizeof(cplx) + (size_t)(m / 2) * (sizeof(cplx) + 2 * sizeof(double) + 2 * sizeof(int)) +
           32 * sizeof(double) + (size_t)m * sizeof(int) + 16;
}

template <int THREADS>
__global__ void __launch_bounds__(THREADS) jacobi_project_kernel(int n, const long long *__restrict__ offs,
                                                                 SvecIo io,
                                                                 int *__restrict__ info, const int *__restrict__ info_idx) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int m = (n + 1) & ~1;
    const int h = m / 2;
    JacobiSmem sm = carve(smem_raw, m);
    cplx *A = sm.A, *V = sm.V;
    const int tid = threadIdx.x;
    const size_t base = (size_t)offs[blockIdx.x];

    // ---- S1: unpack into shared memory (both triangles), V = I -------------
    for (int t = tid; t < m * m; t += THREADS) {
        A[t] = mk(0.0, 0.0);
        V[t] = mk((t / m == t % m) ? 1.0 : 0.0, 0.0);
    }
    __syncthreads();
    double ss = 0.0;
    for (int t = tid; t < n * n; t += THREADS) {
        const int j = t / n, i = t % n;
        if (i < j) continue;
        const size_t c = base + svec_col_off(n, j);
        if (i == j) {
            const double d = io_load(io, c);
            A[(size_t)j * m + i] = mk(d, 0.0);
            ss += d * d;
        } else {
            const int k = i - j - 1;
            const cplx v = mk(io_load(io, c + 1 + 2 * k) / kSqrt2, io_load(io, c + 2 + 2 * k) / kSqrt2);
            A[(size_t)j * m + i] = v;
            A[(size_t)i * m + j] = conj_(v);
            ss += 2.0 * abs2(v);
        }
    }
    // block reduction of ||A||_F^2
    ss = warp_sum(ss);
    if ((tid & 31) == 0) sm.red[tid >> 5] = ss;
    __syncthreads();
    if (tid < 32) {
        double v = (tid < THREADS / 32) ? sm.red[tid] : 0.0;
        v = warp_sum(v);
        if (tid == 0) sm.red[0] = v;
    }
    __syncthreads();
    const double fro2 = sm.red[0];
    if (nonfinite(fro2)) {                     // NaN / Inf in the block (block-uniform): all-NaN output, info = 2
        io_fill_nan(io, base, n, tid, THREADS);
        if (info != nullptr && tid == 0) info[info_idx[blockIdx.x]] = kInfoNonFinite;
        return;
    }
    // |a_pq| <= eps ||A||_F / m is negligible: leaves off(A) <= eps ||A||_F in total
    const double tol2 = (kEps * kEps) * fro2 / ((double)m * (double)m);
    __syncthreads();

    int sweeps = 0;
    bool converged = (fro2 == 0.0) || (m < 2);
    const int nA = h * h, nV = m * h;
    while (!converged && sweeps < kJacobiMaxSweeps) {
        int rot_in_sweep = 0;
        for (int r = 0; r < m - 1; ++r) {
            // ---- phase 1: rotation parameters of the h disjoint pairs --------
            int active = 0;
            if (tid < h) {
                int p, q;
                if (tid == 0) { p = m - 1; q = r; }
                else { p = (r + tid) % (m - 1); q = (r - tid + (m - 1)) % (m - 1); }
                const double al = A[(size_t)p * m + p].x, ga = A[(size_t)q * m + q].x;
                const cplx be = A[(size_t)q * m + p];        // a_pq: row p, column q
                const double b2 = abs2(be);
                double c = 1.0, s = 0.0;
                cplx e = mk(1.0, 0.0);
                if (b2 > tol2) {
                    // the parameters of a rotation are one dependent chain that every round waits for: reciprocal square
                    // roots (each refined by one Newton step to working precision) and one reciprocal instead of three DSQRT
                    // and four DDIV (~300 instead of ~750 cycles)
                    double iab = rsqrt(b2);
                    iab = fma(0.5 * iab, fma(-b2 * iab, iab, 1.0), iab);          // 1 / |beta|
                    const double tau = (ga - al) * (0.5 * iab);
                    double t;
                    if (fabs(tau) < 1e150) {
                        const double x = fma(tau, tau, 1.0);
                        double rx = rsqrt(x);
                        rx = fma(0.5 * rx, fma(-x * rx, rx, 1.0), rx);
                        t = copysign(__drcp_rn(fabs(tau) + x * rx), tau);          // sgn(tau) / (|tau| + sqrt(1 + tau^2))
                    } else t = 0.5 / tau;                                          // tau^2 would overflow
                    const double y = fma(t, t, 1.0);
                    double ry = rsqrt(y);
                    ry = fma(0.5 * ry, fma(-y * ry, ry, 1.0), ry);
                    c = ry;
                    s = t * c;
                    e = mk(be.x * iab, -be.y * iab);         // e^{-i phi}
                    active = 1;
                }
                sm.p[tid] = p; sm.q[tid] = q; sm.c[tid] = c; sm.s[tid] = s; sm.eph[tid] = e;
            }
            rot_in_sweep += __syncthreads_count(active);
            // ---- phase 2: A <- J^H A J block by block, V <- V J --------------
            for (int t = tid; t < nA + nV; t += THREADS) {
                if (t < nA) {
                    const int i = t % h, j = t / h;
                    const double ci = sm.c[i], si = sm.s[i], cj = sm.c[j], sj = sm.s[j];
                    if (si == 0.0 && sj == 0.0) continue;
                    const int pi = sm.p[i], qi = sm.q[i], pj = sm.p[j], qj = sm.q[j];
                    const cplx ei = conj_(sm.eph[i]);        // e^{+i phi_i}
                    const cplx ej = sm.eph[j];               // e^{-i phi_j}
                    cplx b00 = A[(size_t)pj * m + pi], b10 = A[(size_t)pj * m + qi];
                    cplx b01 = A[(size_t)qj * m + pi], b11 = A[(size_t)qj * m + qi];
                    // columns: [b_r0, b_r1] <- [c b_r0 - s e b_r1, s b_r0 + c e b_r1]
                    cplx t01 = ej * b01, t11 = ej * b11;
                    cplx n00 = cj * b00 - sj * t01, n01 = sj * b00 + cj * t01;
                    cplx n10 = cj * b10 - sj * t11, n11 = sj * b10 + cj * t11;
                    // rows: [b_0c; b_1c] <- [c b_0c - s e+ b_1c ; s b_0c + c e+ b_1c]
                    cplx u10 = ei * n10, u11 = ei * n11;
                    b00 = ci * n00 - si * u10; b10 = si * n00 + ci * u10;
                    b01 = ci * n01 - si * u11; b11 = si * n01 + ci * u11;
                    if (i == j) {                            // the annihilated pair: exact zeros, real diagonal
                        b01 = mk(0.0, 0.0); b10 = mk(0.0, 0.0);
                        b00.y = 0.0; b11.y = 0.0;
                    }
                    A[(size_t)pj * m + pi] = b00; A[(size_t)pj * m + qi] = b10;
                    A[(size_t)qj * m + pi] = b01; A[(size_t)qj * m + qi] = b11;
                } else {
                    const int u = t - nA;
                    const int row = u % m, j = u / m;
                    const double cj = sm.c[j], sj = sm.s[j];
                    if (sj == 0.0) continue;
                    const int pj = sm.p[j], qj = sm.q[j];
                    const cplx v0 = V[(size_t)pj * m + row];
                    const cplx t1 = sm.eph[j] * V[(size_t)qj * m + row];
                    V[(size_t)pj * m + row] = cj * v0 - sj * t1;
                    V[(size_t)qj * m + row] = sj * v0 + cj * t1;
                }
            }
            __syncthreads();
        }
        ++sweeps;
        converged = (rot_in_sweep == 0);
    }
    if (info != nullptr && tid == 0) info[info_idx[blockIdx.x]] = converged ? 0 : 1;

    // ---- S6: clamp, W = V_+ diag(sqrt(lambda_+)); list of positive columns ---
    if (tid == 0) {
        int k = 0;
        for (int l = 0; l < n; ++l)
            if (A[(size_t)l * m + l].x > 0.0) sm.poslist[k++] = l;
        sm.p[0] = k;   // pair tables are dead now
    }
    __syncthreads();
    const int kpos = sm.p[0];
    __syncthreads();
    for (int t = tid; t < kpos * n; t += THREADS) {
        const int l = sm.poslist[t / n], i = t % n;
        const double w = sqrt(A[(size_t)l * m + l].x);
        V[(size_t)l * m + i] = w * V[(size_t)l * m + i];
    }
    __syncthreads();
    // ---- S7 + S8: lower triangle of W W^H straight into the svec -----------
    for (int t = tid; t < n * n; t += THREADS) {
        const int j = t / n, i = t % n;
        if (i < j) continue;
        cplx acc = mk(0.0, 0.0);
        for (int k = 0; k < kpos; ++k) {
            const int l = sm.poslist[k];
            const cplx a = V[(size_t)l * m + i], b = V[(size_t)l * m + j];
            // a * conj(b)
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

int jacobi_init() {
    const int maxb = (int)jacobi_smem_bytes(kJacobiMaxN);
    if (cudaFuncSetAttribute(jacobi_project_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, maxb) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(jacobi_project_kernel<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, maxb) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(jacobi_project_kernel<1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, maxb) != cudaSuccess) return HPSD_ECUDA_;
    return 0;
}

int launch_jacobi_project(int n, int count, const long long *offs_dev, const SvecIo &io,
                          int *info_dev, const int *info_idx_dev, cudaStream_t st) {
    if (count <= 0) return 0;
    if (n < 2 || n > kJacobiMaxN) return -1;
    const int m = (n + 1) & ~1;
    const size_t smem = jacobi_smem_bytes(m);
    if (m <= 32) jacobi_project_kernel<256><<<count, 256, smem, st>>>(n, offs_dev, io, info_dev, info_idx_dev);
    else if (m <= 56) jacobi_project_kernel<512><<<count, 512, smem, st>>>(n, offs_dev, io, info_dev, info_idx_dev);
    else jacobi_project_kernel<1024><<<count, 1024, smem, st>>>(n, offs_dev, io, info_dev, info_idx_dev);
    HPSD_LAUNCH_CHECK();
    return 0;
}

}  // namespace hpsd
