// stedc.cu -- S4 of SURVEY.md §8(a): eigenvalues (ascending) and eigenvectors of the real
// symmetric tridiagonal T = (d, e), entirely on the device, no host synchronisation.
//
// Divide and conquer (Cuppen; deflation and the stable eigenvector formula of Gu & Eisenstat):
//   T = diag(T1', T2') + rho u u^T  at every split; leaves (<= 32) by implicit QL in one warp;
//   merge = sort poles, deflate (tiny weights, close poles by a Givens rotation), solve the secular
//   equation 1 + rho sum z_j^2/(d_j - lambda) = 0 for the K surviving roots (one warp per root,
//   two-pole rational interpolation with a bracketing safeguard, origin shifted to the nearest
//   pole so that d_j - lambda_i is accurate), recompute the weights z^ from the roots
//   (Loewner formula) so the eigenvectors are orthogonal by construction, and update
//   Z <- Z_children U with two real DMMA GEMMs that skip the structurally zero halves.
// All sizes that depend on the data (K, column types) live in device memory; kernels are launched
// on worst-case grids and exit early.  Chosen over bisection + inverse iteration because configs 3
// and 5 (617 eigenvalues in +-3e-3; 32-fold exact repeats) are its worst case.
#include "kernels.h"
#include "gemm.cuh"
#include "large.h"

namespace hpsd {

// node j at depth k owns indices [bound(k,j), bound(k,j+1))
__host__ __device__ __forceinline__ int node_bound(int n, int k, int j) { return (int)(((long long)j * n) >> k); }

// Batched use: a batch of 2^d0 tridiagonals of size blk is treated as one virtual problem of size n = blk 2^d0 whose
// top d0 tree levels are never merged; eigenvector blocks are then stored compactly (ldz >= blk rows, n columns):
// the ROW offset of a node is taken inside its top-level block.  Single matrix: blk = n, row offset = lo.
__host__ __device__ __forceinline__ int row_off(int lo, int blk) { return lo - (lo / blk) * blk; }

int stedc_depth(int n) {
    int D = 0;
    while (((n + (1 << D) - 1) >> D) > kLeaf) ++D;
    return D;
}

// ---- K0: scale T to unit max-norm by an exact power of two (the deflation tolerances below
// assume ||T|| ~ 1, as LAPACK's dstedc does) and remove the rank-one tears from the diagonal -----
// (one CTA per top-level block: every matrix of a batch gets its own scale)
__global__ void __launch_bounds__(1024) stedc_prepare_kernel(int n, int depth, int blk, const double *__restrict__ d, const double *__restrict__ e,
                                                             double *__restrict__ dmod, double *__restrict__ es, double *__restrict__ scal) {
    __shared__ double s_max[32];
    __shared__ double s_sigma;
    const int tid = threadIdx.x;
    const int b0 = blockIdx.x * blk, b1 = b0 + blk;
    scal += 2 * blockIdx.x;
    double m = 0.0;
    for (int i = b0 + tid; i < b1; i += 1024) {
        m = fmax(m, fabs(d[i]));
        if (i < n - 1) m = fmax(m, fabs(e[i]));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((tid & 31) == 0) s_max[tid >> 5] = m;
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < 32; ++w) m = fmax(m, s_max[w]);
        double sigma = 1.0;
        if (m > 0.0 && m < 1.7e308) {
            int ex;
            frexp(m, &ex);                 // m = f 2^ex, f in [0.5, 1)
            sigma = ldexp(1.0, -ex);       // sigma m in [0.5, 1)
        }
        s_sigma = sigma;
        scal[0] = sigma; scal[1] = 1.0 / sigma;
    }
    __syncthreads();
    const double sigma = s_sigma;
    // is x a leaf boundary?  x == bound(depth, ceil(x 2^depth / n))
    auto is_bound = [&](int x) -> bool {
        if (x <= 0 || x >= n) return false;
        const long long num = ((long long)x << depth);
        const int j = (int)((num + n - 1) / n);
        return node_bound(n, depth, j) == x;
    };
    for (int i = b0 + tid; i < b1; i += 1024) {
        double v = d[i] * sigma;
        const double ei = (i < n - 1) ? e[i] * sigma : 0.0;
        es[i] = ei;
        if (depth > 0) {
            if (is_bound(i + 1)) v -= fabs(ei);                       // i is the last index of a leaf
            if (is_bound(i)) v -= fabs(e[i - 1] * sigma);             // i is the first index of a leaf
        }
        dmod[i] = v;
    }
}

__global__ void stedc_unscale_kernel(int n, int blk, double *__restrict__ lam, const double *__restrict__ scal) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) lam[i] *= scal[2 * (i / blk) + 1];
}

// ---- K1: leaves -- implicit QL with Wilkinson shift in one warp -----------------------------
__global__ void __launch_bounds__(32) stedc_leaf_kernel(int n, int depth, const double *__restrict__ dmod, const double *__restrict__ e,
                                                        double *__restrict__ Z, int ldz, double *__restrict__ lam, int *info, int blk) {
    __shared__ double dd[kLeaf], ee[kLeaf], cs[kLeaf], sn[kLeaf];
    __shared__ double Zs[kLeaf * (kLeaf + 1)];
    __shared__ int ctrl[4];
    const int lane = threadIdx.x;
    const int lo = node_bound(n, depth, blockIdx.x), hi = node_bound(n, depth, blockIdx.x + 1);
    const int m = hi - lo;
    dd[lane] = (lane < m) ? dmod[lo + lane] : 0.0;
    ee[lane] = (lane < m - 1) ? e[lo + lane] : 0.0;
    for (int c = 0; c < kLeaf; ++c) Zs[c * (kLeaf + 1) + lane] = (c == lane) ? 1.0 : 0.0;
    double an = fabs(dd[lane]) + fabs(ee[lane]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) an = fmax(an, __shfl_xor_sync(0xffffffffu, an, o));
    __syncwarp();
    bool fail = false;
    for (int l = 0; l < m; ++l) {
        int iter = 0;
        for (;;) {
            // first negligible off-diagonal entry at or after l: every lane tests its own entry, one ballot (the serial scan by
            // lane 0 cost ~30 cycles per entry at the head of every QL iteration)
            int mm;
            {
                bool small = false;
                if (lane < m - 1) {
                    const double ae = fabs(ee[lane]);
                    small = ae <= kEps * (fabs(dd[lane]) + fabs(dd[lane + 1])) || ae <= kEps * an;
                }
                const unsigned hit = __ballot_sync(0xffffffffu, small) & (0xffffffffu << l);
                mm = hit ? __ffs(hit) - 1 : m - 1;
            }
            if (lane == 0) {
                int ilo = l;
                if (mm != l) {
                    double g = (dd[l + 1] - dd[l]) / (2.0 * ee[l]);
                    double r;
                    if (fabs(g) < 1e150) {                      // sqrt(g^2 + 1) from a refined reciprocal square root
                        const double x = fma(g, g, 1.0);
                        double ix = rsqrt(x);
                        ix = ix * fma(-0.5 * x * ix, ix, 1.5);
                        r = x * ix;
                    } else r = fabs(g);
                    g = dd[mm] - dd[l] + ee[l] / (g + copysign(r, g));
                    double s = 1.0, c = 1.0, p = 0.0;
                    int i;
                    bool under = false;
                    // the operands of step i are loaded one step ahead: the compiler cannot hoist the loads over the
                    // stores of the previous step (possible alias), and their latency would sit in the dependent chain
                    double e_i = ee[mm - 1], d_i = dd[mm - 1], d_i1 = dd[mm];
                    for (i = mm - 1; i >= l; --i) {
                        const double e_cur = e_i, d_cur = d_i, d_up = d_i1;
                        if (i > l) { e_i = ee[i - 1]; d_i = dd[i - 1]; }
                        const double f = s * e_cur, b = c * e_cur;
                        const double h2 = fma(f, f, g * g);
                        double ir;
                        if (h2 > 1e-280) {                      // T is scaled to unit max-norm: no overflow
                            ir = rsqrt(h2);
                            ir = ir * fma(-0.5 * h2 * ir, ir, 1.5);
                            r = h2 * ir;
                        } else {                                // squares underflowed: take the safe route
                            r = hypot(f, g);
                            ir = (r != 0.0) ? 1.0 / r : 0.0;
                        }
                        ee[i + 1] = r;
                        if (r == 0.0) { dd[i + 1] -= p; ee[mm] = 0.0; under = true; break; }
                        s = f * ir; c = g * ir;
                        g = d_up - p;
                        r = (d_cur - g) * s + 2.0 * c * b;
                        p = s * r;
                        dd[i + 1] = g + p;
                        d_i1 = d_cur;                            // dd[i] is untouched until the next step rewrites it
                        g = c * r - b;
                        cs[i] = c; sn[i] = s;
                    }
                    if (under) ilo = i + 1;
                    else { dd[l] -= p; ee[l] = g; ee[mm] = 0.0; }
                }
                ctrl[1] = ilo;
            }
            __syncwarp();
            const int ilo = ctrl[1];
            if (mm == l) break;
            if (++iter > 80) { fail = true; break; }
            if (lane < m && mm - 1 >= ilo) {
                // column ii of one rotation is column (ii-1)+1 of the next: carried in a register, not through shared memory
                double f = Zs[mm * (kLeaf + 1) + lane];
                for (int ii = mm - 1; ii >= ilo; --ii) {
                    const double q = Zs[ii * (kLeaf + 1) + lane];
                    Zs[(ii + 1) * (kLeaf + 1) + lane] = sn[ii] * q + cs[ii] * f;
                    f = cs[ii] * q - sn[ii] * f;
                }
                Zs[ilo * (kLeaf + 1) + lane] = f;
            }
            __syncwarp();
        }
        if (fail) break;
    }
    if (fail && info && lane == 0) atomicMax(info, 2);
    __syncwarp();
    // ascending rank of each eigenvalue (ties by index), then scatter
    int rank = 0;
    if (lane < m) {
        const double v = dd[lane];
        for (int k = 0; k < m; ++k) rank += (dd[k] < v) || (dd[k] == v && k < lane);
        lam[lo + rank] = v;
    }
    __syncwarp();
    for (int c = 0; c < m; ++c) {
        const int rk = __shfl_sync(0xffffffffu, rank, c);
        if (lane < m) Z[(size_t)(lo + rk) * ldz + row_off(lo, blk) + lane] = Zs[c * (kLeaf + 1) + lane];
    }
}

// ---- M1: per-node merge set-up: z vector, sorted poles, deflation scan ----------------------
// nodeinfo[8*node + {0:K, 1:k1, 2:k2, 3:k3, 4:nrot, 5:ndefl}]
struct MergeArgs {
    int n, ldz, depth;                 // depth = depth of the PARENT nodes being formed
    int blk;                           // top-level block size (= n for a single matrix)
    const double *e;
    const double *Zin; double *Zout; double *Qw; double *U;
    const double *lam_in; double *lam_out;
    double *dt, *zt, *mu, *lamroot, *zhat, *dval, *rc, *rs, *rho;
    int *org, *grow, *gsrc, *dcol, *dest_root, *dest_defl, *rp, *rq, *nodeinfo, *info;
};

__device__ __forceinline__ int lower_bound_d(const double *a, int len, double v) {   // #{a[k] < v}
    int lo = 0, hi = len;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (a[mid] < v) lo = mid + 1; else hi = mid; }
    return lo;
}
__device__ __forceinline__ int upper_bound_d(const double *a, int len, double v) {   // #{a[k] <= v}
    int lo = 0, hi = len;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (a[mid] <= v) lo = mid + 1; else hi = mid; }
    return lo;
}

// exclusive prefix sum of one int per thread over a 256-thread block (every thread gets its offset and the total)
__device__ __forceinline__ int block_excl_scan256(int v, int *s_w, int &total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    __syncthreads();
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    int base = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) { const int t = s_w[w]; if (w < warp) base += t; tot += t; }
    total = tot;
    return base + inc - v;
}

__global__ void __launch_bounds__(256) stedc_merge_setup_kernel(MergeArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int node = blockIdx.x;
    const int lo = node_bound(a.n, a.depth, node), hi = node_bound(a.n, a.depth, node + 1);
    const int mid = node_bound(a.n, a.depth + 1, 2 * node + 1);
    const int N = hi - lo, n1 = mid - lo, n2 = hi - mid;
    const int ro = row_off(lo, a.blk);
    double *ds = reinterpret_cast<double *>(smem_raw);    // N: poles in ascending order
    double *zs = ds + N;                                   // N: weights in the same order
    int *src = reinterpret_cast<int *>(zs + N);            // N: source column (local) | type << 28
    int *list = src + N;                                   // N: kept (front) / deflated (back) sorted indices
    __shared__ double s_red[16];
    __shared__ int s_cnt[8];
    const int tid = threadIdx.x;
    const double beta = a.e[mid - 1];
    const double sgn = beta < 0.0 ? -1.0 : 1.0;
    const double rho = 2.0 * fabs(beta);
    const double *l1 = a.lam_in + lo, *l2 = a.lam_in + mid;
    double dmax = 0.0, zmax = 0.0;
    for (int t = tid; t < N; t += 256) {
        double z, v; int rank, typ;
        if (t < n1) {
            z = a.Zin[(size_t)(lo + t) * a.ldz + (mid - 1 - lo + ro)];
            v = l1[t]; rank = t + lower_bound_d(l2, n2, v); typ = 1;
        } else {
            z = sgn * a.Zin[(size_t)(lo + t) * a.ldz + (mid - lo + ro)];
            v = l2[t - n1]; rank = (t - n1) + upper_bound_d(l1, n1, v); typ = 3;
        }
        z *= 0.7071067811865476;
        ds[rank] = v; zs[rank] = z; src[rank] = t | (typ << 28);
        dmax = fmax(dmax, fabs(v)); zmax = fmax(zmax, fabs(z));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dmax = fmax(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
        zmax = fmax(zmax, __shfl_xor_sync(0xffffffffu, zmax, o));
    }
    if ((tid & 31) == 0) { s_red[tid >> 5] = dmax; s_red[8 + (tid >> 5)] = zmax; }
    __syncthreads();
    __shared__ double s_tol;
    __shared__ int s_w[8];
    if (tid == 0) {
        for (int w = 1; w < 8; ++w) { dmax = fmax(dmax, s_red[w]); zmax = fmax(zmax, s_red[8 + w]); }
        s_tol = 8.0 * kEps * fmax(dmax, zmax);
    }
    __syncthreads();
    const double tol = s_tol;
    // ---- parallel fast path: deflate the negligible weights; if no two surviving neighbours are close poles
    // (the usual case) nothing sequential is left.  Otherwise thread 0 redoes the scan with rotations below.
    bool fast;
    {
        const int chunk = (N + 255) / 256;
        const int r_lo = min(N, tid * chunk), r_hi = min(N, r_lo + chunk);
        int mine = 0;
        for (int r = r_lo; r < r_hi; ++r) mine += !(rho * fabs(zs[r]) <= tol);
        int ns;
        const int off = block_excl_scan256(mine, s_w, ns);
        int qs = off, it = r_lo - off;                       // next survivor slot, next deflated rank
        for (int r = r_lo; r < r_hi; ++r) {
            if (rho * fabs(zs[r]) <= tol) list[N - 1 - it++] = r;   // ascending r = ascending pole: i-th smallest at N-1-i
            else list[qs++] = r;
        }
        __syncthreads();
        int close = 0;
        for (int q = tid; q + 1 < ns; q += 256) {
            const int pj = list[q], r = list[q + 1];
            const double sv = zs[pj], cv = zs[r], t = ds[r] - ds[pj];
            close |= (fabs(t) * fabs(cv * sv) <= tol * (cv * cv + sv * sv));
        }
        fast = !__syncthreads_or(close);
        if (fast) {
            const int K = ns;
            const int ch2 = (K + 255) / 256;
            const int q_lo = min(K, tid * ch2), q_hi = min(K, q_lo + ch2);
            int n1 = 0, n2 = 0, n3 = 0;
            for (int q = q_lo; q < q_hi; ++q) { const int ty = src[list[q]] >> 28; n1 += (ty == 1); n2 += (ty == 2); n3 += (ty == 3); }
            int k1, k2, k3;
            int c1 = block_excl_scan256(n1, s_w, k1);
            int c2 = block_excl_scan256(n2, s_w, k2) + k1;
            int c3 = block_excl_scan256(n3, s_w, k3) + k1 + k2;
            for (int q = q_lo; q < q_hi; ++q) {
                const int ty = src[list[q]] >> 28;
                const int g = (ty == 1) ? c1++ : (ty == 2) ? c2++ : c3++;
                a.grow[lo + q] = g;
                a.gsrc[lo + g] = src[list[q]] & 0x0fffffff;
            }
            if (tid == 0) {
                int *ni = a.nodeinfo + 8 * node;
                ni[0] = K; ni[1] = k1; ni[2] = k2; ni[3] = k3; ni[4] = 0; ni[5] = N - K;
                a.rho[node] = rho;
                s_cnt[0] = K; s_cnt[1] = N - K;
            }
        }
    }
    if (!fast && tid == 0) {
        int K = 0, ndefl = 0, nrot = 0, pj = -1;
        // deflated sorted indices live at list[N-ndefl .. N-1], ascending value towards lower index reversed:
        // the i-th smallest deflated value is list[N-1-i]
        auto push_defl = [&](int idx) {
            const double v = ds[idx];
            int pos = N - 1 - ndefl;
            while (pos < N - 1 && ds[list[pos + 1]] > v) { list[pos] = list[pos + 1]; ++pos; }
            list[pos] = idx;
            ++ndefl;
        };
        // the candidate's pole and weight are carried in registers and those of row r + 1 are loaded one step ahead
        // (rotations only touch rows <= r): the serial chain per row loses three shared-memory latencies
        double zn = zs[0], dn = ds[0], zpj = 0.0, dpj = 0.0;
        for (int r = 0; r < N; ++r) {
            const double zr = zn, dr = dn;
            if (r + 1 < N) { zn = zs[r + 1]; dn = ds[r + 1]; }
            if (rho * fabs(zr) <= tol) { push_defl(r); continue; }
            if (pj < 0) { pj = r; zpj = zr; dpj = dr; continue; }
            double s = zpj, c = zr;
            const double t = dr - dpj;
            // |t c s| <= tol with c = z_r/tau, s = -z_pj/tau, tau^2 = z_r^2 + z_pj^2, tested without sqrt or division
            if (fabs(t) * fabs(c * s) <= tol * (c * c + s * s)) {
                const double tau = sqrt(c * c + s * s);      // weights are <= 1 in magnitude and > tol/rho: no over/underflow
                c /= tau; s = -s / tau;
                // close poles: rotate the weight of pj into r and deflate pj
                zs[r] = tau; zs[pj] = 0.0;
                a.rp[lo + nrot] = src[pj] & 0x0fffffff; a.rq[lo + nrot] = src[r] & 0x0fffffff;
                a.rc[lo + nrot] = c; a.rs[lo + nrot] = s; ++nrot;
                if ((src[pj] >> 28) != (src[r] >> 28)) src[r] = (src[r] & 0x0fffffff) | (2 << 28);
                const double tt = dpj * c * c + dr * s * s;
                const double dnew = dpj * s * s + dr * c * c;
                ds[r] = dnew;
                ds[pj] = tt;
                push_defl(pj);
                pj = r; zpj = tau; dpj = dnew;
            } else {
                list[K++] = pj;
                pj = r; zpj = zr; dpj = dr;
            }
        }
        if (pj >= 0) list[K++] = pj;
        int k1 = 0, k2 = 0, k3 = 0;
        for (int q = 0; q < K; ++q) { const int ty = src[list[q]] >> 28; k1 += (ty == 1); k2 += (ty == 2); k3 += (ty == 3); }
        int c1 = 0, c2 = k1, c3 = k1 + k2;
        for (int q = 0; q < K; ++q) {
            const int ty = src[list[q]] >> 28;
            const int g = (ty == 1) ? c1++ : (ty == 2) ? c2++ : c3++;
            a.grow[lo + q] = g;
            a.gsrc[lo + g] = src[list[q]] & 0x0fffffff;
        }
        int *ni = a.nodeinfo + 8 * node;
        ni[0] = K; ni[1] = k1; ni[2] = k2; ni[3] = k3; ni[4] = nrot; ni[5] = ndefl;
        a.rho[node] = rho;
        s_cnt[0] = K; s_cnt[1] = ndefl;
    }
    __syncthreads();
    const int K = s_cnt[0], ndefl = s_cnt[1];
    for (int q = tid; q < K; q += 256) { a.dt[lo + q] = ds[list[q]]; a.zt[lo + q] = zs[list[q]]; }
    for (int i = tid; i < ndefl; i += 256) {
        const int idx = list[N - 1 - i];
        a.dval[lo + i] = ds[idx]; a.dcol[lo + i] = src[idx] & 0x0fffffff;
    }
}

// ---- M2: apply the deflation rotations to the children's eigenvectors, gather kept columns ----
__global__ void __launch_bounds__(256) stedc_rotate_kernel(MergeArgs a) {
    const int node = blockIdx.y;
    const int lo = node_bound(a.n, a.depth, node), hi = node_bound(a.n, a.depth, node + 1);
    const int N = hi - lo;
    const int r = blockIdx.x * 256 + threadIdx.x;
    const int nrot = a.nodeinfo[8 * node + 4];
    if (r >= N || nrot == 0) return;
    double *Z = const_cast<double *>(a.Zin) + (size_t)lo * a.ldz + row_off(lo, a.blk) + r;    // row r of the node block
    for (int t = 0; t < nrot; ++t) {
        const int p = a.rp[lo + t], q = a.rq[lo + t];
        const double c = a.rc[lo + t], s = a.rs[lo + t];
        const double x = Z[(size_t)p * a.ldz], y = Z[(size_t)q * a.ldz];
        Z[(size_t)p * a.ldz] = c * x + s * y;
        Z[(size_t)q * a.ldz] = c * y - s * x;
    }
}

// Qw[:, g] = Z[:, gsrc[g]] for the K kept columns (grouped order); one CTA copies 256 rows of 8 columns
constexpr int kGatherCols = 8;
__global__ void __launch_bounds__(256) stedc_gather_kernel(MergeArgs a) {
    const int node = blockIdx.z;
    const int lo = node_bound(a.n, a.depth, node), hi = node_bound(a.n, a.depth, node + 1);
    const int N = hi - lo;
    const int K = a.nodeinfo[8 * node];
    const int g0 = blockIdx.y * kGatherCols;
    const int r = blockIdx.x * 256 + threadIdx.x;
    if (g0 >= K || r >= N) return;
    const double *__restrict__ Z = a.Zin + (size_t)lo * a.ldz + row_off(lo, a.blk) + r;
    double *__restrict__ Q = a.Qw + (size_t)lo * a.ldz + row_off(lo, a.blk) + r;
    double v[kGatherCols];
#pragma unroll
    for (int cc = 0; cc < kGatherCols; ++cc) {
        const int g = g0 + cc;
        v[cc] = (g < K) ? Z[(size_t)a.gsrc[lo + g] * a.ldz] : 0.0;
    }
#pragma unroll
    for (int cc = 0; cc < kGatherCols; ++cc) {
        const int g = g0 + cc;
        if (g < K) Q[(size_t)g * a.ldz] = v[cc];
    }
}

// ---- M3: secular equation, one warp per root ------------------------------------------------
// g(mu) = 1 + rho sum_j z_j^2 / (delta_j - mu),  delta_j = d_j - d_org,  lambda = d_org + mu.
struct SecEval { double g, psi, dpsi, phi, dphi, asum; };

// sum over the GL lanes of a group (GL = 32: the warp; GL = 8: a quarter warp, mask = the group's lanes: groups of one warp
// diverge freely, a shuffle only names its own group)
template <int GL>
__device__ __forceinline__ double group_sum(double v, unsigned mask) {
#pragma unroll
    for (int o = GL / 2; o > 0; o >>= 1) v += __shfl_xor_sync(mask, v, o);
    return v;
}

template <int GL>
__device__ __forceinline__ SecEval sec_eval(int K, int i, int org, double mu, double rho, const double *__restrict__ d, const double *__restrict__ z, int lane, unsigned mask) {
    double psi = 0.0, dpsi = 0.0, phi = 0.0, dphi = 0.0, asum = 0.0;
    const double dorg = d[org];
    for (int j = lane; j < K; j += GL) {
        const double del = (d[j] - dorg) - mu;
        const double t = z[j] / del;
        const double term = rho * z[j] * t, dterm = rho * t * t;
        if (j <= i) { psi += term; dpsi += dterm; } else { phi += term; dphi += dterm; }
        asum += fabs(term);
    }
    SecEval r;
    r.psi = group_sum<GL>(psi, mask); r.dpsi = group_sum<GL>(dpsi, mask); r.phi = group_sum<GL>(phi, mask); r.dphi = group_sum<GL>(dphi, mask);
    r.asum = group_sum<GL>(asum, mask);
    r.g = 1.0 + r.psi + r.phi;
    return r;
}

// root eta of  c + s/(D1 - eta) + S/(D2 - eta) = 0  inside (D1, D2)  (D1 < 0 < D2 relative to the
// current point, s, S >= 0); returns false if no usable root
__device__ __forceinline__ bool two_pole_step(double c, double s, double S, double D1, double D2, double &eta) {
    const double qa = c, qb = c * (D1 + D2) + s + S, qc = c * D1 * D2 + s * D2 + S * D1;   // qa e^2 - qb e + qc = 0
    if (qa == 0.0) {
        if (qb == 0.0) return false;
        eta = qc / qb;
    } else {
        double disc = qb * qb - 4.0 * qa * qc;
        if (disc < 0.0) disc = 0.0;
        const double q = 0.5 * (qb + copysign(sqrt(disc), qb));
        const double e1 = (q != 0.0) ? qc / q : 0.0, e2 = q / qa;
        const bool in1 = (e1 > D1 && e1 < D2), in2 = (e2 > D1 && e2 < D2);
        if (in1 && in2) eta = fabs(e1) < fabs(e2) ? e1 : e2;
        else if (in1) eta = e1;
        else if (in2) eta = e2;
        else return false;
    }
    return (eta > D1 && eta < D2) && (eta == eta);
}

// GL lanes per root: a warp for large nodes; a quarter warp for nodes of at most 128 poles (the batched medium path: a root's
// iteration is a latency chain, four roots per warp keep four times as many chains in flight)
template <int GL>
__global__ void __launch_bounds__(256) stedc_secular_kernel(MergeArgs a) {
    const int node = blockIdx.y;
    const int lo = node_bound(a.n, a.depth, node);
    const int K = a.nodeinfo[8 * node];
    const int lane = threadIdx.x & (GL - 1);
    const unsigned mask = (GL == 32) ? 0xffffffffu : (((1u << GL) - 1u) << ((threadIdx.x & 31) & ~(GL - 1)));
    const int i = blockIdx.x * (256 / GL) + (threadIdx.x / GL);
    if (i >= K) return;
    const double *d = a.dt + lo, *z = a.zt + lo;
    const double rho = a.rho[node];
    int org; double mu, blo, bhi;   // bracket blo < mu* < bhi in the shifted variable, g(blo) < 0 < g(bhi)
    const bool last = (i == K - 1);
    if (K == 1) {
        if (lane == 0) { a.mu[lo] = rho * z[0] * z[0]; a.org[lo] = 0; a.lamroot[lo] = d[0] + rho * z[0] * z[0]; }
        return;
    }
    if (!last) {
        const double gap = d[i + 1] - d[i];
        const SecEval m = sec_eval<GL>(K, i, i, 0.5 * gap, rho, d, z, lane, mask);
        const double ti = rho * z[i] * z[i], ti1 = rho * z[i + 1] * z[i + 1];
        const double c0 = m.g - (-2.0 * ti / gap) - (2.0 * ti1 / gap);
        double D1, D2;
        if (m.g > 0.0) { org = i; blo = 0.0; bhi = 0.5 * gap; D1 = 0.0; D2 = gap; }
        else { org = i + 1; blo = -0.5 * gap; bhi = 0.0; D1 = -gap; D2 = 0.0; }
        double eta;
        if (two_pole_step(c0, ti, ti1, D1, D2, eta) && eta > blo && eta < bhi) mu = eta;
        else mu = 0.5 * (blo + bhi);
    } else {
        double zz = 0.0;
        for (int j = lane; j < K; j += GL) zz += z[j] * z[j];
        zz = group_sum<GL>(zz, mask);
        org = K - 1; blo = 0.0; bhi = rho * zz;
        if (!(bhi > 0.0)) bhi = 1.0;
        // g at the upper bound is >= 0; start in the middle
        mu = 0.5 * bhi;
    }
    bool ok = false;
    for (int it = 0; it < 100; ++it) {
        const SecEval ev = sec_eval<GL>(K, i, org, mu, rho, d, z, lane, mask);
        if (ev.g < 0.0) blo = mu; else bhi = mu;
        const double err = kEps * (8.0 * (1.0 + ev.asum) + fabs(mu) * (ev.dpsi + ev.dphi));
        if (fabs(ev.g) <= err || !(ev.g == ev.g)) { ok = (ev.g == ev.g); break; }
        double eta; bool have;
        if (!last) {
            const double D1 = (d[i] - d[org]) - mu, D2 = (d[i + 1] - d[org]) - mu;
            const double s = ev.dpsi * D1 * D1, S = ev.dphi * D2 * D2;
            const double c = ev.g - ev.dpsi * D1 - ev.dphi * D2;
            have = two_pole_step(c, s, S, D1, D2, eta);
        } else {
            // one pole at d_{K-1}: c + s/(D1 - eta) = 0
            const double D1 = -mu, dg = ev.dpsi + ev.dphi;
            const double s = dg * D1 * D1, c = ev.g - dg * D1;
            have = (c > 0.0);
            if (have) eta = D1 + s / c;
        }
        double nm = have ? mu + eta : 0.0;
        if (!have || !(nm > blo && nm < bhi)) nm = 0.5 * (blo + bhi);
        if (nm == mu || bhi - blo <= 2.0 * kEps * fmax(fabs(blo), fabs(bhi))) { ok = true; mu = nm; break; }
        mu = nm;
    }
    if (lane == 0) {
        a.mu[lo + i] = mu; a.org[lo + i] = org; a.lamroot[lo + i] = d[org] + mu;
        if (!ok && a.info) atomicMax(a.info, 3);
    }
}

// ---- M4: z^ (Loewner / Gu-Eisenstat) and final sorted positions ------------------------------
template <int GL>
__global__ void __launch_bounds__(256) stedc_zhat_kernel(MergeArgs a) {
    const int node = blockIdx.y;
    const int lo = node_bound(a.n, a.depth, node), hi = node_bound(a.n, a.depth, node + 1);
    const int N = hi - lo;
    const int *ni = a.nodeinfo + 8 * node;
    const int K = ni[0], ndefl = ni[5];
    const int lane = threadIdx.x & (GL - 1);
    const unsigned mask = (GL == 32) ? 0xffffffffu : (((1u << GL) - 1u) << ((threadIdx.x & 31) & ~(GL - 1)));
    const int j = blockIdx.x * (256 / GL) + (threadIdx.x / GL);
    const double *d = a.dt + lo;
    if (j < K) {
        double p = 1.0;
        const double dj = d[j];
        for (int i = lane; i < K; i += GL) {
            const double del = (dj - d[a.org[lo + i]]) - a.mu[lo + i];      // d_j - lambda_i
            p *= (i == j) ? -del : del / (dj - d[i]);
        }
#pragma unroll
        for (int o = GL / 2; o > 0; o >>= 1) p *= __shfl_xor_sync(mask, p, o);
        if (lane == 0) a.zhat[lo + j] = copysign(sqrt(fabs(p)), a.zt[lo + j]);
    }
    // positions: thread t of the first CTAs handles element t
    const int t = blockIdx.x * 256 + threadIdx.x;
    if (t < K) {
        const double v = a.lamroot[lo + t];
        const int pos = t + lower_bound_d(a.dval + lo, ndefl, v);
        a.dest_root[lo + t] = pos; a.lam_out[lo + pos] = v;
    } else if (t < N && t - K < ndefl) {
        const int m = t - K;
        const double v = a.dval[lo + m];
        const int pos = m + upper_bound_d(a.lamroot + lo, K, v);
        a.dest_defl[lo + m] = pos; a.lam_out[lo + pos] = v;
    }
}

// ---- M5: secular eigenvectors U (rows in grouped order) and copy of the deflated columns ------
template <int GL>
__global__ void __launch_bounds__(256) stedc_form_u_kernel(MergeArgs a) {
    const int node = blockIdx.y;
    const int lo = node_bound(a.n, a.depth, node), hi = node_bound(a.n, a.depth, node + 1);
    const int N = hi - lo;
    const int *ni = a.nodeinfo + 8 * node;
    const int K = ni[0], ndefl = ni[5];
    const int lane = threadIdx.x & (GL - 1);
    const unsigned mask = (GL == 32) ? 0xffffffffu : (((1u << GL) - 1u) << ((threadIdx.x & 31) & ~(GL - 1)));
    const int w = blockIdx.x * (256 / GL) + (threadIdx.x / GL);
    const double *d = a.dt + lo;
    if (w < K) {
        const int i = w;
        const double dorg = d[a.org[lo + i]], mu = a.mu[lo + i];
        double ss = 0.0;
        for (int j = lane; j < K; j += GL) { const double u = a.zhat[lo + j] / ((d[j] - dorg) - mu); ss += u * u; }
        ss = group_sum<GL>(ss, mask);
        const double inv = 1.0 / sqrt(ss);
        double *Ucol = a.U + (size_t)(lo + i) * a.ldz + row_off(lo, a.blk);
        for (int j = lane; j < K; j += GL) Ucol[a.grow[lo + j]] = inv * (a.zhat[lo + j] / ((d[j] - dorg) - mu));
    } else if (w - K < ndefl && w < N) {
        const int m = w - K;
        const double *src = a.Zin + (size_t)(lo + a.dcol[lo + m]) * a.ldz + row_off(lo, a.blk);
        double *dst = a.Zout + (size_t)(lo + a.dest_defl[lo + m]) * a.ldz + row_off(lo, a.blk);
        for (int r = lane; r < N; r += GL) dst[r] = src[r];
    }
}

// ---- M6: Z_out[:, roots] = Qw * U, two real DMMA GEMMs per node (structural zeros skipped) ------
struct ScatterEpi {
    double *C; int ldc; const int *colmap;
    __device__ __forceinline__ void operator()(int i, int j, double re, double) const {
        C[(size_t)colmap[j] * ldc + i] = re;
    }
};

constexpr int DG_MI = 4, DG_NI = 4, DG_WM = 2, DG_WN = 2;   // 64 x 64 CTA tile, 4 warps

__global__ void __launch_bounds__(DG_WM *DG_WN * 32) stedc_gemm_kernel(MergeArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int node = blockIdx.z >> 1, half = blockIdx.z & 1;
    const int lo = node_bound(a.n, a.depth, node), hi = node_bound(a.n, a.depth, node + 1);
    const int mid = node_bound(a.n, a.depth + 1, 2 * node + 1);
    const int *ni = a.nodeinfo + 8 * node;
    const int K = ni[0], k1 = ni[1], k2 = ni[2], k3 = ni[3];
    GemmProblem<double, double> p;
    int rowbase;
    const int ro = row_off(lo, a.blk);
    if (half == 0) { p.M = mid - lo; p.K = k1 + k2; rowbase = ro; p.A = a.Qw + (size_t)lo * a.ldz + ro; p.B = a.U + (size_t)lo * a.ldz + ro; }
    else { p.M = hi - mid; p.K = k2 + k3; rowbase = mid - lo + ro; p.A = a.Qw + (size_t)(lo + k1) * a.ldz + (mid - lo + ro); p.B = a.U + (size_t)lo * a.ldz + ro + k1; }
    p.N = K; p.K2 = 0; p.A2 = nullptr; p.B2 = nullptr; p.lda = a.ldz; p.ldb = a.ldz; p.lda2 = 0; p.ldb2 = 0;
    if ((int)blockIdx.x * 64 >= p.M || (int)blockIdx.y * 64 >= p.N) return;
    ScatterEpi epi{a.Zout + (size_t)lo * a.ldz + rowbase, a.ldz, a.dest_root + lo};
    gemm_tile_body<double, double, MNMAJ, KMAJ, false, false, DG_MI, DG_NI, DG_WM, DG_WN, false>(p, blockIdx.x, blockIdx.y, smem_raw, epi);
}

// ---- host driver ----------------------------------------------------------------------------
static int g_stedc_init_dev = -1;
constexpr size_t kStedcGemmSmem = gemm_smem_bytes<double, double, MNMAJ, KMAJ, DG_MI, DG_NI, DG_WM, DG_WN>();

int stedc_init() {
    int dev = 0;
    cudaGetDevice(&dev);
    if (g_stedc_init_dev == dev) return 0;
    if (cudaFuncSetAttribute(stedc_merge_setup_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 24 * (kMaxLargeN + 1))   /* the top merge asks for 24 (n + 1) bytes */ != cudaSuccess) return HPSD_ECUDA_;
    if (cudaFuncSetAttribute(stedc_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStedcGemmSmem) != cudaSuccess) return HPSD_ECUDA_;
    g_stedc_init_dev = dev;
    return 0;
}

int launch_stedc(const StedcWs &w, const double *d, const double *e, double **lam_out, double **Z_out, cudaStream_t st) {
    const int n = w.n;
    int rc = stedc_init();
    if (rc) return rc;
    const int D = w.depth, d0 = w.d0, blk = w.blk;      // single matrix: d0 = 0, blk = n
    // zero both eigenvector buffers: the off-diagonal quadrants of every node block are structural zeros
    if (cudaMemsetAsync(w.Za, 0, sizeof(double) * (size_t)w.ldz * n, st) != cudaSuccess) return HPSD_ECUDA_;
    if (D > d0 && cudaMemsetAsync(w.Zb, 0, sizeof(double) * (size_t)w.ldz * n, st) != cudaSuccess) return HPSD_ECUDA_;
    stedc_prepare_kernel<<<n / blk, 1024, 0, st>>>(n, D, blk, d, e, w.dmod, w.es, w.scal);
    HPSD_LAUNCH_CHECK();
    e = w.es;    // everything below works on the scaled tridiagonal
    stedc_leaf_kernel<<<1 << D, 32, 0, st>>>(n, D, w.dmod, e, w.Za, w.ldz, w.lamA, w.info, blk);
    HPSD_LAUNCH_CHECK();
    double *Zin = w.Za, *Zout = w.Zb, *lin = w.lamA, *lout = w.lamB;
    for (int k = D - 1; k >= d0; --k) {
        const int nodes = 1 << k;
        const int per = 1 << (k - d0);                   // nodes per top-level block at this depth
        const int maxN = (blk + per - 1) / per + 1;
        MergeArgs a;
        a.n = n; a.ldz = w.ldz; a.depth = k; a.e = e; a.blk = blk;
        a.Zin = Zin; a.Zout = Zout; a.Qw = w.Qw; a.U = w.U; a.lam_in = lin; a.lam_out = lout;
        a.dt = w.dt; a.zt = w.zt; a.mu = w.mu; a.lamroot = w.lamroot; a.zhat = w.zhat; a.dval = w.dval;
        a.rc = w.rc; a.rs = w.rs; a.rho = w.rho;
        a.org = w.org; a.grow = w.grow; a.gsrc = w.gsrc; a.dcol = w.dcol; a.dest_root = w.dest_root; a.dest_defl = w.dest_defl;
        a.rp = w.rp; a.rq = w.rq; a.nodeinfo = w.nodeinfo; a.info = w.info;
        // a quarter warp per root / column in the secular, z^ and U kernels: pays when a level holds many small nodes (the
        // batched medium path: 20736 roots per level in config 2); with few roots a whole warp per root has the shorter chain
        const bool quarter = maxN <= 128 && (long long)nodes * maxN >= 8192;
        stedc_merge_setup_kernel<<<nodes, 256, (size_t)24 * maxN, st>>>(a);
        HPSD_LAUNCH_CHECK();
        stedc_rotate_kernel<<<dim3((maxN + 255) / 256, nodes), 256, 0, st>>>(a);
        HPSD_LAUNCH_CHECK();
        stedc_gather_kernel<<<dim3((maxN + 255) / 256, (maxN + kGatherCols - 1) / kGatherCols, nodes), 256, 0, st>>>(a);
        HPSD_LAUNCH_CHECK();
        if (quarter) stedc_secular_kernel<8><<<dim3((maxN + 31) / 32, nodes), 256, 0, st>>>(a);
        else stedc_secular_kernel<32><<<dim3((maxN + 7) / 8, nodes), 256, 0, st>>>(a);
        HPSD_LAUNCH_CHECK();
        if (quarter) stedc_zhat_kernel<8><<<dim3((maxN + 31) / 32, nodes), 256, 0, st>>>(a);
        else stedc_zhat_kernel<32><<<dim3((maxN + 7) / 8, nodes), 256, 0, st>>>(a);
        HPSD_LAUNCH_CHECK();
        if (quarter) stedc_form_u_kernel<8><<<dim3((maxN + 31) / 32, nodes), 256, 0, st>>>(a);
        else stedc_form_u_kernel<32><<<dim3((maxN + 7) / 8, nodes), 256, 0, st>>>(a);
        HPSD_LAUNCH_CHECK();
        const int mt = (maxN / 2 + 1 + 63) / 64, nt = (maxN + 63) / 64;
        stedc_gemm_kernel<<<dim3(mt, nt, 2 * nodes), DG_WM * DG_WN * 32, kStedcGemmSmem, st>>>(a);
        HPSD_LAUNCH_CHECK();
        double *t = Zin; Zin = Zout; Zout = t;
        t = lin; lin = lout; lout = t;
    }
    stedc_unscale_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, blk, lin, w.scal);
    HPSD_LAUNCH_CHECK();
    *lam_out = lin; *Z_out = Zin;
    return 0;
}

}  // namespace hpsd
