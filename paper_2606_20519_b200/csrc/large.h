// large.h -- internal interfaces of the large-block path (n > kJacobiMaxN):
// S1 unpack -> S2/S3 tridiagonalise -> S4 divide & conquer -> S5 back-transform -> S6-S8.
#pragma once
#include "common.cuh"

namespace hpsd {

constexpr int kNB = 32;       // tridiagonalisation panel width
constexpr int kMaxPanelCtas = 192;   // the cooperative panel kernel runs min(SM count, this) CTAs; sizes its per-CTA partial arrays

// ---- tridiag.cu ---------------------------------------------------------------
struct TridiagWs {
    int n, lda, ldw, ldp;
    cplx *A;        // lda x n, lower triangle in, reflectors out
    cplx *W;        // ldw x kNB
    double *d, *e;  // n, n
    cplx *tau;      // n
    cplx *PR, *PC;  // nblk x ldp each
    cplx *part;     // G x (2 kNB + 1)
    cplx *tot;      // 2 kNB
    double *qpart;  // G
    const int2 *tiles;
    // panel lanes (hpsd_api.cu): from panel `wide_panels` on the cooperative kernel runs on max_ctas CTAs (0: never capped;
    // the kernel needs >= 64); wide_done (may be null) is recorded on the stream after the last full-width panel
    int max_ctas = 0, wide_panels = 0;
    cudaEvent_t wide_done = nullptr;
};
int tridiag_init();
int tridiag_tile_size(int n);
size_t tridiag_tile_count(int n);
void tridiag_fill_tiles(int n, int2 *tiles_host);
int launch_tridiag(const TridiagWs &w, cudaStream_t st);

// ---- tridiag_cluster.cu: S1+S2+S3 in one 16-CTA cluster, matrix resident in distributed shared memory ----
extern int g_overlap_factors;            // option "overlap_factors" (default 1), largepath.cu
extern int g_cluster_tridiag;            // option "cluster_tridiag" (default 1)
int tridiag_cluster_init();
int tridiag_cluster_size_ok(int n);      // device-independent part of the test below
int tridiag_cluster_fits(int n);         // 1 when this device and this n are served by the cluster kernel
int launch_tridiag_cluster(const TridiagWs &w, const double *in, const double *sub, cudaStream_t st, int *nf = nullptr, int f32 = 0);


// ---- stedc.cu (S4) ------------------------------------------------------------
constexpr int kLeaf = 32;         // D&C leaves are solved by one warp each
constexpr int kMaxLargeN = 8192;  // shared-memory bound of the deflation scan (24 N bytes)

struct StedcWs {
    int n, ldz, depth;
    int blk, d0;                       // batched use: n = blk 2^d0 and the top d0 levels are never merged (single: blk = n, d0 = 0)
    double *Za, *Zb, *Qw, *U;          // ldz x n each (eigenvector ping-pong, gathered copy, secular vectors)
    double *lamA, *lamB;               // n: eigenvalue ping-pong
    double *dmod;                      // n: scaled diagonal with the rank-one tears removed
    double *es;                        // n: scaled sub-diagonal
    double *scal;                      // [sigma, 1/sigma] per top-level block: power-of-two scaling of T
    double *dt, *zt;                   // n: sorted non-deflated poles / weights per node segment
    double *mu, *lamroot, *zhat;       // n
    double *dval;                      // n: deflated eigenvalues (ascending) per node segment
    double *rc, *rs;                   // n: deflation rotations
    int *org, *grow, *gsrc, *dcol, *dest_root, *dest_defl, *rp, *rq;   // n each
    int *nodeinfo;                     // 8 ints per node: K, k1, k2, k3, nrot, ndefl
    double *rho;                       // per node
    int *info;                         // device flag (may be null)
};
int stedc_depth(int n);
size_t stedc_ws_doubles(int n, int ldz);   // helper for carving (doubles incl. int arrays)
int stedc_init();
// Eigen-decomposition of the real symmetric tridiagonal (d, e): on return *lam_out / *Z_out point
// at the ping-pong buffers that hold the ascending eigenvalues and the eigenvectors (ldz x n).
int launch_stedc(const StedcWs &w, const double *d, const double *e, double **lam_out, double **Z_out, cudaStream_t st);


// ---- backherk.cu (S5 back-transform, S6 clamp/scale, S7 HERK, S8 pack) --------------------------
constexpr int kNBT = 64;          // reflectors per compact-WY block in the back-transformation
constexpr int kSplitK = 8;        // split of the long K dimension of X = V^H Z

struct BackWs {
    int n, lda, ldz;
    int voff;          // reflector c has its unit entry at row c + voff: 1 (one-stage reduction) or the band width (two-stage, Q1)
    const cplx *A;     // reflectors V (lower part, cleaned), lda x n
    const cplx *tau;   // n (tau[n-1] = 0)
    cplx *VT;          // lda x n : V_b T_b per block
    cplx *Tm;          // nblocks x kNBT x kNBT : Gram, then T
    cplx *Zc;          // ldz x n : complex scaled eigenvectors of the positive part
    cplx *Xp;          // kSplitK x kNBT x n partial products
    cplx *X;           // kNBT x n
    int *cnt;          // [0] = p0 (#lambda <= 0), [1] = kpos, [2] = non-finite input flag (set by S1)
    int *info;         // per-block status word (may be null)
};
int backherk_init();
// lam ascending (n), Zt real eigenvectors of T (ldzt x n); writes the projection's svec (and the ADMM v update) through io.
struct TwoStageWs;
// ts != nullptr: two-stage reduction, Z <- Q1 (Q2 Z) with Q2 from the bulge chasing (backq2.cu, factors already formed)
int launch_back_herk(const BackWs &w, const double *lam, const double *Zt, int ldzt, const SvecIo &io, cudaStream_t st, bool factors_done = false,
                     const TwoStageWs *ts = nullptr);
// the part of S5 that needs the reflectors only (Gram, T_b, V_b T_b); launch_back_herk(..., factors_done = true) then skips it
int launch_bt_factors(const BackWs &w, cudaStream_t st);

}  // namespace hpsd
