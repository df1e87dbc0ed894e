// twostage.h -- internal interfaces of the two-stage reduction and of the second
// back-transformation it needs in S5:
//   S2  he2hb.cu   dense Hermitian -> Hermitian band of width kBW: per panel a Householder QR inside one 16-CTA cluster,
//                  then the two-sided rank-2b trailing update as DMMA GEMMs (HEMM, small corrections, HER2K)
//   S3  hb2st.cu   band -> REAL symmetric tridiagonal by bulge chasing (one CTA per sweep, sweeps pipelined over the SMs)
//   S5' backq2.cu  Z <- Q2 Z: the kBW-long reflectors of S3 applied as diamond-shaped compact-WY blocks
// "Eigendecomposition" of PAPER.md:1536; the paper names no kernel (library call), BASELINE.json's north star asks for
// exactly this split.
#pragma once
#include "common.cuh"

namespace hpsd {

constexpr int kBW = 32;          // band width b of the intermediate band matrix = panel width of S2
constexpr int kQ2G = 32;         // sweeps per diamond block of the Q2 back-transformation
constexpr int kHemmSplitMax = 16;
constexpr int kTwoStageMinN = 96;   // smaller blocks never take the two-stage reduction (and get no workspace for it)
constexpr int kTwoStageMaxN = 4096 + 2 * kBW;   // rows of the first panel must fit the QR cluster's shared memory

struct TwoStageWs {
    int n, lda, ldv, ldab, ldz2;
    cplx *A;             // lda x n: FULL Hermitian matrix (both triangles), destroyed by S2
    cplx *V1;            // ldv x n: stage-1 reflectors; column c has its unit at row c + kBW, explicit zeros above
    cplx *tau1;          // n
    cplx *Tk;            // one kBW x kBW triangular factor per panel
    cplx *AB;            // ldab x n lower band, element (i, j) at AB[(i - j) + j ldab], 0 <= i - j < ldab = 2 kBW (room for the bulge)
    cplx *Zp;            // kHemmSplitMax x ldz2 x kBW: split-K partials of A22 V
    cplx *Z, *X;         // ldz2 x kBW
    cplx *Gp;            // per 64-row slab: kBW x kBW partial of V^H Z
    cplx *S;             // kBW x kBW: -1/2 T^H (V^H A22 V) T
    unsigned *counter;   // last-CTA-done counter of the slab kernel (self-resetting)
    // stage 2
    cplx *V2;            // reflector (sweep s, hop k) at V2[(k n + s) kBW ..], kBW entries (leading 1 explicit)
    cplx *tau2;          // tau2[k n + s]
    int *prog;           // hops completed per sweep (release/acquire flags)
    double *d, *e;       // the real tridiagonal
    cplx *T2;            // kQ2G x kQ2G triangular factor per diamond block
    int *q2flags;        // (n / 32 slabs) x (sweep groups): pipeline flags of the Q2 kernel
};

extern int g_he2hb_lookahead;                 // option "two_stage_lookahead" (default 1): panel QR of panel k+1 next to panel k's HER2K
int twostage_init();
int twostage_available();                     // 1 when 16-CTA clusters with the panel kernel's shared memory can be launched
size_t twostage_hops(int n);                  // max hops of a sweep = ceil((n - 1) / kBW)
size_t twostage_q2_blocks(int n);             // number of diamond blocks
int launch_he2hb(const TwoStageWs &w, cudaStream_t st);           // S2 (A must hold the full matrix)
int launch_hb2st(const TwoStageWs &w, cudaStream_t st);           // S3
int launch_q2_factors(const TwoStageWs &w, cudaStream_t st);      // T factors of the diamond blocks (needs V2, tau2 only)
// Zc (ldz x kpos complex, kpos = cnt[1] on the device) <- Q2 Zc
int launch_q2_apply(const TwoStageWs &w, cplx *Zc, int ldz, const int *cnt, cudaStream_t st);

}  // namespace hpsd
