// largepath.h -- driver of the large-block path (S1..S8 for n > jacobi_max_n).
#pragma once
#include "common.cuh"

namespace hpsd {
int largepath_init();
size_t largepath_ws_bytes(int n);
// One block: svec in -> svec out.  scratch >= largepath_ws_bytes(n), 256-byte aligned.
// lane: -1 on the caller's stream; 0 .. kLargeLanes-1 when several blocks run next to each other on the library's lane
// streams (each lane has its own side stream for the compact-WY factors and needs its own scratch)
constexpr int kLargeLanes = 8;
int largepath_project(int n, const SvecIo &io, unsigned char *scratch, const int2 *tiles, int *info, cudaStream_t st, int lane = -1,
                      int panel_ctas = 0, int wide_panels = 0, cudaEvent_t wide_done = nullptr);   // panel lanes: large.h, TridiagWs
// S1+S2+S3 only (diagnostic / eigenvalue-only entry points).
int largepath_tridiag_only(int n, const double *in, double *d, double *e, unsigned char *scratch, const int2 *tiles, cudaStream_t st);
// S1 + S2 of the two-stage reduction only: the Hermitian band (2 kBW x n complex, element (i, j) at band[(i - j) + j 2 kBW]).
int largepath_band_only(int n, const double *in, cplx *band, unsigned char *scratch, cudaStream_t st);
extern int g_two_stage, g_two_stage_min_n;   // options "two_stage", "two_stage_min_n"
// S1..S4: ascending eigenvalues only.
int largepath_eigvals(int n, const double *in, double *lambda, unsigned char *scratch, const int2 *tiles, cudaStream_t st);
}  // namespace hpsd
