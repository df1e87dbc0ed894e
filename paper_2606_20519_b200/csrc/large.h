// large.h -- internal interfaces of the large-block path (n > kJacobiMaxN):
// S1 unpack -> S2/S3 tridiagonalise -> S4 divide & conquer -> S5 back-transform -> S6-S8.
#pragma once
#include "common.cuh"

namespace hpsd {

constexpr int kNB = 32;       // tridiagonalisation panel width

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
};
int tridiag_init();
int tridiag_tile_size(int n);
size_t tridiag_tile_count(int n);
void tridiag_fill_tiles(int n, int2 *tiles_host);
int launch_tridiag(const TridiagWs &w, cudaStream_t st);

}  // namespace hpsd
