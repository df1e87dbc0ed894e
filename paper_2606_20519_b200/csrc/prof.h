// prof.h -- optional per-stage CUDA-event timers (hpsd_set_option("profile", 1)).
// Events are recorded on the caller's stream around each stage of SURVEY.md §8(a); reading them
// (hpsd_profile_read) synchronises.  Off by default: the projection path then records nothing.
#pragma once
#include <cuda_runtime.h>

namespace hpsd {

enum Stage {
    ST_UNPACK = 0,      // S1
    ST_PANEL,           // S2/S3 panel kernel (one-stage: Householder vectors + Hermitian mat-vec; two-stage: panel QR)
    ST_HER2K,           // S2 trailing update (two-stage: HEMM + corrections + HER2K)
    ST_STEDC,           // S4
    ST_BACK,            // S5 + S6
    ST_HERK_PACK,       // S7 + S8
    ST_JACOBI,          // S9
    ST_MEDIUM,          // S10
    ST_SCALAR,          // n = 1 blocks
    ST_BULGE,           // S3 band -> tridiagonal (two-stage reduction)
    ST_BACKQ2,          // S5, second back-transformation (two-stage reduction)
    ST_COUNT
};

extern bool g_profile;
void prof_begin_(int stage, cudaStream_t st);
void prof_end_(int stage, cudaStream_t st);
inline void prof_begin(int stage, cudaStream_t st) { if (g_profile) prof_begin_(stage, st); }
inline void prof_end(int stage, cudaStream_t st) { if (g_profile) prof_end_(stage, st); }

}  // namespace hpsd
