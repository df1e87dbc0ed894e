// approx.h -- NEXT-4: factorisation-free approximate projection (approx.cu)
#pragma once
#include "common.cuh"

namespace hpsd {
size_t approx_ws_bytes(int n);
// svec in -> svec out, one block; scratch >= approx_ws_bytes(n), 256-byte aligned
int launch_project_approx(int n, const double *in, double *out, int iterations, unsigned char *scratch, cudaStream_t st);
}  // namespace hpsd
