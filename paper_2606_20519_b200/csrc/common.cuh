// common.cuh -- shared device/host helpers for the hpsd CUDA library (sm_100a).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

namespace hpsd {

// complex FP64, interleaved (re, im); 16-byte aligned so one element is one LDG.128/LDS.128
struct __align__(16) cplx {
    double x, y;
};

__host__ __device__ __forceinline__ cplx mk(double x, double y) { cplx r; r.x = x; r.y = y; return r; }
__host__ __device__ __forceinline__ cplx conj_(cplx a) { return mk(a.x, -a.y); }
__host__ __device__ __forceinline__ cplx operator+(cplx a, cplx b) { return mk(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ cplx operator-(cplx a, cplx b) { return mk(a.x - b.x, a.y - b.y); }
__host__ __device__ __forceinline__ cplx operator*(cplx a, cplx b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__host__ __device__ __forceinline__ cplx operator*(double s, cplx a) { return mk(s * a.x, s * a.y); }
__host__ __device__ __forceinline__ double abs2(cplx a) { return a.x * a.x + a.y * a.y; }
// acc += a*b
__device__ __forceinline__ void cfma(cplx &acc, cplx a, cplx b) {
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a)*b
__device__ __forceinline__ void cfma_conj(cplx &acc, cplx a, cplx b) {
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
}

// L2-coherent loads (bypass L1) for data produced by other CTAs of the same kernel
__device__ __forceinline__ double ldcg_(const double *p) { return __ldcg(p); }
__device__ __forceinline__ cplx ldcg_(const cplx *p) { const double2 v = __ldcg(reinterpret_cast<const double2 *>(p)); return mk(v.x, v.y); }

// NaN / Inf contract (include/hpsd.h): a block whose input holds a non-finite value gets an all-NaN output block
// and info[b] = kInfoNonFinite; the arithmetic in between runs on a sanitised copy (zeros), so nothing downstream
// (sorts, searches, iteration counts) ever sees a NaN.
constexpr int kInfoNonFinite = 2;
__device__ __forceinline__ bool nonfinite(double x) { return !(fabs(x) <= 1.79769313486231570e308); }
__device__ __forceinline__ double nan_() { return __longlong_as_double(0x7ff8000000000000LL); }

constexpr double kSqrt2 = 1.4142135623730951;      // nearest double to sqrt(2)
constexpr double kEps = 2.220446049250313e-16;     // 2^-52

// svec layout (include/hpsd.h): start of column j of the lower triangle
__host__ __device__ __forceinline__ size_t svec_col_off(int n, int j) { return (size_t)j * (size_t)(2 * n - j); }

// svec input/output of one call.  Plain projection: x = in, out = P(x).  ADMM step, Eqs. (D33)-(D34)
// (PAPER.md:1466-1472): x = in - sub with in = u~ and sub = v;  out = u = P(x);  vout = sub - in + u.
// vout may alias sub, out may alias in: every element is read before it is written, by the same thread.
// Storage precision ("a fixed number of initial iterations is performed in single
// precision"): with f32 = 1 every svec of the call is stored as FP32 (complex64 entries, 4 n^2 bytes per block); the pointers
// below then address floats and must only be dereferenced through sv_ld / sv_st.  The arithmetic between load and store is
// FP64 on every route.
struct SvecIo {
    const double *in;
    const double *sub;     // nullptr for a plain projection
    double *out;
    double *vout;
    int f32;
};
__device__ __forceinline__ double sv_ld(const double *p, size_t i, int f32) {
    return f32 ? (double)reinterpret_cast<const float *>(p)[i] : p[i];
}
__device__ __forceinline__ void sv_st(double *p, size_t i, double v, int f32) {
    if (f32) reinterpret_cast<float *>(p)[i] = (float)v;
    else p[i] = v;
}
__device__ __forceinline__ double io_load(const SvecIo &io, size_t i) {
    double x = sv_ld(io.in, i, io.f32);
    if (io.sub) x -= sv_ld(io.sub, i, io.f32);
    return x;
}
__device__ __forceinline__ void io_store(const SvecIo &io, size_t i, double u) {
    if (io.sub) sv_st(io.vout, i, (sv_ld(io.sub, i, io.f32) - sv_ld(io.in, i, io.f32)) + u, io.f32);
    sv_st(io.out, i, u, io.f32);
}
// all n^2 svec entries of one block <- NaN (and the ADMM v update with it), by nthreads threads
__device__ __forceinline__ void io_fill_nan(const SvecIo &io, size_t base, int n, int tid, int nthreads) {
    for (size_t t = tid; t < (size_t)n * n; t += nthreads) io_store(io, base + t, nan_());
}
// element offset on a pointer that may address floats (never dereferenced as double in that case)
template <class P> inline P sv_adv(P p, long long off, int f32) {
    return f32 ? reinterpret_cast<P>(reinterpret_cast<uintptr_t>(p) + (uintptr_t)(off * 4)) : p + off;
}
inline SvecIo io_offset(const SvecIo &io, long long off) {
    SvecIo r = io;
    r.in = sv_adv(io.in, off, io.f32); r.out = sv_adv(io.out, off, io.f32);
    if (io.sub) { r.sub = sv_adv(io.sub, off, io.f32); r.vout = sv_adv(io.vout, off, io.f32); }
    return r;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ cplx warp_sum(cplx v) { return mk(warp_sum(v.x), warp_sum(v.y)); }

// Per-thread launch counter (hpsd_last_launch_count)
extern thread_local int g_launches;

#define HPSD_CUDA_OK(expr)                                        \
    do {                                                          \
        cudaError_t e__ = (expr);                                 \
        if (e__ != cudaSuccess) return HPSD_ECUDA_;               \
    } while (0)
constexpr int HPSD_ECUDA_ = -3;

#define HPSD_LAUNCH_CHECK()                                       \
    do {                                                          \
        ::hpsd::g_launches++;                                     \
        if (cudaPeekAtLastError() != cudaSuccess) return ::hpsd::HPSD_ECUDA_; \
    } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace hpsd
