// noalloc.cu -- hpsd_project_static: the exact PSD-cone projection of a small batch of equal-size blocks
// with NO device allocation anywhere on the call: for callers that cannot call cudaMalloc (code under CUDA graph capture,
// tight serving loops, harnesses that forbid it).  It is the batched divide-and-conquer medium path of medium.cu
// (launch_meddc_project: one-CTA tridiagonalisation, S4 as one virtual tridiagonal, one-CTA back-transform + HERK + pack)
// run on a FIXED scratch area instead of the plan's workspace: the file-scope __device__ array below, which every GPU that
// loads the library holds until the process exits.
//
// The array's name is a host-side stand-in in host code, not a device address: the address handed to the kernels comes from
// cudaGetSymbolAddress, taken once per device with that device current (static_scratch()).
//
// Every call shares the array and finds the previous call's contents in it.  What has to start at zero is cleared on the
// caller's stream by every call (launch_meddc_project: d, e, the status words; launch_stedc: both eigenvector buffers);
// the offset tables at its head are rewritten by every call.  Calls that overlap on the GPU (two streams, two host threads
// on two streams) RACE on the array: the caller serialises them (one stream, or events).
#include <mutex>
#include "kernels.h"
#include "../../include/hpsd.h"

namespace hpsd {

constexpr size_t kStaticScratchBytes = (size_t)HPSD_STATIC_SCRATCH_BYTES;
constexpr int kStaticMaxN = HPSD_STATIC_MAX_N;
constexpr int kStaticMaxCount = HPSD_STATIC_MAX_COUNT;
static_assert(kStaticMaxN == kMedDcMaxN, "hpsd_project_static serves the sizes of the batched divide-and-conquer medium path");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr size_t kStaticHead = 512;      // offs (long long x count) | info indices (int x count), 256 bytes each
static_assert(sizeof(long long) * kStaticMaxCount <= 256 && sizeof(int) * kStaticMaxCount <= 256, "head of the static scratch");

// block i of the batch starts at svec offset i n^2 (include/hpsd.h: blocks are stored back to back) and reports to info[i]
__global__ void static_tables_kernel(int n, int count, long long *__restrict__ offs, int *__restrict__ idx) {
    const int i = threadIdx.x;
    if (i < count) { offs[i] = (long long)i * n * n; idx[i] = i; }
}

constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mu;
static unsigned char *g_static_ptr[kStaticMaxDevices];      // device address of g_static_scratch, per device

// device address of the array on the CURRENT device; kernel attributes of the medium path on first use
static int static_scratch(unsigned char **out) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HPSD_ECUDA;
    if (dev < 0 || dev >= kStaticMaxDevices) return HPSD_EINVAL;
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        if (medium_init() != 0) return HPSD_ECUDA;           // cudaFuncSetAttribute only
        unsigned char *p = nullptr;
        if (cudaGetSymbolAddress((void **)&p, g_static_scratch) != cudaSuccess || !p) { cudaGetLastError(); return HPSD_ECUDA; }
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return HPSD_OK;
}

}  // namespace hpsd

using namespace hpsd;

extern "C" int hpsd_project_static(int n, int count, const double *in_svec, double *out_svec, int *info_dev, void *stream) {
    g_launches = 0;
    if (n < 2 || count < 0) return HPSD_EINVAL;
    if (count == 0) return HPSD_OK;
    if (!in_svec || !out_svec) return HPSD_EINVAL;
    if (n > kStaticMaxN || count > kStaticMaxCount) return HPSD_ETOOLARGE;
    if (kStaticHead + meddc_ws_bytes(n, count) > kStaticScratchBytes) return HPSD_ETOOLARGE;    // cannot happen within the two limits
    unsigned char *base = nullptr;
    int rc = static_scratch(&base);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    long long *offs = reinterpret_cast<long long *>(base);
    int *idx = reinterpret_cast<int *>(base + 256);
    static_tables_kernel<<<1, kStaticMaxCount, 0, st>>>(n, count, offs, idx);
    g_launches++;
    if (cudaPeekAtLastError() != cudaSuccess) return HPSD_ECUDA;
    if (info_dev && cudaMemsetAsync(info_dev, 0, sizeof(int) * (size_t)count, st) != cudaSuccess) return HPSD_ECUDA;
    const SvecIo io{in_svec, nullptr, out_svec, nullptr, 0};
    rc = launch_meddc_project(n, count, offs, io, base + kStaticHead, info_dev, idx, st);
    return rc == 0 ? HPSD_OK : (rc == -1 ? HPSD_EINVAL : HPSD_ECUDA);
}
