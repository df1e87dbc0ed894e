// largepath.cu -- large-block pipeline: S1 unpack -> S2/S3 tridiagonalise -> S4 D&C ->
// S5 back-transform -> S6 clamp/scale -> S7 HERK -> S8 pack.
#include "kernels.h"
#include "large.h"
#include "largepath.h"

namespace hpsd {

namespace {

int g_sms = 0;

struct LargeWs {
    TridiagWs t;
    size_t bytes;
};

// Carve the scratch area.  base may be nullptr (size query).
LargeWs carve(int n, unsigned char *base) {
    LargeWs w;
    size_t off = 0;
    auto take = [&](size_t bytes) -> unsigned char * {
        unsigned char *p = base ? base + off : nullptr;
        off += align_up(bytes, 256);
        return p;
    };
    const int N = (int)align_up((size_t)n, 8);
    const int ts = tridiag_tile_size(n);
    const int nblk = (n + ts - 1) / ts;
    const int G = g_sms > 0 ? g_sms : 148;
    w.t.n = n; w.t.lda = N; w.t.ldw = N; w.t.ldp = nblk * ts;
    w.t.A = reinterpret_cast<cplx *>(take(sizeof(cplx) * (size_t)N * n));
    w.t.W = reinterpret_cast<cplx *>(take(sizeof(cplx) * (size_t)N * kNB));
    w.t.d = reinterpret_cast<double *>(take(sizeof(double) * (size_t)N));
    w.t.e = reinterpret_cast<double *>(take(sizeof(double) * (size_t)N));
    w.t.tau = reinterpret_cast<cplx *>(take(sizeof(cplx) * (size_t)N));
    w.t.PR = reinterpret_cast<cplx *>(take(sizeof(cplx) * (size_t)nblk * w.t.ldp));
    w.t.PC = reinterpret_cast<cplx *>(take(sizeof(cplx) * (size_t)nblk * w.t.ldp));
    w.t.part = reinterpret_cast<cplx *>(take(sizeof(cplx) * (size_t)G * (2 * kNB + 1)));
    w.t.tot = reinterpret_cast<cplx *>(take(sizeof(cplx) * 2 * kNB));
    w.t.qpart = reinterpret_cast<double *>(take(sizeof(double) * (size_t)G));
    w.t.tiles = nullptr;
    w.bytes = off;
    return w;
}

}  // namespace

int largepath_init() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return HPSD_ECUDA_;
    return 0;
}

size_t largepath_ws_bytes(int n) { return carve(n, nullptr).bytes; }

int largepath_tridiag_only(int n, const double *in, double *d, double *e, unsigned char *scratch, const int2 *tiles, cudaStream_t st) {
    LargeWs w = carve(n, scratch);
    w.t.tiles = tiles;
    int rc = launch_unpack(n, in, w.t.A, w.t.lda, 0, st);
    if (rc) return rc;
    rc = launch_tridiag(w.t, st);
    if (rc) return rc;
    if (cudaMemcpyAsync(d, w.t.d, sizeof(double) * n, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return HPSD_ECUDA_;
    if (n > 1 && cudaMemcpyAsync(e, w.t.e, sizeof(double) * (n - 1), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return HPSD_ECUDA_;
    return 0;
}

int largepath_project(int n, const double *in, double *out, unsigned char *scratch, const int2 *tiles, int *info, cudaStream_t st) {
    (void)n; (void)in; (void)out; (void)scratch; (void)tiles; (void)info; (void)st;
    return -1;   // S4..S8 land next
}

}  // namespace hpsd
