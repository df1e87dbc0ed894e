// largepath.cu -- large-block pipeline: S1 unpack -> S2/S3 tridiagonalise -> S4 D&C ->
// S6 clamp/scale -> S5 back-transform -> S7 HERK -> S8 pack.
#include "kernels.h"
#include "large.h"
#include "largepath.h"
#include "twostage.h"
#include "prof.h"

namespace hpsd {

namespace {

int g_sms = 0;
}  // namespace
int g_overlap_factors = 1;    // option "overlap_factors"
int g_two_stage = 0;          // option "two_stage": 0 one-stage reduction, 1 two-stage (S2 dense -> band, S3 bulge chasing) for every large block,
                              // 2 by size (route measured on B200)
int g_two_stage_min_n = 1024; // "two_stage" = 2: blocks of at least this size take the two-stage reduction
namespace {

struct LargeWs {
    TridiagWs t;
    StedcWs s;
    BackWs b;
    TwoStageWs q;
    size_t bytes;
};

bool use_two_stage(int n) {
    if (n < kTwoStageMinN || n > kTwoStageMaxN) return false;
    if (g_two_stage == 1) return twostage_available() != 0;
    if (g_two_stage == 2 && n >= g_two_stage_min_n) return twostage_available() != 0;
    return false;
}

// Carve the scratch area.  base may be nullptr (size query).
LargeWs carve(int n, unsigned char *base) {
    LargeWs w;
    size_t off = 0;
    auto take = [&](size_t bytes) -> unsigned char * {
        unsigned char *p = base ? base + off : nullptr;
        off += align_up(bytes, 256);
        return p;
    };
    auto dbl = [&](size_t cnt) { return reinterpret_cast<double *>(take(sizeof(double) * cnt)); };
    auto cpx = [&](size_t cnt) { return reinterpret_cast<cplx *>(take(sizeof(cplx) * cnt)); };
    auto itg = [&](size_t cnt) { return reinterpret_cast<int *>(take(sizeof(int) * cnt)); };
    const int N = (int)align_up((size_t)n, 8);
    const int ts = tridiag_tile_size(n);
    const int nblk = (n + ts - 1) / ts;
    const int G = kMaxPanelCtas;          // an upper bound, NOT the SM count of the device at hand: the size must not depend on whether init has run
    // ---- S2/S3
    w.t.n = n; w.t.lda = N; w.t.ldw = N; w.t.ldp = nblk * ts;
    w.t.A = cpx((size_t)N * n);
    w.t.W = cpx((size_t)N * kNB);
    w.t.d = dbl(N);
    w.t.e = dbl(N);
    w.t.tau = cpx(N);
    w.t.PR = cpx((size_t)nblk * w.t.ldp);
    w.t.PC = cpx((size_t)nblk * w.t.ldp);
    w.t.part = cpx((size_t)G * (2 * kNB + 1));
    w.t.tot = cpx(2 * kNB);
    w.t.qpart = dbl(G);
    w.t.tiles = nullptr;
    // ---- S4
    w.s.n = n; w.s.ldz = N; w.s.depth = stedc_depth(n); w.s.blk = n; w.s.d0 = 0;
    w.s.Za = dbl((size_t)N * n); w.s.Zb = dbl((size_t)N * n); w.s.Qw = dbl((size_t)N * n); w.s.U = dbl((size_t)N * n);
    w.s.lamA = dbl(N); w.s.lamB = dbl(N); w.s.dmod = dbl(N); w.s.es = dbl(N); w.s.scal = dbl(2); w.s.dt = dbl(N); w.s.zt = dbl(N);
    w.s.mu = dbl(N); w.s.lamroot = dbl(N); w.s.zhat = dbl(N); w.s.dval = dbl(N); w.s.rc = dbl(N); w.s.rs = dbl(N);
    w.s.org = itg(N); w.s.grow = itg(N); w.s.gsrc = itg(N); w.s.dcol = itg(N);
    w.s.dest_root = itg(N); w.s.dest_defl = itg(N); w.s.rp = itg(N); w.s.rq = itg(N);
    const int maxnodes = 1 << (w.s.depth > 0 ? w.s.depth - 1 : 0);
    w.s.nodeinfo = itg((size_t)8 * maxnodes);
    w.s.rho = dbl(maxnodes);
    w.s.info = nullptr;
    // ---- S5..S8
    const int nblocks = (n + kNBT - 1) / kNBT;
    w.b.n = n; w.b.lda = N; w.b.ldz = N; w.b.voff = 1;
    w.b.A = w.t.A; w.b.tau = w.t.tau;
    w.b.VT = cpx((size_t)N * n);
    w.b.Tm = cpx((size_t)nblocks * kNBT * kNBT);
    w.b.Zc = cpx((size_t)N * n);
    w.b.Xp = cpx((size_t)kSplitK * kNBT * align_up((size_t)n, kNBT));
    w.b.X = cpx((size_t)kNBT * n);
    w.b.cnt = itg(8);
    w.b.info = nullptr;
    // ---- two-stage reduction (S2 dense -> band, S3 band -> tridiagonal, Q2)
    w.q = TwoStageWs{};
    if (n >= kTwoStageMinN && n <= kTwoStageMaxN) {
        const size_t nk = twostage_hops(n);
        const size_t npan = (size_t)(n + kBW - 1) / kBW;
        w.q.n = n; w.q.lda = N; w.q.ldv = N; w.q.ldab = 2 * kBW; w.q.ldz2 = N;
        w.q.A = w.t.A;
        w.q.V1 = cpx((size_t)N * n);
        w.q.tau1 = cpx(N);
        w.q.Tk = cpx(npan * kBW * kBW);
        w.q.AB = cpx((size_t)2 * kBW * n);
        w.q.Zp = cpx((size_t)kHemmSplitMax * N * kBW);
        w.q.Z = cpx((size_t)N * kBW);
        w.q.X = cpx((size_t)N * kBW);
        w.q.Gp = cpx(((size_t)N / 64 + 1) * kBW * kBW);
        w.q.S = cpx((size_t)kBW * kBW);
        w.q.counter = reinterpret_cast<unsigned *>(itg(64));
        w.q.V2 = cpx(nk * n * kBW);
        w.q.tau2 = cpx(nk * n);
        w.q.prog = itg(N);
        w.q.d = w.t.d; w.q.e = w.t.e;
        w.q.T2 = cpx(twostage_q2_blocks(n) * kQ2G * kQ2G);
        w.q.q2flags = itg(((size_t)n / 32 + 1) * ((size_t)n / kQ2G + 1));
    }
    w.bytes = off;
    return w;
}

// Side stream of the large path: the compact-WY factors of S5 run next to the divide & conquer (fork after S2/S3,
// join before the back-transform; capturable in a CUDA graph like any fork/join of events).
struct Side {
    cudaStream_t st = nullptr;
    cudaEvent_t fork = nullptr, join = nullptr;
    int dev = -1;
};
constexpr int kSides = 1 + kLargeLanes;      // slot 0: the caller's stream, slots 1..: the lanes of concurrent blocks
thread_local Side g_sides[kSides];

bool side_ready(int slot) {
    Side &g_side = g_sides[slot];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    if (g_side.st && g_side.dev == dev) return true;
    if (g_side.st) { cudaStreamDestroy(g_side.st); cudaEventDestroy(g_side.fork); cudaEventDestroy(g_side.join); g_side = Side(); }
    if (cudaStreamCreateWithFlags(&g_side.st, cudaStreamNonBlocking) != cudaSuccess) { g_side = Side(); cudaGetLastError(); return false; }
    if (cudaEventCreateWithFlags(&g_side.fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&g_side.join, cudaEventDisableTiming) != cudaSuccess) {
        cudaStreamDestroy(g_side.st); g_side = Side(); cudaGetLastError(); return false;
    }
    g_side.dev = dev;
    return true;
}

int reduce_to_tridiagonal(LargeWs &w, int n, const double *in, const double *sub, cudaStream_t st, bool two_stage, int f32 = 0) {
    int *nf = w.b.cnt + 2;
    if (cudaMemsetAsync(w.b.cnt, 0, sizeof(int) * 8, st) != cudaSuccess) return HPSD_ECUDA_;
    if (two_stage) {
        if (cudaMemsetAsync(w.t.e, 0, sizeof(double) * (size_t)w.t.lda, st) != cudaSuccess) return HPSD_ECUDA_;
        prof_begin(ST_UNPACK, st);
        int rc = launch_unpack(n, in, sub, w.t.A, w.t.lda, 1, st, nf, f32);      // both triangles: the HEMM of S2 reads a plain full matrix
        prof_end(ST_UNPACK, st);
        if (rc) return rc;
        rc = launch_he2hb(w.q, st);
        if (rc) return rc;
        return launch_hb2st(w.q, st);
    }
    if (g_cluster_tridiag && tridiag_cluster_fits(n)) return launch_tridiag_cluster(w.t, in, sub, st, nf, f32);
    if (cudaMemsetAsync(w.t.tau, 0, sizeof(cplx) * (size_t)w.t.lda, st) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaMemsetAsync(w.t.e, 0, sizeof(double) * (size_t)w.t.lda, st) != cudaSuccess) return HPSD_ECUDA_;
    prof_begin(ST_UNPACK, st);
    int rc = launch_unpack(n, in, sub, w.t.A, w.t.lda, 0, st, nf, f32);
    prof_end(ST_UNPACK, st);
    if (rc) return rc;
    return launch_tridiag(w.t, st);
}

}  // namespace

int largepath_init() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HPSD_ECUDA_;
    if (cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return HPSD_ECUDA_;
    int rc = stedc_init();
    if (rc) return rc;
    return backherk_init();
}

size_t largepath_ws_bytes(int n) { return carve(n, nullptr).bytes; }

int largepath_tridiag_only(int n, const double *in, double *d, double *e, unsigned char *scratch, const int2 *tiles, cudaStream_t st) {
    LargeWs w = carve(n, scratch);
    w.t.tiles = tiles;
    int rc = reduce_to_tridiagonal(w, n, in, nullptr, st, use_two_stage(n));
    if (rc) return rc;
    if (cudaMemcpyAsync(d, w.t.d, sizeof(double) * n, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return HPSD_ECUDA_;
    if (n > 1 && cudaMemcpyAsync(e, w.t.e, sizeof(double) * (n - 1), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return HPSD_ECUDA_;
    return 0;
}

int largepath_band_only(int n, const double *in, cplx *band, unsigned char *scratch, cudaStream_t st) {
    LargeWs w = carve(n, scratch);
    if (n < kTwoStageMinN || n > kTwoStageMaxN) return -1;     // HPSD_EINVAL
    if (!twostage_available()) return HPSD_ECUDA_;
    int rc = launch_unpack(n, in, nullptr, w.t.A, w.t.lda, 1, st);
    if (rc) return rc;
    rc = launch_he2hb(w.q, st);
    if (rc) return rc;
    if (cudaMemcpyAsync(band, w.q.AB, sizeof(cplx) * (size_t)w.q.ldab * n, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return HPSD_ECUDA_;
    return 0;
}

int largepath_eigvals(int n, const double *in, double *lambda, unsigned char *scratch, const int2 *tiles, cudaStream_t st) {
    LargeWs w = carve(n, scratch);
    w.t.tiles = tiles;
    int rc = reduce_to_tridiagonal(w, n, in, nullptr, st, use_two_stage(n));
    if (rc) return rc;
    double *lam, *Z;
    rc = launch_stedc(w.s, w.t.d, w.t.e, &lam, &Z, st);
    if (rc) return rc;
    if (cudaMemcpyAsync(lambda, lam, sizeof(double) * n, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return HPSD_ECUDA_;
    return 0;
}

int largepath_project(int n, const SvecIo &io, unsigned char *scratch, const int2 *tiles, int *info, cudaStream_t st, int lane,
                      int panel_ctas, int wide_panels, cudaEvent_t wide_done) {
    const int slot = (lane >= 0 && lane < kLargeLanes) ? lane + 1 : 0;
    Side &g_side = g_sides[slot];
    LargeWs w = carve(n, scratch);
    w.t.tiles = tiles;
    w.t.max_ctas = panel_ctas; w.t.wide_panels = wide_panels; w.t.wide_done = wide_done;
    w.s.info = info;
    w.b.info = info;
    const bool ts = use_two_stage(n);
    if (ts) { w.b.A = w.q.V1; w.b.tau = w.q.tau1; w.b.voff = kBW; }
    int rc = reduce_to_tridiagonal(w, n, io.in, io.sub, st, ts, io.f32);
    if (rc) return rc;
    bool forked = false;
    if (g_overlap_factors && side_ready(slot) && cudaEventRecord(g_side.fork, st) == cudaSuccess &&
        cudaStreamWaitEvent(g_side.st, g_side.fork, 0) == cudaSuccess) {
        if (ts) rc = launch_q2_factors(w.q, g_side.st);
        if (!rc) rc = launch_bt_factors(w.b, g_side.st);
        forked = true;                                    // joined below even on error: a capture must not be left forked
        if (cudaEventRecord(g_side.join, g_side.st) != cudaSuccess && !rc) rc = HPSD_ECUDA_;
    }
    double *lam, *Z;
    prof_begin(ST_STEDC, st);
    int rc2 = launch_stedc(w.s, w.t.d, w.t.e, &lam, &Z, st);
    prof_end(ST_STEDC, st);
    if (forked && cudaStreamWaitEvent(st, g_side.join, 0) != cudaSuccess && !rc) rc = HPSD_ECUDA_;
    if (rc) return rc;
    if (rc2) return rc2;
    return launch_back_herk(w.b, lam, Z, w.s.ldz, io, st, forked, ts ? &w.q : nullptr);
}

}  // namespace hpsd
