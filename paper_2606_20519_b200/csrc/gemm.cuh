// gemm.cuh -- FP64 tensor-pipe (DMMA, mma.sync m8n8k4 f64) tile GEMM engine, sm_100a.
//
// tcgen05/wgmma have no FP64 kind, so "tensor pipe" for this path is the warp-level
// DMMA.8x8x4.  Complex products are four real DMMAs on the (re, im)
// halves of interleaved 16-byte elements: one LDS.128 yields both fragment halves.
//
// Operands are staged global -> shared with cp.async (zero-fill on ragged edges) in a
// 3-stage ring; shared pitches are chosen so every fragment LDS is bank-conflict free.
// One kernel template serves: HER2K (S2 trailing update), HERK + pack (S7/S8) and the
// real merges of the divide-and-conquer tridiagonal solver (S4).
#pragma once
#include "common.cuh"

namespace hpsd {

// D(8x8) += A(8x4, row) * B(4x8, col).  Lane T holds A[T/4][T%4], B[T%4][T/4],
// D[T/4][2(T%4)], D[T/4][2(T%4)+1].
__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async_16(void *smem, const void *g, bool valid) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(g), "r"(sz));
}
__device__ __forceinline__ void cp_async_8(void *smem, const void *g, bool valid) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    const int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(g), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

template <typename T> struct is_cplx { static constexpr bool v = false; };
template <> struct is_cplx<cplx> { static constexpr bool v = true; };

template <typename T>
__device__ __forceinline__ void cp_async_elem(T *smem, const T *g, bool valid) {
    if constexpr (is_cplx<T>::v) cp_async_16(smem, g, valid);
    else cp_async_8(smem, g, valid);
}

// Operand storage.  MNMAJ: element (mn, k) at base[mn + k*ld]   (column-major, not transposed)
//                   KMAJ : element (mn, k) at base[k + mn*ld]   (the operand is the (conj) transpose
//                          of a column-major matrix)
enum { MNMAJ = 0, KMAJ = 1 };

constexpr int kGemmBK = 16;
constexpr int kGemmStages = 3;

template <typename T, int LAYOUT, int EXT>
struct TileGeom {
    // pitch in elements; see header comment of this file for the bank analysis
    static constexpr int pitch = (LAYOUT == MNMAJ) ? (is_cplx<T>::v ? EXT + 2 : EXT + 4) : (kGemmBK + 4);
    static constexpr int elems = (LAYOUT == MNMAJ) ? kGemmBK * pitch : EXT * pitch;
};

// Cooperative copy of one EXT x BK operand tile.
template <typename T, int LAYOUT, int EXT, int NT>
__device__ __forceinline__ void load_tile(T *sm, const T *__restrict__ g, int ld, int mn0, int k0, int mn_lim, int k_lim, int tid) {
    constexpr int P = TileGeom<T, LAYOUT, EXT>::pitch;
    constexpr int TOT = EXT * kGemmBK;
#pragma unroll
    for (int it = 0; it < (TOT + NT - 1) / NT; ++it) {
        const int idx = tid + it * NT;
        if (TOT % NT != 0 && idx >= TOT) break;
        int mn, k;
        if (LAYOUT == MNMAJ) { mn = idx % EXT; k = idx / EXT; }
        else { k = idx % kGemmBK; mn = idx / kGemmBK; }
        const bool valid = (mn0 + mn < mn_lim) && (k0 + k < k_lim);
        const T *src = valid ? (LAYOUT == MNMAJ ? g + (size_t)(k0 + k) * ld + (mn0 + mn) : g + (size_t)(mn0 + mn) * ld + (k0 + k)) : g;
        T *dst = (LAYOUT == MNMAJ) ? sm + k * P + mn : sm + mn * P + k;
        cp_async_elem<T>(dst, src, valid);
    }
}

template <typename T, int LAYOUT, int EXT>
__device__ __forceinline__ T frag(const T *sm, int mn, int k) {
    constexpr int P = TileGeom<T, LAYOUT, EXT>::pitch;
    return (LAYOUT == MNMAJ) ? sm[k * P + mn] : sm[mn * P + k];
}

// One GEMM problem: C(MxN) (+)= op(A)(MxK) op(B)(KxN), optional second K segment (A2, B2, K2)
// accumulated into the same tile (HER2K = V W^H + W V^H).
template <typename TA, typename TB>
struct GemmProblem {
    const TA *A; const TB *B; const TA *A2; const TB *B2;
    int lda, ldb, lda2, ldb2;
    int M, N, K, K2;
};

// Accumulator fragment of one warp: MI x NI blocks of 8x8, complex or real.
template <bool CPLX, int MI, int NI>
struct Acc {
    double re[MI][NI][2];
    double im[CPLX ? MI : 1][CPLX ? NI : 1][2];
};

// Epilogue interface:  epi(row, col, re, im) called for every in-range element of the tile; an epilogue that
// declares `static constexpr bool kRmw = true` instead provides load(row, col) and store(row, col, old, re, im),
// and the tile body issues the loads of a row of blocks together.
template <class E, class = void> struct epi_is_rmw { static constexpr bool value = false; };
template <class E> struct epi_is_rmw<E, decltype((void)E::kRmw)> { static constexpr bool value = true; };

// LOWER: only tiles with (tile row block) >= (tile col block) are computed; the epilogue masks i<j.
template <typename TA, typename TB, int LA, int LB, bool CONJA, bool CONJB, int MI, int NI, int WM, int WN, bool LOWER, int STAGES = kGemmStages, class Epi>
__device__ __forceinline__ void gemm_tile_body(const GemmProblem<TA, TB> &p, int tile_m, int tile_n, unsigned char *smem_raw, Epi &epi) {
    constexpr bool CA = is_cplx<TA>::v, CB = is_cplx<TB>::v, CC = CA || CB;
    constexpr int BM = WM * MI * 8, BN = WN * NI * 8, NT = WM * WN * 32;
    using GA = TileGeom<TA, LA, BM>;
    using GB = TileGeom<TB, LB, BN>;
    TA *smA = reinterpret_cast<TA *>(smem_raw);
    TB *smB = reinterpret_cast<TB *>(smem_raw + sizeof(TA) * GA::elems * STAGES);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp % WM, wn = warp / WM;
    const int m0 = tile_m * BM, n0 = tile_n * BN;
    const int KT1 = (p.K + kGemmBK - 1) / kGemmBK;
    const int KT2 = (p.K2 + kGemmBK - 1) / kGemmBK;
    const int KT = KT1 + KT2;

    Acc<CC, MI, NI> acc;
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NI; ++j) {
            acc.re[i][j][0] = acc.re[i][j][1] = 0.0;
            if constexpr (CC) acc.im[i][j][0] = acc.im[i][j][1] = 0.0;
        }

    auto issue = [&](int kt) {
        if (kt < KT) {
            const int slot = kt % STAGES;
            if (kt < KT1) {
                load_tile<TA, LA, BM, NT>(smA + slot * GA::elems, p.A, p.lda, m0, kt * kGemmBK, p.M, p.K, tid);
                load_tile<TB, LB, BN, NT>(smB + slot * GB::elems, p.B, p.ldb, n0, kt * kGemmBK, p.N, p.K, tid);
            } else {
                load_tile<TA, LA, BM, NT>(smA + slot * GA::elems, p.A2, p.lda2, m0, (kt - KT1) * kGemmBK, p.M, p.K2, tid);
                load_tile<TB, LB, BN, NT>(smB + slot * GB::elems, p.B2, p.ldb2, n0, (kt - KT1) * kGemmBK, p.N, p.K2, tid);
            }
        }
        cp_async_commit();
    };

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) issue(s);

    const int fr = lane >> 2, fk = lane & 3;
    for (int kt = 0; kt < KT; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        issue(kt + STAGES - 1);
        const TA *sa = smA + (kt % STAGES) * GA::elems;
        const TB *sb = smB + (kt % STAGES) * GB::elems;
#pragma unroll
        for (int k4 = 0; k4 < kGemmBK; k4 += 4) {
            double ar[MI], ai[MI], br[NI], bi[NI];
#pragma unroll
            for (int i = 0; i < MI; ++i) {
                const TA v = frag<TA, LA, BM>(sa, wm * MI * 8 + i * 8 + fr, k4 + fk);
                if constexpr (CA) { ar[i] = v.x; ai[i] = CONJA ? -v.y : v.y; }
                else { ar[i] = v; ai[i] = 0.0; }
            }
#pragma unroll
            for (int j = 0; j < NI; ++j) {
                const TB v = frag<TB, LB, BN>(sb, wn * NI * 8 + j * 8 + fr, k4 + fk);
                if constexpr (CB) { br[j] = v.x; bi[j] = CONJB ? -v.y : v.y; }
                else { br[j] = v; bi[j] = 0.0; }
            }
#pragma unroll
            for (int i = 0; i < MI; ++i)
#pragma unroll
                for (int j = 0; j < NI; ++j) {
                    dmma(acc.re[i][j][0], acc.re[i][j][1], ar[i], br[j]);
                    if constexpr (CA && CB) dmma(acc.re[i][j][0], acc.re[i][j][1], -ai[i], bi[j]);
                    if constexpr (CB) dmma(acc.im[i][j][0], acc.im[i][j][1], ar[i], bi[j]);
                    if constexpr (CA) dmma(acc.im[i][j][0], acc.im[i][j][1], ai[i], br[j]);
                }
        }
    }
    cp_async_wait<0>();

    // epilogue: lane holds D[fr][2*fk + {0,1}] of each 8x8 block
    if constexpr (epi_is_rmw<Epi>::value) {
        // read-modify-write epilogues (C -= acc): a plain load/subtract/store per element is one dependent chain of
        // 2 MI NI global round trips per thread (a store may alias the next load, so the compiler keeps the order).
        // Here the 2 NI loads of one row of blocks are issued together, then their stores: MI round trips.
#pragma unroll
        for (int i = 0; i < MI; ++i) {
            const int row = m0 + wm * MI * 8 + i * 8 + fr;
            decltype(epi.load(0, 0)) old[NI][2];
#pragma unroll
            for (int j = 0; j < NI; ++j)
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const int col = n0 + wn * NI * 8 + j * 8 + 2 * fk + c;
                    if (row < p.M && col < p.N && (!LOWER || row >= col)) old[j][c] = epi.load(row, col);
                }
#pragma unroll
            for (int j = 0; j < NI; ++j)
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const int col = n0 + wn * NI * 8 + j * 8 + 2 * fk + c;
                    if (row < p.M && col < p.N && (!LOWER || row >= col)) {
                        if constexpr (CC) epi.store(row, col, old[j][c], acc.re[i][j][c], acc.im[i][j][c]);
                        else epi.store(row, col, old[j][c], acc.re[i][j][c], 0.0);
                    }
                }
        }
    } else {
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
            for (int j = 0; j < NI; ++j)
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const int row = m0 + wm * MI * 8 + i * 8 + fr;
                    const int col = n0 + wn * NI * 8 + j * 8 + 2 * fk + c;
                    if (row < p.M && col < p.N && (!LOWER || row >= col)) {
                        if constexpr (CC) epi(row, col, acc.re[i][j][c], acc.im[i][j][c]);
                        else epi(row, col, acc.re[i][j][c], 0.0);
                    }
                }
    }
}

template <typename TA, typename TB, int LA, int LB, int MI, int NI, int WM, int WN, int STAGES = kGemmStages>
constexpr size_t gemm_smem_bytes() {
    return (size_t)STAGES * (sizeof(TA) * TileGeom<TA, LA, WM * MI * 8>::elems + sizeof(TB) * TileGeom<TB, LB, WN * NI * 8>::elems);
}

}  // namespace hpsd
