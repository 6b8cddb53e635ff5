// potf2_blocked.cuh -- k_potf2: Cholesky factor AND inverse factor of one nb x nb (nb <= 64) diagonal block per
// chain (Eq. 10, at block scale), the serial step between two tensor-core phases of bdk_potrf.
//
// The block is split 32 + 32:   A = [A11 . ; A21 A22]
//   1. L11 = chol(A11) by warp 0 (one row per lane, registers + shuffles, warp_chol.cuh) while warp 1 forms
//      W11 = L11^-1 by forward substitution 4 pivots behind it
//   2. L21 = A21 W11^T                      (8 warps, DMMA m8n8k4, operands in shared memory)
//   3. A22 -= L21 L21^T
//   4. L22 = chol(A22), W22 = L22^-1        (as step 1)
//   5. W21 = -W22 (L21 W11)
// The first version eliminated all 64 pivots with one CTA barrier per pivot and then inverted with 64 threads
// (37 us at c4, 66 us at c3 where 172 registers allowed one CTA per SM only); here the 64 dependent pivots run
// at the warp-level chain latency.  A non-positive (or NaN) pivot records info = 1-based global row.
#pragma once
#include "bd_internal.cuh"
#include "warp_chol.cuh"

namespace potf2 {

constexpr int HB = 32;            // half block
constexpr int SLDP = 68;          // row stride of the 64 x 64 working copies: (4 g + t) mod 16 is distinct over a half-warp, so the 8-byte DMMA fragment loads
                                  // of the products are conflict free (65 gave up to 4-way conflicts there; the column accesses of the factoring warp are 4-way now, once per pivot)

// out = sum_p X[i][p] * Y(j, p): product of two 32 x 32 operands held in shared memory on the FP64 tensor cores.
// Warp w owns output rows 8 (w & 3) .. +7 and columns 16 (w >> 2) .. +15 (two m8n8k4 accumulators, 8 k-steps);
// yt selects Y(j, p) = Y[p][j] (plain product X Y) or Y[j][p] (X Y^T).  Triangular operands carry explicit zeros.
// Lane (g, t) ends up with out[nn][0..1] = element (row 8 (w & 3) + g, column 16 (w >> 2) + 8 nn + 2 t + {0, 1}).
__device__ __forceinline__ void gemm32(const double* __restrict__ X, const double* __restrict__ Y, bool yt, int warp, int lane,
                                       double (&out)[2][2])
{
    const int g = lane >> 2, t = lane & 3, mt = warp & 3, nt0 = (warp >> 2) * 2;
    out[0][0] = out[0][1] = out[1][0] = out[1][1] = 0.0;
#pragma unroll
    for (int ks = 0; ks < HB / 4; ++ks) {
        const double a = X[(8 * mt + g) * SLDP + 4 * ks + t];
#pragma unroll
        for (int nn = 0; nn < 2; ++nn) {
            const int j = 8 * (nt0 + nn) + g, p = 4 * ks + t;
            const double b = yt ? Y[p * SLDP + j] : Y[j * SLDP + p];
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(out[nn][0]), "+d"(out[nn][1])
                         : "d"(a), "d"(b));
        }
    }
}

// The same for 64 x 64 operands (the 128 x 128 diagonal tile of the tile kernel, split 64 + 64): warp w owns output rows
// 16 (w & 3) .. +15 and columns 32 (w >> 2) .. +31 (2 x 4 accumulators, 16 k-steps).  Lane (g, t) ends up with
// out[mm][nn][0..1] = element (row 16 (w & 3) + 8 mm + g, column 32 (w >> 2) + 8 nn + 2 t + {0, 1}).
__device__ __forceinline__ void gemm64(const double* __restrict__ X, const double* __restrict__ Y, bool yt, int warp, int lane,
                                       double (&out)[2][4][2])
{
    const int g = lane >> 2, t = lane & 3, r0 = 16 * (warp & 3), c0 = 32 * (warp >> 2);
#pragma unroll
    for (int mm = 0; mm < 2; ++mm)
#pragma unroll
        for (int nn = 0; nn < 4; ++nn) out[mm][nn][0] = out[mm][nn][1] = 0.0;
#pragma unroll 4
    for (int ks = 0; ks < 16; ++ks) {
        double a[2];
#pragma unroll
        for (int mm = 0; mm < 2; ++mm) a[mm] = X[(r0 + 8 * mm + g) * SLDP + 4 * ks + t];
#pragma unroll
        for (int nn = 0; nn < 4; ++nn) {
            const int j = c0 + 8 * nn + g, p = 4 * ks + t;
            const double b = yt ? Y[p * SLDP + j] : Y[j * SLDP + p];
#pragma unroll
            for (int mm = 0; mm < 2; ++mm)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                             : "+d"(out[mm][nn][0]), "+d"(out[mm][nn][1])
                             : "d"(a[mm]), "d"(b));
        }
    }
}

// rows / columns o .. o+31 of the working copy: warp 0 factors (L back into S, 1 / L_kk into s_rinv); the inverse of that
// 32 x 32 factor is formed in Wm as 16 + 16 so that it ends right behind the factorisation instead of 7 k cycles later
// (a single warp inverting all 32 rows by substitution is slower than the factoring warp: 17.5 k against 10 k cycles,
// profiles/r02_summary.md):
//     warp 1   W11 = L11^-1   rows 0..15,  4 pivots behind the factoring warp           (named barriers 1..4)
//     warp 2   W22 = L22^-1   rows 16..31, 4 pivots behind                              (named barriers 5..8)
//              then W21 = -W22 (L21 W11): two 16 x 16 x 16 products on the tensor cores (named barrier 10: W11 is ready)
// Called from ONE place (a loop over the two halves): the fully unrolled pivot loops are ~1700 straight-line
// instructions, and a second inlined copy ran 4x slower.
template <bool DEFER>
__device__ __forceinline__ void factor_half(double* __restrict__ S, double* __restrict__ Wm, double* __restrict__ sCol,
                                            double* __restrict__ sRinv, const int o, const int lane, const int warp, const int j0,
                                            int* sFail)
{
    constexpr int QB = HB / 2;
    if (warp == 0) {
        double x[HB];
#pragma unroll
        for (int j = 0; j < HB; ++j) x[j] = S[(o + max(lane, j)) * SLDP + o + min(lane, j)];
        __syncwarp();
        auto store_l = [&](int k, double l) { S[(o + lane) * SLDP + o + k] = (lane >= k) ? l : 0.0; };
        int f;
        if constexpr (DEFER) f = warp_chol_deferred<HB, 4>(x, lane, sCol, sRinv + o, 1, store_l);
        else f = warp_chol<HB, 4>(x, lane, sCol, sRinv + o, 1, store_l);
        if (lane == 0 && f != 0 && *sFail == 0) *sFail = j0 + o + f;
    } else if (warp == 1) {
        warp_inverse_f<QB, 4>(lane, QB, sRinv + o, 1, [&](int k, int j) { return S[(o + k) * SLDP + o + j]; },
                              [&](int k, double v) {
                                  if (lane < QB) Wm[(o + k) * SLDP + o + lane] = v;
                              });
        named_arrive(10, 64);
    } else if (warp == 2) {
        const int o2 = o + QB;
        warp_inverse_f<QB, 4>(lane, QB, sRinv + o2, 1 + QB / 4, [&](int k, int j) { return S[(o2 + k) * SLDP + o2 + j]; },
                              [&](int k, double v) {
                                  if (lane < QB) Wm[(o2 + k) * SLDP + o2 + lane] = v;
                              });
        named_sync(10, 64);
        // T = L21 W11 (into the W21 area), then W21 = -W22 T; lane (g, t) holds elements (8 mt + g, 8 nt + 2 t + {0, 1})
        const int g = lane >> 2, t = lane & 3;
        double o4[2][2][2];
#pragma unroll
        for (int pass = 0; pass < 2; ++pass) {
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) {
                    double c0 = 0.0, c1 = 0.0;
#pragma unroll
                    for (int ks = 0; ks < QB / 4; ++ks) {
                        const int i = 8 * mt + g, k = 4 * ks + t, j = 8 * nt + g;
                        // pass 0: A = L21 (S), B = W11;  pass 1: A = W22, B = T (both in Wm)
                        const double av = pass ? Wm[(o2 + i) * SLDP + o2 + k] : S[(o2 + i) * SLDP + o + k];
                        const double bv = pass ? Wm[(o2 + k) * SLDP + o + j] : Wm[(o + k) * SLDP + o + j];
                        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                                     : "+d"(c0), "+d"(c1)
                                     : "d"(av), "d"(bv));
                    }
                    o4[mt][nt][0] = c0;
                    o4[mt][nt][1] = c1;
                }
            __syncwarp();
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) {
                    double* dst = Wm + (o2 + 8 * mt + g) * SLDP + o + 8 * nt + 2 * t;
                    dst[0] = pass ? -o4[mt][nt][0] : o4[mt][nt][0];
                    dst[1] = pass ? -o4[mt][nt][1] : o4[mt][nt][1];
                }
            __syncwarp();
        }
    }
}

// Factor AND invert one 64 x 64 block held in shared memory: on entry S holds the lower triangle of the block (row stride
// SLDP), Wm is zero; on exit S = L (lower, zeros above the diagonal) and Wm = L^-1.  nh = 2 does both 32-column halves
// (steps 1-5 of the header), nh = 1 only the first (blocks of <= 32 rows, identity padded).  All 8 warps of the calling
// group take part; `sync()` is the barrier of that group (the whole CTA in k_potf2, a named barrier in the tile kernel).
// row0 = 0-based global row of the block (for the failing-pivot report in *sFail, 1-based).
//
// ONE copy of the factor / inverse code, run once per half: a second inlined copy (64 KB further into the kernel) ran 4x
// slower than the first one (22 k against 5.5 k cycles for the same 32 pivots -- instruction fetch of ~1700 straight-line
// instructions that are cold at every launch), a loop re-runs warm instructions.
template <bool DEFER = false, class Sync>
__device__ __forceinline__ void block64(double* __restrict__ S, double* __restrict__ Wm, double* __restrict__ sCol,
                                        double* __restrict__ sRinv, const int nh, const int lane, const int warp, const int row0,
                                        int* sFail, Sync&& sync)
{
    const int oi = 8 * (warp & 3) + (lane >> 2), oj = 16 * (warp >> 2) + 2 * (lane & 3);   // this lane's outputs: (oi, oj + 8 nn + {0, 1})
    double out[2][2];
#pragma unroll 1
    for (int hh = 0; hh < nh; ++hh) {
        factor_half<DEFER>(S, Wm, sCol, sRinv, hh * HB, lane, warp, row0, sFail);
        sync();
        if (hh == 0 && nh == 2) {
            gemm32(S + HB * SLDP, Wm, false, warp, lane, out);         // L21 = A21 W11^T
            sync();
#pragma unroll
            for (int nn = 0; nn < 2; ++nn)
#pragma unroll
                for (int e = 0; e < 2; ++e) S[(HB + oi) * SLDP + oj + 8 * nn + e] = out[nn][e];
            sync();
            gemm32(S + HB * SLDP, S + HB * SLDP, false, warp, lane, out);   // A22 -= L21 L21^T (lower part)
#pragma unroll
            for (int nn = 0; nn < 2; ++nn)
#pragma unroll
                for (int e = 0; e < 2; ++e)
                    if (oj + 8 * nn + e <= oi) S[(HB + oi) * SLDP + HB + oj + 8 * nn + e] -= out[nn][e];
            sync();
        }
    }
    if (nh == 2) {
        gemm32(S + HB * SLDP, Wm, true, warp, lane, out);          // T = L21 W11 -> the (still empty) W21 area
#pragma unroll
        for (int nn = 0; nn < 2; ++nn)
#pragma unroll
            for (int e = 0; e < 2; ++e) Wm[(HB + oi) * SLDP + oj + 8 * nn + e] = out[nn][e];
        sync();
        gemm32(Wm + HB * SLDP + HB, Wm + HB * SLDP, true, warp, lane, out);   // W21 = -W22 T
        sync();
#pragma unroll
        for (int nn = 0; nn < 2; ++nn)
#pragma unroll
            for (int e = 0; e < 2; ++e) Wm[(HB + oi) * SLDP + oj + 8 * nn + e] = -out[nn][e];
        sync();
    }
}

}  // namespace potf2
