// dtile.cuh -- the 128 x 128 DIAGONAL tile of the tile Cholesky (potrf_tiles.cu): L = chol(S) and W = L^-1 in shared
// memory (Eq. 10, at tile scale).  This is the serial spine of the factorisation: for one chain it is
// the critical path (one tile per 128 columns), for an ensemble of mid-size chains 10 % of the SM time, so it is built
// around the dependent-pivot chain:
//
//   right-looking over 8 panels of 16 columns; per panel p (k0 = 16 p):
//     A_p   warp 0 factors the 16 x 16 diagonal block in registers, one row per lane (warp_chol); warp 1 forms its
//           inverse 4 pivots behind (named barriers).  Meanwhile warps 2..7 apply panel p-1 to the columns >= k0 + 16
//           (C2_{p-1}: the part of the trailing update that the next block does not need).
//     B_p   rows below:  L[i][k0..k0+15] = A[i][k0..] W_pp^T                  (DMMA m8n8k4, all 8 warps)
//     C1_p  the NEXT block column only (columns k0+16..k0+31) -= L_p L_p^T    (DMMA), so that A_{p+1} can start
//   then W = L^-1 by doubling: for s = 16, 32, 64 and every pair of neighbouring s-blocks (a above c):
//     T = L_ca W_aa,  W_ca = -W_cc T                                           (DMMA, all pairs of a level at once)
//
//   Storage: ONE 128 x 129 array X holds L in its lower triangle (diagonal included) and W TRANSPOSED in its strict
//   upper triangle (W[i][j], i > j, at X[j][i]); the diagonal of W is rinv[i] = 1 / L_ii.  With the 64 x 65 scratch T the
//   whole working set is 167 KB and fits in the (idle) operand ring of the tile kernel.
//   Round-2 measurement behind this design: the 64 + 64 version on 32-pivot warp blocks took 70 us per tile, of which
//   4 x 17.5 k cycles were the inverse warp trailing a 32-pivot factor and ~25 k cycles sixteen small latency-bound
//   products between CTA barriers (profiles/r02_summary.md).
#pragma once
#include "bd_internal.cuh"
#include "warp_chol.cuh"

namespace dtile {

constexpr int N = 128;             // tile size
constexpr int LDX = 129;           // row stride of X (odd: rows and columns both conflict free for 8-byte accesses)
constexpr int PB = 16;             // panel width
constexpr int LDT = 65;            // row stride of the scratch T
constexpr int SMEM_DOUBLES = N * LDX + 64 * LDT + N + 64;     // X, T, rinv, column buffer of warp_chol

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// W[i][j] of the inverse under construction (valid where it has been computed)
__device__ __forceinline__ double w_el(const double* __restrict__ X, const double* __restrict__ rinv, int i, int j)
{
    return (i > j) ? X[j * LDX + i] : ((i == j) ? rinv[i] : 0.0);
}

// One 8 x 8 output tile of  sum_k A(row, k) B(k, col)  over k = 4 ks0 .. 4 ks1 - 1: lane (g, t) supplies A(8 mt + g, 4 ks + t)
// and B(4 ks + t, 8 nt + g) and receives elements (8 mt + g, 8 nt + 2 t + {0, 1}).  Two accumulator pairs (even / odd
// k-steps) halve the dependent DMMA chain.
template <class FA, class FB>
__device__ __forceinline__ void tile_mma(const int ks0, const int ks1, const int g, const int t, FA&& A, FB&& B, double& o0, double& o1)
{
    double e0 = 0.0, e1 = 0.0, f0 = 0.0, f1 = 0.0;
    int ks = ks0;
    for (; ks + 1 < ks1; ks += 2) {
        const double a0 = A(g, 4 * ks + t), b0 = B(4 * ks + t, g);
        const double a1 = A(g, 4 * ks + 4 + t), b1 = B(4 * ks + 4 + t, g);
        dmma(e0, e1, a0, b0);
        dmma(f0, f1, a1, b1);
    }
    if (ks < ks1) dmma(e0, e1, A(g, 4 * ks + t), B(4 * ks + t, g));
    o0 = e0 + f0;
    o1 = e1 + f1;
}

// Factor and invert.  On entry X holds the lower triangle of the SPD tile (rows / columns >= nloc: identity padding);
// on exit X = L (lower) and W^T (strict upper), rinv = diag(W).  All 8 consumer warps (256 threads) take part; sync() is
// their barrier.  row0 = 0-based global row of the tile (failing-pivot report in *sFail, 1-based, first failure wins).
template <class Sync>
__device__ __forceinline__ void factor_invert(double* __restrict__ X, double* __restrict__ T, double* __restrict__ rinv,
                                              double* __restrict__ sCol, const int lane, const int warp, const int row0, int* sFail,
                                              Sync&& sync)
{
    const int g = lane >> 2, t = lane & 3;

    // trailing update of the 8 x 8 tiles (mt, nt), nt <= mt, nt in [nt_lo, nt_hi), mt < 16, with panel p; the tiles are
    // dealt to `nw` warps, this one being number `w`
    auto update = [&](const int k0, const int nt_lo, const int nt_hi, const int w, const int nw) {
        int idx = 0;
        for (int nt = nt_lo; nt < nt_hi; ++nt)
            for (int mt = nt; mt < N / 8; ++mt, ++idx) {
                if (idx % nw != w) continue;
                double o0, o1;
                tile_mma(0, PB / 4, g, t, [&](int r, int k) { return X[(8 * mt + r) * LDX + k0 + k]; },
                         [&](int k, int c) { return X[(8 * nt + c) * LDX + k0 + k]; }, o0, o1);
                const int row = 8 * mt + g, col = 8 * nt + 2 * t;
                if (col <= row) X[row * LDX + col] -= o0;
                if (col + 1 <= row) X[row * LDX + col + 1] -= o1;
            }
    };

#pragma unroll 1
    for (int p = 0; p < N / PB; ++p) {
        const int k0 = PB * p;
        // ---- A_p (warps 0, 1)  ||  C2_{p-1} (warps 2..7) ------------------------------------------------------------
        if (warp == 0) {
            double x[PB];
#pragma unroll
            for (int j = 0; j < PB; ++j) {
                double v = (lane == j) ? 1.0 : 0.0;
                if (lane < PB) v = X[(k0 + max(lane, j)) * LDX + k0 + min(lane, j)];
                x[j] = v;
            }
            __syncwarp();
            const int f = warp_chol<PB, 4>(x, lane, sCol, rinv + k0, 1, [&](int k, double l) {
                if (lane < PB && lane >= k) X[(k0 + lane) * LDX + k0 + k] = l;       // the upper part belongs to W^T
            });
            if (lane == 0 && f != 0 && *sFail == 0) *sFail = row0 + k0 + f;
        } else if (warp == 1) {
            warp_inverse_f<PB, 4>(lane, PB, rinv + k0, 1, [&](int k, int j) { return X[(k0 + k) * LDX + k0 + j]; },
                                  [&](int k, double v) {
                                      if (lane < k) X[(k0 + lane) * LDX + k0 + k] = v;       // W[k][lane], transposed
                                  });
        } else if (p > 0) {
            update(k0 - PB, (k0 + PB) / 8, N / 8, warp - 2, 6);
        }
        sync();
        // ---- B_p: rows below the block, L[i][k0 + c] = sum_{q <= c} A[i][k0 + q] W_pp[c][q] -----------------------------
        for (int mt = (k0 + PB) / 8 + warp; mt < N / 8; mt += 8) {
            double a[PB / 4];
#pragma unroll
            for (int ks = 0; ks < PB / 4; ++ks) a[ks] = X[(8 * mt + g) * LDX + k0 + 4 * ks + t];
            double o[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
            for (int nt = 0; nt < 2; ++nt)
#pragma unroll
                for (int ks = 0; ks < PB / 4; ++ks)
                    if (4 * ks <= 8 * nt + 7) dmma(o[nt][0], o[nt][1], a[ks], w_el(X, rinv, k0 + 8 * nt + g, k0 + 4 * ks + t));
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                X[(8 * mt + g) * LDX + k0 + 8 * nt + 2 * t] = o[nt][0];
                X[(8 * mt + g) * LDX + k0 + 8 * nt + 2 * t + 1] = o[nt][1];
            }
        }
        sync();
        // ---- C1_p: the next block column (16 columns) gets panel p now, the rest while the next block is factored ------
        if (k0 + PB < N) update(k0, (k0 + PB) / 8, (k0 + 2 * PB) / 8, warp, 8);
        sync();
    }

    // ---- W = L^-1 by doubling ---------------------------------------------------------------------------------------------
#pragma unroll 1
    for (int s = PB; s < N; s *= 2) {
        const int st = s / 8, per_pair = st * st, npairs = N / (2 * s);
        // T = L_ca W_aa :  T[i][j] = sum_{k >= j} L[c0 + i][a0 + k] W[a0 + k][a0 + j]
        for (int idx = warp; idx < npairs * per_pair; idx += 8) {
            const int pr = idx / per_pair, rem = idx - pr * per_pair, mt = rem / st, nt = rem - mt * st;
            const int a0 = 2 * s * pr, c0 = a0 + s;
            double o0, o1;
            tile_mma(2 * nt, s / 4, g, t, [&](int r, int k) { return X[(c0 + 8 * mt + r) * LDX + a0 + k]; },
                     [&](int k, int c) { return w_el(X, rinv, a0 + k, a0 + 8 * nt + c); }, o0, o1);
            double* Tp = T + pr * s * LDT;
            Tp[(8 * mt + g) * LDT + 8 * nt + 2 * t] = o0;
            Tp[(8 * mt + g) * LDT + 8 * nt + 2 * t + 1] = o1;
        }
        sync();
        // W_ca = -W_cc T :  W[c0 + i][a0 + j] = -sum_{k <= i} W[c0 + i][c0 + k] T[k][j], stored transposed
        for (int idx = warp; idx < npairs * per_pair; idx += 8) {
            const int pr = idx / per_pair, rem = idx - pr * per_pair, mt = rem / st, nt = rem - mt * st;
            const int a0 = 2 * s * pr, c0 = a0 + s;
            const double* Tp = T + pr * s * LDT;
            double o0, o1;
            tile_mma(0, 2 * mt + 2, g, t, [&](int r, int k) { return w_el(X, rinv, c0 + 8 * mt + r, c0 + k); },
                     [&](int k, int c) { return Tp[k * LDT + 8 * nt + c]; }, o0, o1);
            X[(a0 + 8 * nt + 2 * t) * LDX + c0 + 8 * mt + g] = -o0;
            X[(a0 + 8 * nt + 2 * t + 1) * LDX + c0 + 8 * mt + g] = -o1;
        }
        sync();
    }
}

}  // namespace dtile
