// warp_chol.cuh -- Cholesky factor AND inverse factor of one small SPD block (NB <= 32 rows) by ONE warp,
// one matrix row per lane, everything in registers (Eq. 10, at block scale).
//
// Why: the diagonal-block factorisation is the serial spine of every blocked Cholesky (M dependent pivots
// per matrix).  The first version (a G x G thread grid, one CTA barrier and a full FP64 division per pivot)
// took ~1100 cycles per pivot (profiles/r01_baseline_first_path.md).  Here the per-pivot dependency chain is
//     SHFL (pivot broadcast) -> rsqrt (approx + one cubic correction) -> DMUL -> DFMA (next pivot, own lane)
// ~ 100 cycles, and everything else (the rank-1 update of the trailing columns, the update of the inverse)
// hangs off that chain: column k of L goes lane -> shared memory -> 16-byte broadcast loads.
//
// Right-looking elimination on x[] = row `lane`:   columns j > k hold the Schur complement a[lane][j],
// columns c <= k hold the (unscaled) inverse of the unit-lower factor, w[lane][c] -- the two triangles never
// overlap in time, so ONE register array of NB doubles carries both.  At pivot k
//     l_ik = a_ik / sqrt(d_k)             (final column k of L, handed to store_l)
//     a_ij -= l_ik l_jk                   (j > k)
//     w_i. -= (l_ik / sqrt(d_k)) w_k.     (c < k),   w_ik = -l_ik / sqrt(d_k)
// and at the end W = L^-1 has rows w_i. / sqrt(d_i).
#pragma once
#include <cuda_runtime.h>

// 1/sqrt(d), d > 0 normal: hardware seed (rsqrt.approx.ftz.f64, ~2^-20 or better) + one third-order step
// y (1 + e/2 + 3 e^2/8), e = 1 - d y^2, and one Newton step on top -> <= 1 ulp-level error
// (measured against rsqrt(): see tests).  9 dependent FP64 ops instead of the branchy library routine.
__device__ __forceinline__ double fast_rsqrt_pos(double d)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
    double t = d * y;
    double e = fma(-t, y, 1.0);
    double p = fma(0.375, e, 0.5);
    double q = e * p;
    y = fma(y, q, y);
#ifndef BD_RSQRT_ONE_STEP
    t = d * y;
    e = fma(-t, y, 1.0);
    y = fma(0.5 * y, e, y);
#endif
    return y;
}

// x[j]   in : A[lane][j] (symmetric block; only lanes < NB matter, lanes >= NB must hold zeros)
//        out: W[lane][j] = (L^-1)[lane][j] for j <= lane, 0 for j > lane
// s_col  : shared, 2*32 doubles, 16-byte aligned (column broadcast buffer, double buffered)
// s_wrow : shared, NB rows of stride WS doubles (WS even, 16-byte aligned): scratch for the unscaled inverse rows
// store_l(k, l): called by every lane at pivot k with l = L[lane][k] (valid for lane >= k)
// returns 0, or 1 + the first pivot index with d <= 0 (or NaN); the results are then meaningless.
template <int NB, int WS, class StoreL>
__device__ __forceinline__ int warp_chol_inv(double (&x)[NB], const int lane, double* __restrict__ s_col,
                                             double* __restrict__ s_wrow, StoreL&& store_l)
{
    static_assert(NB <= 32 && (NB % 2) == 0 && (WS % 2) == 0, "warp_chol_inv: NB even, <= 32");
    int fail = 0;
    double my_rinv = 1.0;
    double d = __shfl_sync(0xffffffffu, x[0], 0);
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        // row k of the unscaled inverse (columns < k) is final: its owner publishes it
        if (lane == k) {
#pragma unroll
            for (int c = 0; c < k; c += 2)
                *reinterpret_cast<double2*>(s_wrow + k * WS + c) = make_double2(x[c], x[c + 1 < NB ? c + 1 : c]);
        }
        if (!(d > 0.0) && fail == 0) fail = k + 1;
        const double rinv = fast_rsqrt_pos(d);
        const double l = x[k] * rinv;
        if (lane == k) my_rinv = rinv;
        store_l(k, l);
        if (k + 1 < NB) {                                   // next pivot first: it is the critical path
            const double dn = fma(-l, l, x[k + 1 < NB ? k + 1 : k]);
            d = __shfl_sync(0xffffffffu, dn, k + 1);
        }
        const double lm = (lane > k) ? l : 0.0;
        double* col = s_col + (k & 1) * 32;
        col[lane] = lm;
        __syncwarp();
        const double m = lm * rinv;
        // Schur complement columns j > k
        if ((k + 1) & 1) {
            if (k + 1 < NB) x[k + 1 < NB ? k + 1 : k] = fma(-lm, col[k + 1], x[k + 1 < NB ? k + 1 : k]);
#pragma unroll
            for (int j = k + 2; j + 1 < NB; j += 2) {
                const double2 c2 = *reinterpret_cast<const double2*>(col + j);
                x[j] = fma(-lm, c2.x, x[j]);
                x[j + 1] = fma(-lm, c2.y, x[j + 1]);
            }
        } else {
#pragma unroll
            for (int j = k + 1; j + 1 < NB; j += 2) {
                const double2 c2 = *reinterpret_cast<const double2*>(col + j);
                x[j] = fma(-lm, c2.x, x[j]);
                x[j + 1] = fma(-lm, c2.y, x[j + 1]);
            }
        }
        // inverse columns c < k, then the new column k
#pragma unroll
        for (int c = 0; c + 1 < k; c += 2) {
            const double2 w2 = *reinterpret_cast<const double2*>(s_wrow + k * WS + c);
            x[c] = fma(-m, w2.x, x[c]);
            x[c + 1] = fma(-m, w2.y, x[c + 1]);
        }
        if (k & 1) x[k - 1 >= 0 ? k - 1 : 0] = fma(-m, s_wrow[k * WS + (k - 1 >= 0 ? k - 1 : 0)], x[k - 1 >= 0 ? k - 1 : 0]);
        x[k] = (lane == k) ? 1.0 : -m;
    }
#pragma unroll
    for (int c = 0; c < NB; ++c) x[c] *= my_rinv;
    return fail;
}
