// warp_chol.cuh -- the serial spine of the fused short-chain Cholesky: one small SPD block (NB <= 32 rows) is
// factored by ONE warp, one matrix row per lane, in registers (Eq. 10, at block scale), while
// a SECOND warp follows a few pivots behind and forms the inverse factor W = L^-1 by forward substitution.
//
// Why: the diagonal-block factorisation is the serial part of every blocked Cholesky (M dependent pivots per
// matrix).  Per pivot the dependency chain is
//     SHFL (pivot broadcast) -> rsqrt (approx + one cubic correction + one Newton step) -> DMUL -> DFMA (next pivot)
// ~ 130 cycles; everything else hangs off that chain.  Measured (profiles/r01_summary.md): a version that also
// carried the inverse in the same warp executed ~95 instructions per pivot at IPC 0.2 (566 cycles per pivot) --
// the time went into issue slots, not into the chain -- so the inverse moved to its own warp.
#pragma once
#include <cuda_runtime.h>

// 1/sqrt(d), d > 0 normal: hardware seed (rsqrt.approx.ftz.f64, ~2^-20 or better) + one third-order step
// y (1 + e/2 + 3 e^2/8), e = 1 - d y^2, and one Newton step on top -> <= 1 ulp-level error.
__device__ __forceinline__ double fast_rsqrt_pos(double d)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
    double t = d * y;
    double e = fma(-t, y, 1.0);
    double p = fma(0.375, e, 0.5);
    double q = e * p;
    y = fma(y, q, y);
    t = d * y;
    e = fma(-t, y, 1.0);
    y = fma(0.5 * y, e, y);
    return y;
}

// named-barrier producer / consumer pair (PTX ISA, bar.arrive / bar.sync example): the producer's shared-memory
// stores before bar.arrive are visible to the consumer after its bar.sync on the same barrier
__device__ __forceinline__ void named_arrive(int id, int nthreads) { asm volatile("bar.arrive %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory"); }
__device__ __forceinline__ void named_sync(int id, int nthreads) { asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory"); }

// Right-looking elimination on x[] = row `lane` of the symmetric block (lanes >= NB hold zeros):
//     l_ik = a_ik / sqrt(d_k)   (column k of L, handed to store_l(k, l) by every lane, valid for lane >= k)
//     a_ij -= l_ik l_jk         (j > k), l_jk broadcast through s_col (double buffered, one __syncwarp per pivot)
// s_rinv[k] = 1/L_kk.  After pivots CH-1, 2CH-1, .. the warp arrives on named barrier bar0, bar0+1, .. (64 threads)
// so that the inverse warp can start on the finished rows.  Returns 0 or 1 + the first pivot with d <= 0 (or NaN).
template <int NB, int CH, class StoreL>
__device__ __forceinline__ int warp_chol(double (&x)[NB], const int lane, double* __restrict__ s_col,
                                         double* __restrict__ s_rinv, const int bar0, StoreL&& store_l)
{
    static_assert(NB <= 32 && (NB % 2) == 0 && (NB % CH) == 0, "warp_chol: NB even, <= 32, multiple of CH");
    int fail = 0;
    double d = __shfl_sync(0xffffffffu, x[0], 0);
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        if (!(d > 0.0) && fail == 0) fail = k + 1;
        const double rinv = fast_rsqrt_pos(d);
        const double l = x[k] * rinv;
        if (k + 1 < NB) {                                   // next pivot first: it is the critical path
            const double dn = fma(-l, l, x[k + 1 < NB ? k + 1 : k]);
            d = __shfl_sync(0xffffffffu, dn, k + 1);
        }
        store_l(k, l);
        if (lane == k) s_rinv[k] = rinv;
        const double lm = (lane > k) ? l : 0.0;
        double* col = s_col + (k & 1) * 32;
        col[lane] = lm;
        __syncwarp();
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
        if ((k + 1) % CH == 0) named_arrive(bar0 + k / CH, 64);
    }
    return fail;
}

// The same elimination with the rank-1 update DEFERRED by one pivot.  One warp issues in order, so in warp_chol every
// update FMA that follows the LDS of the column just broadcast stalls the whole warp, chain included (measured: 390
// cycles per pivot for a dependent chain of ~130: MUFU.RSQ64H, 10 FP64 ops, SHFL).  Here pivot k
//   - applies pivot k-1 to the columns j >= k+1 from REGISTERS (cp[], loaded one pivot ago: the data has arrived),
//   - takes the one value the chain needs now, l_{k+1,k}, by shuffle and updates column k+1 with it at once,
//   - issues the loads of column k (j >= k+2) for the next pivot.
// Costs NB more registers (cp[]); inside the tile kernel that pressure makes ptxas spill in the DMMA loops, so it is used
// only by the kernel instance for latency-bound factorisations (few tiles per column: the diagonal tiles are the
// critical path and the DMMA loops are not the limiter).
template <int NB, int CH, class StoreL>
__device__ __forceinline__ int warp_chol_deferred(double (&x)[NB], const int lane, double* __restrict__ s_col,
                                                  double* __restrict__ s_rinv, const int bar0, StoreL&& store_l)
{
    static_assert(NB <= 32 && (NB % 2) == 0 && (NB % CH) == 0, "warp_chol_deferred: NB even, <= 32, multiple of CH");
    int fail = 0;
    double d = __shfl_sync(0xffffffffu, x[0], 0);
    double lm_prev = 0.0;                     // this lane's l of pivot k-1 (0 for lanes <= k-1)
    double cp[NB];                            // column k-1 of L (cp[j] = l_{j,k-1}), valid for j >= k+1
#pragma unroll
    for (int j = 0; j < NB; ++j) cp[j] = 0.0;
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        if (!(d > 0.0) && fail == 0) fail = k + 1;
        const double rinv = fast_rsqrt_pos(d);
        const double l = x[k] * rinv;          // x[k] carries every pivot < k (pivot k-1 was applied eagerly below)
        if (k >= 1) {
#pragma unroll
            for (int j = k + 1; j < NB; ++j) x[j] = fma(-lm_prev, cp[j], x[j]);      // pivot k-1, deferred
        }
        if (k + 1 < NB) {
            const double dn = fma(-l, l, x[k + 1 < NB ? k + 1 : k]);
            d = __shfl_sync(0xffffffffu, dn, k + 1);
        }
        store_l(k, l);
        if (lane == k) s_rinv[k] = rinv;
        const double lm = (lane > k) ? l : 0.0;
        double* col = s_col + (k & 1) * 32;
        col[lane] = lm;
        __syncwarp();
        if (k + 1 < NB) {
            const double lk1 = __shfl_sync(0xffffffffu, lm, k + 1);                 // l_{k+1,k}: column k+1 is needed next
            x[k + 1 < NB ? k + 1 : k] = fma(-lm, lk1, x[k + 1 < NB ? k + 1 : k]);
        }
        // column k for the next pivot's deferred update (j >= k+2), 16-byte loads where the pair is aligned
        if ((k & 1) == 0) {
#pragma unroll
            for (int j = k + 2; j + 1 < NB; j += 2) {
                const double2 c2 = *reinterpret_cast<const double2*>(col + j);
                cp[j] = c2.x; cp[j + 1] = c2.y;
            }
        } else {
            if (k + 2 < NB) cp[k + 2 < NB ? k + 2 : k] = col[k + 2 < NB ? k + 2 : k];
#pragma unroll
            for (int j = k + 3; j + 1 < NB; j += 2) {
                const double2 c2 = *reinterpret_cast<const double2*>(col + j);
                cp[j] = c2.x; cp[j + 1] = c2.y;
            }
        }
        lm_prev = lm;
        if ((k + 1) % CH == 0) named_arrive(bar0 + k / CH, 64);
    }
    return fail;
}

// Inverse factor by forward substitution, lane c = column c of W = L^-1 (lower):
//     W[k][c] = (delta_kc - sum_{j<k} L[k][j] W[j][c]) / L[k][k]
// L(k, j) (j < k) and s_rinv[k] come from shared memory as broadcast loads once the factoring warp has arrived on the
// chunk's named barrier; rows k >= nrows (padding of a ragged block) are identity rows.  Row k goes to s_w[k*WS + c].
template <int NB, int CH, class LoadL, class StoreW>
__device__ __forceinline__ void warp_inverse_f(const int lane, const int nrows, const double* __restrict__ s_rinv, const int bar0,
                                               LoadL&& L, StoreW&& store_w)
{
    double w[NB];
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        if (k % CH == 0) named_sync(bar0 + k / CH, 64);
        double s0 = (lane == k) ? 1.0 : 0.0, s1 = 0.0;
        if (k < nrows) {
#pragma unroll
            for (int j = 0; j + 1 < k; j += 2) {
                s0 = fma(-L(k, j), w[j], s0);
                s1 = fma(-L(k, j + 1), w[j + 1], s1);
            }
            if (k & 1) s0 = fma(-L(k, k - 1 >= 0 ? k - 1 : 0), w[k - 1 >= 0 ? k - 1 : 0], s0);
            w[k] = (s0 + s1) * s_rinv[k];
        } else {
            w[k] = s0;
        }
        store_w(k, w[k]);                                   // W[k][lane]
    }
}

// the same with row k of W stored at s_w[k*WS + c]
template <int NB, int CH, int WS, class LoadL>
__device__ __forceinline__ void warp_inverse(const int lane, const int nrows, const double* __restrict__ s_rinv,
                                             double* __restrict__ s_w, const int bar0, LoadL&& L)
{
    warp_inverse_f<NB, CH>(lane, nrows, s_rinv, bar0, L, [&](int k, double v) {
        if (lane < NB) s_w[k * WS + lane] = v;
    });
}
