// potrf.cu -- a3: in-place FP64 Cholesky D = L L^T of the lower triangle (Eq. 10),
// batched over chains.  The paper calls cusolverDnDpotrf once per chain per step (:172); this is a
// hand-written blocked right-looking factorisation for sm_100a:
//
//   outer panels of NB columns (right-looking trailing update, K = NB), each factored RECURSIVELY (left half,
//   update of the right half with K = half, right half) down to 64-column diagonal blocks:
//     k_potf2   64x64 diagonal block, register-resident, one CTA per chain, also forms W = L_jj^-1
//     k_trsm    rows below the diagonal block:  X = A W^T on the tensor cores
//     k_syrk    C -= P P^T with FP64 tensor-core DMMA (mma.sync m8n8k4), 128x128 tiles, cp.async operand
//               pipeline; K = 64, 128, 256, .. inside a panel, K = NB for the trailing update.
//
// FP64 has no tcgen05 kind; the FP64 tensor path on sm_100a is warp-level DMMA (measured 37.07
// TFLOP/s on B200), so operands go global -> cp.async -> padded smem -> registers.
// Matrices are ROW-major, lower triangle: L[i][j], j <= i, so both SYRK operands are K-contiguous
// rows of the same panel ("NT" form) and the DMMA A and B fragments use the same access pattern.
#include "bd_internal.cuh"
#include "potf2_blocked.cuh"

namespace {

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, int src_bytes)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}


// k_potf2 (64 x 64 diagonal blocks, one CTA per chain): the block is factored and inverted in shared memory by
// potf2::block64 (potf2_blocked.cuh)
constexpr int POTF2_SMEM = (2 * 64 * potf2::SLDP + 128) * (int)sizeof(double);

__global__ void __launch_bounds__(256) k_potf2(double* __restrict__ A_all, int64_t ld, int64_t stride, int j0, int nloc,
                                               int32_t* __restrict__ info, double* __restrict__ Winv)
{
    using namespace potf2;
    extern __shared__ __align__(16) double sm[];
    double* S = sm;                       // [64][SLDP] the block, then L (lower, zeros above the diagonal)
    double* Wm = S + 64 * SLDP;           // [64][SLDP] W = L^-1
    double* sCol = Wm + 64 * SLDP;        // [64] column broadcast buffer of warp_chol
    double* sRinv = sCol + 64;            // [64] 1 / L_kk
    __shared__ int sFail;
    const int c = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* A = A_all + (size_t)c * stride + (size_t)j0 * ld + j0;
    {
        double v[16];                                              // all 16 loads of a thread in flight at once
#pragma unroll
        for (int it = 0; it < 16; ++it) {
            const int idx = tid + 256 * it, i = idx >> 6, j = idx & 63;
            v[it] = (i == j) ? 1.0 : 0.0;                          // identity padding for a ragged block
            if (i < nloc && j <= i) v[it] = A[(size_t)i * ld + j];
        }
#pragma unroll
        for (int it = 0; it < 16; ++it) {
            const int idx = tid + 256 * it, i = idx >> 6, j = idx & 63;
            S[i * SLDP + j] = (j <= i) ? v[it] : 0.0;
            Wm[i * SLDP + j] = 0.0;
        }
    }
    if (tid == 0) sFail = 0;
    __syncthreads();

    block64(S, Wm, sCol, sRinv, (nloc > HB) ? 2 : 1, lane, warp, j0, &sFail, [] { __syncthreads(); });

    if (tid == 0 && sFail != 0 && info != nullptr && info[c] == 0) info[c] = sFail;
    for (int idx = tid; idx < 64 * 64; idx += 256) {
        const int r = idx >> 6, j = idx & 63;
        if (r < nloc && j <= r) A[(size_t)r * ld + j] = S[r * SLDP + j];
    }
    if (Winv != nullptr && nloc == 64) {
        double* W = Winv + (size_t)c * 64 * 64;
        for (int idx = tid; idx < 64 * 64; idx += 256) W[idx] = Wm[(idx >> 6) * SLDP + (idx & 63)];
    }
}


// =================================================================================================
// k_trsm: rows gi in [r_lo, r_hi) of the panel at columns [j0, j0+64): X L^T = A  <=>  X = A W^T with
// W = L^-1 (from k_potf2), i.e. X[r][c] = sum_{p <= c} A[r][p] W[c][p] -- a (rows x 64 x 64) product
// on the FP64 tensor cores instead of a serial substitution per row.  One CTA = 128 rows; A tile and W
// are staged once (cp.async) into shared memory with rows padded to 68 doubles (conflict-free 8-byte
// fragment loads); 8 warps = 4 (32 rows) x 2 (column blocks nt = 2i + wn, interleaved so that the
// triangular work 2(nt+1) k-steps per block balances); k-steps beyond the diagonal of W are skipped
// with real branches.  In place: the tile is fully in shared memory before anything is written.
// =================================================================================================
constexpr int TRSM_ROWS = 128;
constexpr int TRSM_SLD = 68;
constexpr int TRSM_SMEM = (TRSM_ROWS + 64) * TRSM_SLD * (int)sizeof(double);

template <int WN>
__device__ __forceinline__ void trsm_warp(const double* __restrict__ a_base, const double* __restrict__ w_base, double (&acc)[4][4][2])
{
#pragma unroll
    for (int ks = 0; ks < 16; ++ks) {
        double af[4];
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) af[mt] = a_base[mt * 8 * TRSM_SLD + ks * 4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            constexpr int dummy = 0; (void)dummy;
            const int nt = 2 * i + WN;                       // columns 8nt .. 8nt+7 need p <= 8nt+7
            if (4 * ks <= 8 * nt + 7) {
                const double bf = w_base[nt * 8 * TRSM_SLD + ks * 4];
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) dmma884(acc[mt][i][0], acc[mt][i][1], af[mt], bf);
            }
        }
    }
}

__global__ void __launch_bounds__(256, 2) k_trsm(double* __restrict__ A_all, int64_t ld, int64_t stride, int j0, int r_lo,
                                                  int r_hi, const double* __restrict__ Winv)
{
    extern __shared__ __align__(16) double smem[];
    double* sA = smem;                           // [128][68]
    double* sW = smem + TRSM_ROWS * TRSM_SLD;    // [64][68]
    const int nrb = (r_hi - r_lo + TRSM_ROWS - 1) / TRSM_ROWS;
    const int c = blockIdx.x / nrb;                        // chain and row block both on grid.x
    double* A = A_all + (size_t)c * stride;
    const double* W = Winv + (size_t)c * 64 * 64;
    const int row0 = r_lo + (blockIdx.x - c * nrb) * TRSM_ROWS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3, wm = warp & 3, wn = warp >> 2;
    {
        const int lrow = tid >> 5, lch = tid & 31;           // 32 chunks of 16 bytes per 64-double row
#pragma unroll
        for (int it = 0; it < TRSM_ROWS / 8; ++it) {
            const int rr = lrow + 8 * it;
            const int gi = row0 + rr;
            const bool ok = gi < r_hi;
            cp_async16(sA + (size_t)rr * TRSM_SLD + 2 * lch, A + (size_t)(ok ? gi : r_hi - 1) * ld + j0 + 2 * lch, ok ? 16 : 0);
        }
#pragma unroll
        for (int it = 0; it < 64 / 8; ++it) {
            const int rr = lrow + 8 * it;
            cp_async16(sW + (size_t)rr * TRSM_SLD + 2 * lch, W + (size_t)rr * 64 + 2 * lch, 16);
        }
        cp_async_commit();
        cp_async_wait<0>();
        __syncthreads();
    }
    double acc[4][4][2];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[mt][i][0] = acc[mt][i][1] = 0.0;
    const double* a_base = sA + (size_t)(wm * 32 + g) * TRSM_SLD + t;
    const double* w_base = sW + (size_t)g * TRSM_SLD + t;
    if (wn == 0) trsm_warp<0>(a_base, w_base, acc); else trsm_warp<1>(a_base, w_base, acc);
#pragma unroll
    for (int mt = 0; mt < 4; ++mt) {
        const int gi = row0 + wm * 32 + mt * 8 + g;
        if (gi >= r_hi) continue;
        double* xrow = A + (size_t)gi * ld + j0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int nt = 2 * i + wn;
            *reinterpret_cast<double2*>(xrow + nt * 8 + 2 * t) = make_double2(acc[mt][i][0], acc[mt][i][1]);
        }
    }
}

// =================================================================================================
// k_syrk: for gi in [lo, m_hi), gj in [lo, n_hi), gj <= gi:
//     A[gi][gj] -= sum_{p in [k_lo, k_lo+K)} A[gi][p] * A[gj][p]
// PERSISTENT: one CTA per SM walks the list of lower-triangular 128 x 128 tiles of all chains
// (tile = blockIdx.x, + gridDim.x, ...).  8 warps (4 along m x 2 along n), warp tile 32 x 64 = 4 x 8
// DMMA m8n8k4 accumulators (64 FP64 accumulators per thread).
//   - C is loaded STRAIGHT INTO the accumulators (negated) when a tile starts and stored (negated back)
//     when it ends: acc = -C + P P^T.  No load of C depends on anything in the epilogue, so the tensor
//     pipe never waits on a DRAM round trip there (the first version's epilogue took 28 % of the
//     kernel, profiles/r01_summary.md); the next tile's C is prefetched into L2 meanwhile.
//   - the operand pipeline (cp.async ring of 128 x BK slabs, BK = 32, 2 stages) runs ACROSS tile boundaries: the
//     load cursor is STAGES-1 k-slabs ahead of the compute cursor and simply moves on to the next tile.
//   smem rows are padded to BK + 8 doubles: the 16-byte fragment loads (two k-steps each) are conflict free.
// =================================================================================================
constexpr int BM = 128, BN = 128, NTW = BN / 16, SYRK_CTAS = 1, BK = 32, STAGES = 2, SLD = BK + 8;   // SLD % 16 == 8: conflict-free 16-byte fragment loads
constexpr int CPR = BK / 2, RPP = 256 / CPR;          // 16-byte chunks per slab row, rows copied per pass of the CTA
constexpr int SYRK_SMEM = STAGES * (BM + BN) * SLD * (int)sizeof(double);

struct SyrkArgs {
    double* A;
    int64_t ld, stride;
    int lo, m_hi, n_hi, k_lo, K;     // rows [lo, m_hi), columns [lo, n_hi), inner range [k_lo, k_lo+K)
    int TN, T2, tri, per_chain, total;   // tile columns, triangular tile rows, tiles in them, tiles per chain / launch
};

// tile index -> (chain, first row, first column).  Tiles (ty, tx), tx <= ty, tx < TN, row-major within a chain.
__device__ __forceinline__ void syrk_tile(const SyrkArgs& a, int idx, int& chain, int& tm0, int& tn0)
{
    chain = idx / a.per_chain;
    const int t = idx - chain * a.per_chain;
    // row ty of tiles has min(TN, R (ty + 1)) column tiles, R = BM / BN (tiles up to and including the diagonal)
    constexpr int R = BM / BN;
    int ty, tx;
    if (t < a.tri) {
        // rows 0 .. T2-1 are triangular: R (ty+1) tiles each, R ty (ty+1) / 2 before row ty
        ty = (int)((sqrt(8.0 * (double)t / R + 1.0) - 1.0) * 0.5);
        while (R * (ty + 1) * (ty + 2) / 2 <= t) ++ty;
        while (R * ty * (ty + 1) / 2 > t) --ty;
        tx = t - R * ty * (ty + 1) / 2;
    } else {
        const int u = t - a.tri;
        ty = a.T2 + u / a.TN;
        tx = u - (u / a.TN) * a.TN;
    }
    tm0 = a.lo + ty * BM;
    tn0 = a.lo + tx * BN;
}

__global__ void __launch_bounds__(256, SYRK_CTAS) k_syrk(const SyrkArgs a)
{
    extern __shared__ __align__(16) double smem[];
    double* sA = smem;                                   // [STAGES][BM][SLD]
    double* sB = smem + STAGES * BM * SLD;               // [STAGES][BN][SLD]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp & 3, wn = warp >> 2;
    const int g = lane >> 2, t = lane & 3;
    const int KT = a.K / BK;
    const int64_t ld = a.ld;

    // ---- load cursor (runs STAGES-1 slabs ahead of the compute cursor) -----------------------------
    // Per tile, each thread keeps ONE source pointer per operand (its first row, clamped into the matrix) and the
    // row stride between its passes; per slab a copy then costs one 64-bit add (the first version recomputed
    // chain * stride + row * ld per copy: ~120 integer instructions per slab in front of the DMMAs).
    int l_idx = blockIdx.x, l_kt = 0, l_tm0 = 0, l_tn0 = 0, l_chain = 0;
    const int lrow = tid / CPR, lch = tid % CPR;         // this thread copies rows lrow, lrow+RPP, .. chunk lch
    const int64_t pass_stride = (int64_t)RPP * ld;       // doubles between the rows of two passes
    const double* pA = a.A;
    const double* pB = a.A;
    auto set_tile = [&]() {
        syrk_tile(a, l_idx, l_chain, l_tm0, l_tn0);
        const double* base = a.A + (size_t)l_chain * a.stride + a.k_lo + 2 * lch;
        pA = base + (size_t)min(l_tm0 + lrow, a.m_hi - 1) * ld;
        pB = base + (size_t)min(l_tn0 + lrow, a.n_hi - 1) * ld;
    };
    if (l_idx < a.total) set_tile();
    auto load_next = [&](int slot) {
        if (l_idx < a.total) {
            const int kofs = l_kt * BK;
            double* dA = sA + ((size_t)slot * BM + lrow) * SLD + 2 * lch;
            double* dB = sB + ((size_t)slot * BN + lrow) * SLD + 2 * lch;
#pragma unroll
            for (int it = 0; it < BM / RPP; ++it) {
                const bool ok = l_tm0 + lrow + RPP * it < a.m_hi;
                cp_async16(dA + (size_t)it * RPP * SLD, pA + kofs + (ok ? it * pass_stride : 0), ok ? 16 : 0);
            }
#pragma unroll
            for (int it = 0; it < BN / RPP; ++it) {
                const bool ok = l_tn0 + lrow + RPP * it < a.n_hi;
                cp_async16(dB + (size_t)it * RPP * SLD, pB + kofs + (ok ? it * pass_stride : 0), ok ? 16 : 0);
            }
            if (++l_kt == KT) {
                l_kt = 0;
                l_idx += gridDim.x;
                if (l_idx < a.total) set_tile();
            }
        }
    };

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        load_next(s);
        cp_async_commit();
    }

    uint32_t git = 0;                                    // slabs consumed so far (ring position)
    for (int idx = blockIdx.x; idx < a.total; idx += gridDim.x) {
        int chain, tm0, tn0;
        syrk_tile(a, idx, chain, tm0, tn0);
        double* A = a.A + (size_t)chain * a.stride;
        // this warp's 32 x 64 block lies entirely above the diagonal -> no arithmetic (still loads/syncs)
        const bool warp_active = (tn0 + wn * (BN / 2)) <= (tm0 + wm * 32 + 31);

        // L2 prefetch of the NEXT tile's C (128 rows x 1 KB): its loads then cost an L2 hit, not a DRAM trip
        if (idx + (int)gridDim.x < a.total) {
            int nc, nm0, nn0;
            syrk_tile(a, idx + gridDim.x, nc, nm0, nn0);
            const double* Cn = a.A + (size_t)nc * a.stride;
#pragma unroll
            for (int it = 0; it < BN / 32; ++it) {
                const int q = tid + 256 * it;
                const int gr = nm0 + q / (BN / 16), gc = nn0 + (q % (BN / 16)) * 16;
                if (gr < a.m_hi && gc <= gr && gc < a.n_hi) prefetch_l2(Cn + (size_t)gr * ld + gc);
            }
        }

        double acc[4][NTW][2];
        if (warp_active) {
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const int gi = tm0 + wm * 32 + mt * 8 + g;
                const double* crow = A + (size_t)gi * ld;
#pragma unroll
                for (int nt = 0; nt < NTW; ++nt) {
                    const int gj = tn0 + wn * (BN / 2) + nt * 8 + 2 * t;
                    double c0 = 0.0, c1 = 0.0;
                    if (gi < a.m_hi) {
                        if (gj + 1 < a.n_hi && gj + 1 <= gi) {
                            const double2 cv = *reinterpret_cast<const double2*>(crow + gj);
                            c0 = cv.x; c1 = cv.y;
                        } else if (gj < a.n_hi && gj <= gi) {
                            c0 = crow[gj];
                        }
                    }
                    acc[mt][nt][0] = -c0;
                    acc[mt][nt][1] = -c1;
                }
            }
        }

        for (int kt = 0; kt < KT; ++kt, ++git) {
            cp_async_wait<STAGES - 2>();
            __syncthreads();
            load_next((git + STAGES - 1) % STAGES);
            cp_async_commit();
            if (warp_active) {
                // One 16-byte load per fragment row and PAIR of k-steps: within a group of 8 columns k-step 0 takes the
                // even columns (.x of lane t = column 2t), k-step 1 the odd ones (.y).  A and B use the same column
                // permutation, so the sum over k is the same set of products; half the shared-memory load instructions.
                const double* a_base = sA + ((size_t)(git % STAGES) * BM + wm * 32 + g) * SLD + 2 * t;
                const double* b_base = sB + ((size_t)(git % STAGES) * BN + wn * (BN / 2) + g) * SLD + 2 * t;
#pragma unroll
                for (int k8 = 0; k8 < BK / 8; ++k8) {
                    double2 af[4], bf[NTW];
#pragma unroll
                    for (int mt = 0; mt < 4; ++mt) af[mt] = *reinterpret_cast<const double2*>(a_base + mt * 8 * SLD + k8 * 8);
#pragma unroll
                    for (int nt = 0; nt < NTW; ++nt) bf[nt] = *reinterpret_cast<const double2*>(b_base + nt * 8 * SLD + k8 * 8);
#pragma unroll
                    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                        for (int nt = 0; nt < NTW; ++nt) dmma884(acc[mt][nt][0], acc[mt][nt][1], af[mt].x, bf[nt].x);
#pragma unroll
                    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                        for (int nt = 0; nt < NTW; ++nt) dmma884(acc[mt][nt][0], acc[mt][nt][1], af[mt].y, bf[nt].y);
                }
            }
        }
        if (warp_active) {
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const int gi = tm0 + wm * 32 + mt * 8 + g;
                if (gi >= a.m_hi) continue;
                double* crow = A + (size_t)gi * ld;
#pragma unroll
                for (int nt = 0; nt < NTW; ++nt) {
                    const int gj = tn0 + wn * (BN / 2) + nt * 8 + 2 * t;
                    if (gj + 1 < a.n_hi && gj + 1 <= gi) {
                        *reinterpret_cast<double2*>(crow + gj) = make_double2(-acc[mt][nt][0], -acc[mt][nt][1]);
                    } else if (gj < a.n_hi && gj <= gi) {
                        crow[gj] = -acc[mt][nt][0];
                    }
                }
            }
        }
    }
    cp_async_wait<0>();
}

// host side: rows [lo, m_hi) x columns [lo, n_hi) of every chain, inner range [k_lo, k_lo + K), K % 16 == 0
int launch_syrk(bd_ctx* ctx, double* A, int64_t ld, int64_t stride, int lo, int m_hi, int n_hi, int k_lo, int K)
{
    SyrkArgs a;
    a.A = A; a.ld = ld; a.stride = stride;
    a.lo = lo; a.m_hi = m_hi; a.n_hi = n_hi; a.k_lo = k_lo; a.K = K;
    const int TM = (m_hi - lo + BM - 1) / BM;
    a.TN = (n_hi - lo + BN - 1) / BN;
    constexpr int R = BM / BN;
    a.T2 = a.TN / R;                                     // tile rows that end at the diagonal: R (ty + 1) tiles each
    a.tri = R * a.T2 * (a.T2 + 1) / 2;
    a.per_chain = a.tri + (TM - a.T2) * a.TN;
    a.total = a.per_chain * ctx->C;
    const int slots = SYRK_CTAS * ctx->num_sms;
    const int grid = a.total < slots ? a.total : slots;
    BD_LAUNCH(ctx, k_syrk, dim3(grid), dim3(256), SYRK_SMEM, a);
    return 0;
}

}  // namespace

int bdk_potrf_launches(bd_ctx* ctx, double* A, int64_t ld, int64_t stride, int32_t* info)
{
    const int trsm_smem = TRSM_SMEM;
    if (!ctx->attr_potrf) {
        BD_CUDA(ctx, cudaFuncSetAttribute(k_syrk, cudaFuncAttributeMaxDynamicSharedMemorySize, SYRK_SMEM));
        BD_CUDA(ctx, cudaFuncSetAttribute(k_trsm, cudaFuncAttributeMaxDynamicSharedMemorySize, trsm_smem));
        BD_CUDA(ctx, cudaFuncSetAttribute(k_potf2, cudaFuncAttributeMaxDynamicSharedMemorySize, POTF2_SMEM));
        ctx->attr_potrf = true;
    }
    const int n = ctx->M, C = ctx->C;
    // outer panel width, from sweeps on B200 (profiles/r01_summary.md): with the recursive panel below, wide outer
    // panels win (c4: 256 -> 0.641, 1024 -> 0.688, 4096 -> 0.695 of peak; c5: 0.686 / 0.769 / 0.781)
    const int NB = (n >= 4096) ? 4096 : 1024;
    // Outer level: right-looking.  (A left-looking outer loop -- block column J updated by all finished columns in one
    // pass, K = J -- measured equal at c3 / c4 and slower at c5, profiles/r01_summary.md.)
    // In-panel factorisation of columns [J0, J1), all rows below included, RECURSIVELY: left half, update of the
    // right half with K = (J1 - J0) / 2, right half.  Against a plain right-looking sweep of 64-column blocks (every
    // block updated once per preceding block, always K = 64, DMMA pipe ~50 % busy) each column block now sees
    // log2((J1 - J0) / 64) updates with K = 64, 128, 256, ..
    struct Rec {
        bd_ctx* ctx; double* A; int64_t ld, stride; int32_t* info; int n, C, trsm_smem;
        int run(int J0, int J1)
        {
            if (J1 - J0 <= BD_NB_INNER) {
                const int nloc = J1 - J0;
                BD_LAUNCH(ctx, k_potf2, dim3(C), dim3(256), POTF2_SMEM, A, ld, stride, J0, nloc, info, ctx->Winv);
                if (J1 < n)
                    BD_LAUNCH(ctx, k_trsm, dim3((unsigned)((int64_t)((n - J1 + TRSM_ROWS - 1) / TRSM_ROWS) * C)), dim3(256), trsm_smem, A, ld,
                              stride, J0, J1, n, ctx->Winv);
                return 0;
            }
            const int half = ((J1 - J0) / 2 + BD_NB_INNER - 1) / BD_NB_INNER * BD_NB_INNER;
            const int mid = J0 + half;
            int rc = run(J0, mid);
            if (rc != 0) return rc;
            if ((rc = launch_syrk(ctx, A, ld, stride, mid, n, J1, J0, half)) != 0) return rc;
            return run(mid, J1);
        }
    } rec{ctx, A, ld, stride, info, n, C, trsm_smem};
    for (int J = 0; J < n; J += NB) {
        const int Jend = (J + NB < n) ? J + NB : n;
        int rc = rec.run(J, Jend);
        if (rc != 0) return rc;
        if (Jend < n) {
            rc = launch_syrk(ctx, A, ld, stride, Jend, n, n, J, Jend - J);
            if (rc != 0) return rc;
        }
    }
    return 0;
}
