// potrf.cu -- a3: in-place FP64 Cholesky D = L L^T of the lower triangle (Eq. 10),
// batched over chains.  The paper calls cusolverDnDpotrf once per chain per step (:172); this is a
// hand-written blocked right-looking factorisation for sm_100a:
//
//   two-level blocking: outer panels of NB columns, inner diagonal blocks of 64 columns
//     k_potf2   64x64 diagonal block, register-resident, one CTA per chain
//     k_trsm    rows below the diagonal block:  X L_jj^T = A   (one thread per row, L_jj broadcast from smem)
//     k_syrk    C -= P P^T with FP64 tensor-core DMMA (mma.sync m8n8k4), 128x128 tiles, 4-stage cp.async
//               pipeline; used both for the in-panel update (K = 64) and the trailing update (K = NB),
//               so the trailing matrix is read and written once per NB columns, not once per 64.
//
// FP64 has no tcgen05 kind; the FP64 tensor path on sm_100a is warp-level DMMA (measured 37.07
// TFLOP/s on B200), so operands go global -> cp.async -> padded smem -> registers.
// Matrices are ROW-major, lower triangle: L[i][j], j <= i, so both SYRK operands are K-contiguous
// rows of the same panel ("NT" form) and the DMMA A and B fragments use the same access pattern.
#include "bd_internal.cuh"

namespace {

// =================================================================================================
// k_potf2: unblocked Cholesky of one nb x nb (nb <= 64) diagonal block per chain.  256 threads as a
// 16 x 16 grid, thread (ty,tx) keeps the 4x4 sub-block rows 4ty.., cols 4tx.. in registers.  Step k
// broadcasts column k through shared memory (double buffered: one barrier per step) and applies
// the rank-1 update A[i][j] -= A[i][k] A[j][k] / d_k; columns are scaled by 1/sqrt(d_k) at the end.
// A non-positive (or NaN) pivot d_k records info = 1-based global row (first failure wins).
// =================================================================================================
__global__ void __launch_bounds__(256) k_potf2(double* __restrict__ A_all, int64_t ld, int64_t stride, int j0, int nloc,
                                               int32_t* __restrict__ info)
{
    __shared__ double s_col[2][64];
    __shared__ double s_d[64];
    const int c = blockIdx.x;
    double* A = A_all + (size_t)c * stride + (size_t)j0 * ld + j0;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    const bool active = ty >= tx;
    double a[4][4];
#pragma unroll
    for (int rr = 0; rr < 4; ++rr)
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
            const int i = 4 * ty + rr, j = 4 * tx + cc;
            double val = (i == j) ? 1.0 : 0.0;                    // identity padding for a ragged block
            if (active && i < nloc && j <= i) val = A[(size_t)i * ld + j];
            a[rr][cc] = val;
        }
    int fail_row = 0;
    for (int k = 0; k < nloc; ++k) {
        const int buf = k & 1;
        if (tx == (k >> 2) && active) {
            const int kc = k & 3;
#pragma unroll
            for (int rr = 0; rr < 4; ++rr) {
                double val = a[rr][0];
                if (kc == 1) val = a[rr][1];
                if (kc == 2) val = a[rr][2];
                if (kc == 3) val = a[rr][3];
                s_col[buf][4 * ty + rr] = val;
            }
        }
        __syncthreads();
        const double d = s_col[buf][k];
        if (!(d > 0.0) && fail_row == 0) fail_row = j0 + k + 1;
        if (threadIdx.x == 0) s_d[k] = d;
        if (active && 4 * ty + 3 > k) {
            const double invd = 1.0 / d;
            double li[4], lj[4];
#pragma unroll
            for (int rr = 0; rr < 4; ++rr) li[rr] = s_col[buf][4 * ty + rr] * invd;
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) lj[cc] = s_col[buf][4 * tx + cc];
#pragma unroll
            for (int rr = 0; rr < 4; ++rr)
#pragma unroll
                for (int cc = 0; cc < 4; ++cc)
                    if (4 * tx + cc > k) a[rr][cc] -= li[rr] * lj[cc];
        }
    }
    __syncthreads();
    if (threadIdx.x == 0 && fail_row != 0 && info != nullptr && info[c] == 0) info[c] = fail_row;
    if (active) {
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
            const int j = 4 * tx + cc;
            if (j >= nloc) continue;
            const double piv = sqrt(s_d[j]);
            const double inv = 1.0 / piv;
#pragma unroll
            for (int rr = 0; rr < 4; ++rr) {
                const int i = 4 * ty + rr;
                if (i < nloc && j <= i) A[(size_t)i * ld + j] = (i == j) ? piv : a[rr][cc] * inv;
            }
        }
    }
}

// =================================================================================================
// k_trsm: rows gi in [r_lo, r_hi) of the panel at columns [j0, j0+64): solve X L^T = A in place with
// the freshly factored 64x64 block L = A[j0.., j0..].  One thread per row (64 doubles in registers),
// right-looking over the columns so that every FMA of a step is independent; L^T is broadcast from
// shared memory with 16-byte loads.  Rows are staged through shared memory for coalesced global access.
// =================================================================================================
constexpr int TRSM_ROWS = 128;
constexpr int TRSM_SLD = 65;          // odd stride: conflict-free row reads

__global__ void __launch_bounds__(TRSM_ROWS) k_trsm(double* __restrict__ A_all, int64_t ld, int64_t stride, int j0,
                                                    int r_lo, int r_hi)
{
    extern __shared__ __align__(16) double smem[];
    double* s_Lt = smem;                         // [64][64]  s_Lt[c][cp] = L[cp][c]  (column c of L, contiguous in cp)
    double* s_inv = s_Lt + 64 * 64;              // [64]      1 / L[c][c]
    double* s_X = s_inv + 64;                    // [TRSM_ROWS][TRSM_SLD]
    const int c = blockIdx.y;
    double* A = A_all + (size_t)c * stride;
    const int row0 = r_lo + blockIdx.x * TRSM_ROWS;
    const int tid = threadIdx.x;
    // L block (lower) -> transposed smem
    for (int q = tid; q < 64 * 64; q += TRSM_ROWS) {
        const int i = q >> 6, j = q & 63;
        const double val = (j <= i) ? A[(size_t)(j0 + i) * ld + j0 + j] : 0.0;
        s_Lt[j * 64 + i] = val;
        if (i == j) s_inv[i] = 1.0 / val;
    }
    // panel rows -> smem (coalesced: 64 consecutive doubles per row)
    for (int q = tid; q < TRSM_ROWS * 64; q += TRSM_ROWS) {
        const int rr = q >> 6, cc = q & 63;
        const int gi = row0 + rr;
        s_X[rr * TRSM_SLD + cc] = (gi < r_hi) ? A[(size_t)gi * ld + j0 + cc] : 0.0;
    }
    __syncthreads();
    double x[64];
#pragma unroll
    for (int cc = 0; cc < 64; ++cc) x[cc] = s_X[tid * TRSM_SLD + cc];
#pragma unroll
    for (int cc = 0; cc < 64; ++cc) {
        const double xc = x[cc] * s_inv[cc];
        x[cc] = xc;
        const double* lt = s_Lt + cc * 64;
#pragma unroll
        for (int cp = cc + 1; cp < 64; ++cp) x[cp] -= xc * lt[cp];
    }
#pragma unroll
    for (int cc = 0; cc < 64; ++cc) s_X[tid * TRSM_SLD + cc] = x[cc];
    __syncthreads();
    for (int q = tid; q < TRSM_ROWS * 64; q += TRSM_ROWS) {
        const int rr = q >> 6, cc = q & 63;
        const int gi = row0 + rr;
        if (gi < r_hi) A[(size_t)gi * ld + j0 + cc] = s_X[rr * TRSM_SLD + cc];
    }
}

// =================================================================================================
// k_syrk: for gi in [m_lo, m_hi), gj in [n_lo, n_hi), gj <= gi:
//     A[gi][gj] -= sum_{p in [k_lo, k_lo+K)} A[gi][p] * A[gj][p]
// 128 x 128 tile per CTA, 8 warps (4 along m x 2 along n), warp tile 32 x 64 = 4 x 8 DMMA m8n8k4
// accumulators (64 FP64 accumulators per thread).  Operands stream through a 4-stage cp.async
// pipeline of 128 x 16 slabs; smem rows are padded to 20 doubles so the 8-byte fragment loads of a
// warp fall in distinct bank pairs.
// =================================================================================================
constexpr int BM = 128, BN = 128, BK = 16, STAGES = 4, SLD = 20;
constexpr int SYRK_SMEM = STAGES * (BM + BN) * SLD * (int)sizeof(double);

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, int src_bytes)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256, 1) k_syrk(double* __restrict__ A_all, int64_t ld, int64_t stride, int m_lo, int m_hi,
                                                 int n_lo, int n_hi, int k_lo, int K)
{
    const int tm0 = m_lo + blockIdx.y * BM, tn0 = n_lo + blockIdx.x * BN;
    if (tn0 > tm0 + BM - 1) return;                      // tile entirely above the diagonal
    extern __shared__ __align__(16) double smem[];
    double* sA = smem;                                   // [STAGES][BM][SLD]
    double* sB = smem + STAGES * BM * SLD;               // [STAGES][BN][SLD]
    double* A = A_all + (size_t)blockIdx.z * stride;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp & 3, wn = warp >> 2;
    const int g = lane >> 2, t = lane & 3;
    const int KT = K / BK;

    auto load_stage = [&](int slot, int kt) {
        const double* src_k = A + k_lo + kt * BK;
#pragma unroll
        for (int it = 0; it < (BM * BK / 2) / 256; ++it) {
            const int chunk = tid + it * 256;
            const int row = chunk >> 3, ch = chunk & 7;
            const int gr = tm0 + row;
            const bool ok = gr < m_hi;
            cp_async16(sA + ((size_t)slot * BM + row) * SLD + 2 * ch, src_k + (size_t)(ok ? gr : m_hi - 1) * ld + 2 * ch, ok ? 16 : 0);
        }
#pragma unroll
        for (int it = 0; it < (BN * BK / 2) / 256; ++it) {
            const int chunk = tid + it * 256;
            const int row = chunk >> 3, ch = chunk & 7;
            const int gr = tn0 + row;
            const bool ok = gr < n_hi;
            cp_async16(sB + ((size_t)slot * BN + row) * SLD + 2 * ch, src_k + (size_t)(ok ? gr : n_hi - 1) * ld + 2 * ch, ok ? 16 : 0);
        }
    };

    double acc[4][8][2];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    // this warp's 32 x 64 block lies entirely above the diagonal -> no arithmetic (still loads/syncs)
    const bool warp_active = (tn0 + wn * 64) <= (tm0 + wm * 32 + 31);

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < KT) load_stage(s, s);
        cp_async_commit();
    }
    for (int kt = 0; kt < KT; ++kt) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        if (kt + STAGES - 1 < KT) load_stage((kt + STAGES - 1) % STAGES, kt + STAGES - 1);
        cp_async_commit();
        if (warp_active) {
            const double* a_base = sA + ((size_t)(kt % STAGES) * BM + wm * 32 + g) * SLD + t;
            const double* b_base = sB + ((size_t)(kt % STAGES) * BN + wn * 64 + g) * SLD + t;
#pragma unroll
            for (int ks = 0; ks < BK / 4; ++ks) {
                double af[4], bf[8];
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) af[mt] = a_base[mt * 8 * SLD + ks * 4];
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) bf[nt] = b_base[nt * 8 * SLD + ks * 4];
#pragma unroll
                for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                    for (int nt = 0; nt < 8; ++nt) dmma884(acc[mt][nt][0], acc[mt][nt][1], af[mt], bf[nt]);
            }
        }
    }
    cp_async_wait<0>();
    if (!warp_active) return;
    // epilogue: C -= acc on the lower triangle
#pragma unroll
    for (int mt = 0; mt < 4; ++mt) {
        const int gi = tm0 + wm * 32 + mt * 8 + g;
        if (gi >= m_hi) continue;
        double* crow = A + (size_t)gi * ld;
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
            const int gj = tn0 + wn * 64 + nt * 8 + 2 * t;
            if (gj + 1 < n_hi && gj + 1 <= gi) {
                double2 cv = *reinterpret_cast<double2*>(crow + gj);
                cv.x -= acc[mt][nt][0];
                cv.y -= acc[mt][nt][1];
                *reinterpret_cast<double2*>(crow + gj) = cv;
            } else if (gj < n_hi && gj <= gi) {
                crow[gj] -= acc[mt][nt][0];
            }
        }
    }
}

}  // namespace

int bdk_potrf(bd_ctx* ctx, double* A, int64_t ld, int64_t stride, int32_t* info)
{
    static bool attr_set = false;
    const int trsm_smem = (64 * 64 + 64 + TRSM_ROWS * TRSM_SLD) * (int)sizeof(double);
    if (!attr_set) {
        BD_CUDA(ctx, cudaFuncSetAttribute(k_syrk, cudaFuncAttributeMaxDynamicSharedMemorySize, SYRK_SMEM));
        BD_CUDA(ctx, cudaFuncSetAttribute(k_trsm, cudaFuncAttributeMaxDynamicSharedMemorySize, trsm_smem));
        attr_set = true;
    }
    const int n = ctx->M, C = ctx->C;
    const int NB = (n >= 8192) ? 512 : 256;
    for (int J = 0; J < n; J += NB) {
        const int Jend = (J + NB < n) ? J + NB : n;
        for (int j = J; j < Jend; j += BD_NB_INNER) {
            const int nloc = (n - j < BD_NB_INNER) ? n - j : BD_NB_INNER;
            BD_LAUNCH(ctx, k_potf2, dim3(C), dim3(256), 0, A, ld, stride, j, nloc, info);
            const int r_lo = j + BD_NB_INNER;
            if (r_lo < n) {
                BD_LAUNCH(ctx, k_trsm, dim3((n - r_lo + TRSM_ROWS - 1) / TRSM_ROWS, C), dim3(TRSM_ROWS), trsm_smem, A, ld, stride, j,
                          r_lo, n);
                if (r_lo < Jend) {
                    dim3 grid((Jend - r_lo + BN - 1) / BN, (n - r_lo + BM - 1) / BM, C);
                    BD_LAUNCH(ctx, k_syrk, grid, dim3(256), SYRK_SMEM, A, ld, stride, r_lo, n, r_lo, Jend, j, BD_NB_INNER);
                }
            }
        }
        if (Jend < n) {
            dim3 grid((n - Jend + BN - 1) / BN, (n - Jend + BM - 1) / BM, C);
            BD_LAUNCH(ctx, k_syrk, grid, dim3(256), SYRK_SMEM, A, ld, stride, Jend, n, Jend, n, J, Jend - J);
        }
    }
    return 0;
}
