// brownian.cu -- a0 (Brownian increments, Philox4x32-10 + Box-Muller) and a5 (y = L dW, the lower
// triangular matvec of Eq. 6's third term).  HBM-read bound: 4 M^2 bytes per chain.
#include "bd_internal.cuh"
#include "philox.cuh"

namespace {

// one thread per pair p: dW[2p], dW[2p+1]
__global__ void __launch_bounds__(256) k_noise(int M, int nblk, uint64_t seed, uint64_t chain0, uint64_t step, int kind,
                                               double dt, double* __restrict__ dW_all)
{
    const int c = blockIdx.x / nblk;                       // chain and block both on grid.x: no 65535-chain limit
    const int p = (blockIdx.x - c * nblk) * blockDim.x + threadIdx.x;
    if (2 * p >= M) return;
    double w0, w1;
    brownian_pair(seed, (uint32_t)p, chain0 + (uint64_t)c, step, kind, dt, w0, w1);
    double* dW = dW_all + (size_t)c * M;
    dW[2 * p] = w0;
    if (2 * p + 1 < M) dW[2 * p + 1] = w1;
}

// y_i = sum_{j<=i} L_ij dW_j.  One warp per row; lanes read 16-byte pairs, 4 independent loads in
// flight per lane; rows are dealt to warps so that long and short rows mix inside a CTA.
constexpr int kTrmvWarps = 8;

__global__ void __launch_bounds__(kTrmvWarps * 32) k_trmv(int M, const double* __restrict__ L_all, int64_t ld, int64_t stride,
                                                         const double* __restrict__ dW_all, double* __restrict__ y_all)
{
    const int nblk = (M + kTrmvWarps - 1) / kTrmvWarps;
    const int c = blockIdx.x / nblk, bx = blockIdx.x - c * nblk;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // pair short rows with long rows: CTA b takes rows b*4..b*4+3 from the top and the mirrored rows
    const int half = nblk * (kTrmvWarps / 2);
    int row;
    if (warp < kTrmvWarps / 2) row = bx * (kTrmvWarps / 2) + warp;
    else row = 2 * half - 1 - (bx * (kTrmvWarps / 2) + (warp - kTrmvWarps / 2));
    if (row >= M) return;
    const double* Lr = L_all + (size_t)c * stride + (size_t)row * ld;
    const double* dW = dW_all + (size_t)c * M;
    const int n = row + 1;                 // columns 0..row
    const int n2 = n & ~1;
    double acc0 = 0, acc1 = 0, acc2 = 0, acc3 = 0;
    int j = 2 * lane;
    for (; j + 192 < n2; j += 256) {
        const double2 l0 = *reinterpret_cast<const double2*>(Lr + j);
        const double2 l1 = *reinterpret_cast<const double2*>(Lr + j + 64);
        const double2 l2 = *reinterpret_cast<const double2*>(Lr + j + 128);
        const double2 l3 = *reinterpret_cast<const double2*>(Lr + j + 192);
        // dW rows are only 8-byte aligned (M is odd): scalar loads, L1-resident
        const double2 w0 = make_double2(dW[j], dW[j + 1]);
        const double2 w1 = make_double2(dW[j + 64], dW[j + 65]);
        const double2 w2 = make_double2(dW[j + 128], dW[j + 129]);
        const double2 w3 = make_double2(dW[j + 192], dW[j + 193]);
        acc0 += l0.x * w0.x + l0.y * w0.y;
        acc1 += l1.x * w1.x + l1.y * w1.y;
        acc2 += l2.x * w2.x + l2.y * w2.y;
        acc3 += l3.x * w3.x + l3.y * w3.y;
    }
    for (; j < n2; j += 64) {
        const double2 l0 = *reinterpret_cast<const double2*>(Lr + j);
        acc0 += l0.x * dW[j] + l0.y * dW[j + 1];
    }
    if (lane == 0 && (n & 1)) acc1 += Lr[n - 1] * dW[n - 1];
    const double s = warp_sum((acc0 + acc1) + (acc2 + acc3));
    if (lane == 0) y_all[(size_t)c * M + row] = s;
}

// Variant for M > TRMV_STAGED_MIN_M.  A CTA takes a block of 16 adjacent rows, two rows per warp; the blocks with the
// longest rows are scheduled first.  dW is staged through shared memory in chunks of TRMV_CHUNK columns, double
// buffered, and re-used by all rows of the CTA: at M = 30003 the vector (240 KB) no longer fits in L1 and the
// one-row-per-warp kernel fetched as many bytes of dW from L2 as of L from HBM.  Measured on B200 (GB/s at c3 / c4 / c5,
// HBM copy peak 6553): one row per warp 4945 / 5073 / 4265; this kernel with 4 rows per warp 4500 / 4540 / 4560, with
// 1 row per warp - / 5524 / 5995, with 2 rows per warp 5186 / 5454 / 6042 (fewer rows per CTA = a finer tail); pairing a
// long with a short block per CTA: 4037 at c5 (half the CTAs, half the bytes in flight).  Lanes read 16-byte pairs.
constexpr int TRMV_STAGED_MIN_M = 1024;           // below: one row per warp, dW through L1
constexpr int TRMV_WARPS = 8, TRMV_RPW = 2, TRMV_BLK = TRMV_WARPS * TRMV_RPW, TRMV_CHUNK = 2048;

__global__ void __launch_bounds__(TRMV_WARPS * 32) k_trmv_staged(int M, const double* __restrict__ L_all, int64_t ld, int64_t stride,
                                                         const double* __restrict__ dW_all, double* __restrict__ y_all)
{
    __shared__ __align__(16) double s_w[2][TRMV_CHUNK];
    const int nblk = (M + TRMV_BLK - 1) / TRMV_BLK;
    const int c = blockIdx.x / nblk;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int blk = nblk - 1 - (blockIdx.x - c * nblk);                         // longest rows are scheduled first
    const int row0 = blk * TRMV_BLK + warp * TRMV_RPW;
    const double* Lc = L_all + (size_t)c * stride;
    const double* dW = dW_all + (size_t)c * M;
    const int ncols_cta = min(M, (blk + 1) * TRMV_BLK);                         // longest row of the CTA + 1

    int n[TRMV_RPW];
    const double* Lr[TRMV_RPW];
    double acc[TRMV_RPW];
#pragma unroll
    for (int r = 0; r < TRMV_RPW; ++r) {
        const int row = row0 + r;
        n[r] = (row >= M) ? 0 : row + 1;
        Lr[r] = Lc + (size_t)min(row, M - 1) * ld;
        acc[r] = 0.0;
    }
    int nmax = 0;                                                              // rows grow with r; rows >= M have n = 0
#pragma unroll
    for (int r = 0; r < TRMV_RPW; ++r) nmax = max(nmax, n[r]);

    auto stage = [&](int ch, int buf) {
        const int j0 = ch * TRMV_CHUNK;
        for (int j = threadIdx.x; j < TRMV_CHUNK; j += TRMV_WARPS * 32) s_w[buf][j] = (j0 + j < M) ? dW[j0 + j] : 0.0;
    };
    const int nch = (ncols_cta + TRMV_CHUNK - 1) / TRMV_CHUNK;
    stage(0, 0);
    __syncthreads();
    for (int ch = 0; ch < nch; ++ch) {
        if (ch + 1 < nch) stage(ch + 1, (ch + 1) & 1);
        const int j0 = ch * TRMV_CHUNK;
        const int jend = min(nmax - j0, TRMV_CHUNK);                            // columns of this chunk this warp needs
        const double* w = s_w[ch & 1];
        for (int j = 2 * lane; j < jend; j += 128) {
            double2 l[2][TRMV_RPW];
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
                for (int r = 0; r < TRMV_RPW; ++r) {
                    const int col = j0 + j + 64 * u;
                    l[u][r] = (col < n[r]) ? *reinterpret_cast<const double2*>(Lr[r] + col) : make_double2(0.0, 0.0);
                }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int jj = j + 64 * u;
                const double2 wv = (jj < TRMV_CHUNK) ? *reinterpret_cast<const double2*>(w + jj) : make_double2(0.0, 0.0);
#pragma unroll
                for (int r = 0; r < TRMV_RPW; ++r) {
                    const int col = j0 + jj;
                    const double ly = (col + 1 < n[r]) ? l[u][r].y : 0.0;        // the pair may straddle the diagonal
                    acc[r] += l[u][r].x * wv.x + ly * wv.y;
                }
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < TRMV_RPW; ++r) {
        const double s = warp_sum(acc[r]);
        if (lane == 0 && n[r] > 0) y_all[(size_t)c * M + row0 + r] = s;
    }
}

}  // namespace

int bdk_noise(bd_ctx* ctx, uint64_t step, double* dW)
{
    const int pairs = (ctx->M + 1) / 2;
    const int nblk = (pairs + 255) / 256;
    BD_LAUNCH(ctx, k_noise, dim3((unsigned)((int64_t)nblk * ctx->C)), dim3(256), 0, ctx->M, nblk, ctx->p.seed, ctx->p.chain_id0, step,
              ctx->p.noise_kind, ctx->p.dt, dW);
    return 0;
}

int bdk_trmv(bd_ctx* ctx, const double* L, int64_t ld, int64_t stride, const double* dW, double* y)
{
    if (ctx->M > TRMV_STAGED_MIN_M) {
        const int nb = (ctx->M + TRMV_BLK - 1) / TRMV_BLK;
        BD_LAUNCH(ctx, k_trmv_staged, dim3((unsigned)((int64_t)nb * ctx->C)), dim3(TRMV_WARPS * 32), 0, ctx->M, L, ld, stride, dW, y);
        return 0;
    }
    const int nblk = (ctx->M + kTrmvWarps - 1) / kTrmvWarps;
    BD_LAUNCH(ctx, k_trmv, dim3((unsigned)((int64_t)nblk * ctx->C)), dim3(kTrmvWarps * 32), 0, ctx->M, L, ld, stride, dW, y);
    return 0;
}
