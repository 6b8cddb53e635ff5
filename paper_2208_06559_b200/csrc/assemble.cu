// assemble.cu -- a2: pairwise RPY hydrodynamic-interaction tensor (Eqs. 7-9) written
// as 3x3 blocks at rows 3i.., cols 3j.. (Eqs. 18-19, :214-223).
//
// The paper's kernel (Alg. 1, :383-407) launches one thread per SCALAR element and so evaluates the
// pair geometry nine times.  Here one thread evaluates one bead PAIR (one rsqrt, no division), the
// CTA stages its 24 x 96 tile of D in shared memory, and the tile is written out row by row with
// 16-byte stores: every row segment is 768 contiguous, 128-byte aligned bytes.  HBM-write bound:
// 4 M^2 + 4 M bytes per chain for the lower triangle.
#include "bd_internal.cuh"

namespace {

constexpr int TI = 8;                 // beads per tile, row direction  (24 rows)
constexpr int TJ = 32;                // beads per tile, column direction (96 columns)
constexpr int TROWS = 3 * TI;
constexpr int TCOLS = 3 * TJ;
constexpr int TLD = TCOLS + 2;        // padded smem row (keeps 16-byte alignment of pairs)

__global__ void __launch_bounds__(TI * TJ) k_assemble(int Nb, double hstar, double a_s, double inv_a, double inv_b,
                                                      const double* __restrict__ r_all, double* __restrict__ D_all,
                                                      int64_t ld, int64_t stride, int full)
{
    const int i0 = blockIdx.y * TI, j0 = blockIdx.x * TJ;
    if (j0 > i0 + TI - 1) return;                       // tile entirely above the diagonal
    __shared__ __align__(16) double s_tile[TROWS][TLD];
    const int c = blockIdx.z;                           // the host launches at most 65535 chains at a time
    const int M = 3 * Nb;
    const double* r = r_all + (size_t)c * M;
    double* D = D_all + (size_t)c * stride;
    const int tj = threadIdx.x & (TJ - 1), ti = threadIdx.x / TJ;
    const int i = i0 + ti, j = j0 + tj;

    double B[3][3];
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int l = 0; l < 3; ++l) B[k][l] = (k == l && i == j) ? 1.0 : 0.0;     // Eq. 7
    if (i < Nb && j < i) {
        const double dx = (r[3 * i] - r[3 * j]) * inv_b, dy = (r[3 * i + 1] - r[3 * j + 1]) * inv_b,
                     dz = (r[3 * i + 2] - r[3 * j + 2]) * inv_b;
        double cI, cRR;
        rpy_coeffs(dx * dx + dy * dy + dz * dz, hstar, a_s, inv_a, cI, cRR);              // Eqs. 8-9
        const double d[3] = {dx, dy, dz};
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
            for (int l = 0; l < 3; ++l) B[k][l] = cRR * d[k] * d[l] + ((k == l) ? cI : 0.0);
        if (full) {                                                                 // mirrored block (j,i)
#pragma unroll
            for (int l = 0; l < 3; ++l)
#pragma unroll
                for (int k = 0; k < 3; ++k) D[(size_t)(3 * j + l) * ld + 3 * i + k] = B[k][l];
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int l = 0; l < 3; ++l) s_tile[3 * ti + k][3 * tj + l] = B[k][l];
    __syncthreads();

    // write-out: TROWS rows x (TCOLS/2) 16-byte chunks; column limit = the diagonal (lower triangle),
    // or the end of the diagonal block row in full mode.
    for (int q = threadIdx.x; q < TROWS * (TCOLS / 2); q += TI * TJ) {
        const int rr = q / (TCOLS / 2), cc = q - rr * (TCOLS / 2);
        const int gr = 3 * i0 + rr, gc = 3 * j0 + 2 * cc;
        if (gr >= M) continue;
        const int lim = full ? min(M - 1, 3 * (gr / 3) + 2) : gr;     // last writable column of this row
        double* dst = D + (size_t)gr * ld + gc;
        const double2 val = *reinterpret_cast<const double2*>(&s_tile[rr][2 * cc]);
        if (gc + 1 <= lim) *reinterpret_cast<double2*>(dst) = val;
        else if (gc <= lim) dst[0] = val.x;
    }
}

}  // namespace

int bdk_assemble(bd_ctx* ctx, const double* r, double* D, int64_t ld, int64_t stride, int full)
{
    // grid.z carries the chain and is limited to 65535: larger ensembles go in slices (a block index decoded with
    // integer divisions instead cost 10 % of this short, store-bound kernel)
    for (int c0 = 0; c0 < ctx->C; c0 += 65535) {
        const int nc = (ctx->C - c0 < 65535) ? ctx->C - c0 : 65535;
        dim3 grid((ctx->Nb + TJ - 1) / TJ, (ctx->Nb + TI - 1) / TI, nc);
        BD_LAUNCH(ctx, k_assemble, grid, dim3(TI * TJ), 0, ctx->Nb, ctx->p.hstar, ctx->p.a / ctx->p.b, ctx->p.b / ctx->p.a, 1.0 / ctx->p.b,
                  r + (size_t)c0 * ctx->M, D + (size_t)c0 * stride, ld, stride, full);
    }
    return 0;
}
