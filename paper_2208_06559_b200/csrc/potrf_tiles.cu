// potrf_tiles.cu -- a3: in-place FP64 Cholesky D = L L^T of the lower triangle (Eq. 10), batched over
// chains, as ONE persistent kernel per factorisation: a LEFT-LOOKING TILE Cholesky driven by a ticket counter and
// per-tile ready flags (the paper calls cusolverDnDpotrf once per chain and step, :172).
//
//   The matrix is cut into 128 x 128 tiles (i, j), i >= j.  Tile (i, j) is owned by one CTA from start to finish:
//     acc = -D_ij + sum_{k < 128 j} L[i-rows][k] L[j-rows][k]       K-deep FP64 tensor-core (DMMA m8n8k4) loop, the
//                                                                    C tile never leaves the accumulators
//     i > j:  S = -acc;  L_ij = S W_j^T  with W_j = L_jj^-1          a second, 128-deep pass through the same pipeline
//     i = j:  L_jj = chol(S), W_j = L_jj^-1                          in shared memory (potf2_blocked.cuh, 64 + 64)
//   Tickets are handed out column by column (j outer, then chain, then i, the next diagonal tile early); a tile waits (ld.acquire on the ready flag
//   of the tiles it reads) only for tiles with SMALLER tickets, which running CTAs own, so the schedule cannot
//   deadlock and needs no co-residency.  Later columns start while the diagonal block of the current one is still being
//   factored: the lookahead that the multi-launch version (potrf.cu) does not have, and one launch instead of
//   ~6 M / 64 of them.
//
//   Operands come through TMA: a 3-D tensor map over the row-major storage (column, row, chain), boxes of 128 rows x 16
//   columns (= 128 B rows, SWIZZLE_128B), two boxes per operand and stage, 3-stage ring of 64 KB stages with full /
//   empty mbarriers; one producer thread (warp 8; its warpgroup gives its registers away with setmaxnreg) issues the copies, 8 consumer warps (4 x 2, warp tile 32 x 64) never
//   meet at a CTA barrier inside the K loop.  Rows beyond M are zero-filled by the TMA unit (ragged last tile).
//   SYRK/GEMM symmetry: A and B fragments index the k dimension identically, so a lane may read ANY k of the slab as
//   long as both operands use the same map: lane (g, t) reads 16-byte chunk (2 t + j) ^ g of row g (j = 0, 1), which
//   is conflict free under the 128-byte swizzle (the 8 lanes of a quarter-warp hit 8 distinct chunks).
#include <mutex>
#include <type_traits>

#include <cuda.h>          // CUtensorMap and its enums only; cuTensorMapEncodeTiled is fetched through the runtime (no -lcuda)

#include "bd_internal.cuh"
#include "potf2_blocked.cuh"
#include "tma.cuh"

namespace {

constexpr int TB = 128;                       // tile size
constexpr int BOXK = 16;                      // columns per TMA box (128 bytes = the swizzle span)
constexpr int BK = 32;                        // columns per ring stage (two boxes per operand)
constexpr int SPB = TB / BK;                  // stages per 128-column block
constexpr int STAGES = 3;
constexpr int QD = 2;                         // depth of the ticket queue between the producer and the consumers
constexpr int BOX_BYTES = TB * BOXK * 8;      // 16 KB
constexpr int STAGE_BYTES = 4 * BOX_BYTES;    // A box 0, A box 1, B box 0, B box 1
constexpr int NCONS = 256;                    // consumer threads (8 warps)
constexpr int NTHREADS = NCONS + 128;         // + the producer warpgroup (one lane of it works; setmaxnreg is per warpgroup)
constexpr int REGS_PRODUCER = 40, REGS_CONSUMER = 232;   // 8 x 32 x 232 + 4 x 32 x 40 = 64512 <= 65536 registers
constexpr int RING_BYTES = STAGES * STAGE_BYTES;
constexpr int TILE_SMEM = RING_BYTES + 1024;  // + slack to align the ring to 1024 B (SWIZZLE_128B atom)
constexpr long long SPIN_LIMIT = 8000000000LL;   // ~4 s of SM clocks: a lost dependency flags an error instead of hanging

struct TileArgs {
    double* A;
    int64_t ld, stride;
    int M, C, T, nsm;        // nsm = CTAs of the launch (one wave of tickets)
    double* Wbuf;            // [C][T][128][128] inverse diagonal blocks
    int* flags;              // [C][T][T]: == epoch when tile (i, j) of chain c is final
    int epoch;
    unsigned* ticket;
    unsigned ticket_base, total;
    int32_t* info;           // [C]
    int* err;                // set when a dependency wait timed out
};

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}
__device__ __forceinline__ void cons_sync() { asm volatile("bar.sync 9, 256;\n" ::: "memory"); }   // the 8 consumer warps

__device__ __forceinline__ void wait_flag(const int* f, int epoch, int* err)
{
    if (ld_acquire_gpu(f) == epoch) return;
    const long long t0 = clock64();
    while (ld_acquire_gpu(f) != epoch) {
        __nanosleep(100);
        if (clock64() - t0 > SPIN_LIMIT) { atomicExch(err, 1); return; }
        if (*reinterpret_cast<volatile int*>(err) != 0) return;
    }
}

// ticket -> (row i, column j, chain c).  Order: first the diagonal tile (0, 0) of every chain; then, for j = 0 .. T-2
// ("phase j"), the tiles of column j chain by chain, with the NEXT diagonal tile (j+1, j+1) slipped in early: it only
// needs row j+1 up to column j, so it is factored while the rest of column j is still being computed, and when the
// tiles of column j+1 come up L_{j+1,j+1} and its inverse have long been published.
//   one chain, or few:   (j+1, j), (j+1, j+1), (j+2, j), .., (T-1, j)                          per chain
//   many chains:         the diagonal tile of chain c follows the column tiles of chain c + delta, delta chosen so that
//                        about one wave of tickets (the grid size) lies between tile (j+1, j) and the diagonal tile that
//                        reads it (otherwise the CTA that draws the diagonal tile waits ~20 us for its neighbour's
//                        epilogue: 3 % of the c3 step); the last delta diagonal tiles close the phase.
// Every tile depends on tiles with smaller tickets only.
__device__ __forceinline__ void decode_ticket(unsigned tk, int C, int T, int nsm, int& j, int& c, int& i)
{
    if (tk < (unsigned)C) { i = 0; j = 0; c = (int)tk; return; }
    const unsigned u = tk - (unsigned)C;
    const long long q = (long long)(u / (unsigned)C);          // entries of one chain in the phases before: j T - j (j-1) / 2 <= q
    const double b = 2.0 * T + 1.0;
    int jj = (int)((b - sqrt(fmax(b * b - 8.0 * (double)q, 0.0))) * 0.5);
    jj = max(0, min(jj, T - 2));
    auto before = [&](int x) { return (long long)x * T - (long long)x * (x - 1) / 2; };
    while (jj + 1 <= T - 2 && before(jj + 1) * C <= (long long)u) ++jj;
    while (jj > 0 && before(jj) * C > (long long)u) --jj;
    const long long rem = (long long)u - before(jj) * C;
    const int w = T - jj;                                       // entries per chain in phase jj: w - 1 column tiles + 1 diagonal tile
    const int delta = min(C / 2, (nsm + 12 + w - 1) / w);
    j = jj;
    if (delta == 0) {
        c = (int)(rem / w);
        const int idx = (int)(rem - (long long)c * w);
        if (idx == 1) { i = jj + 1; j = jj + 1; }
        else i = jj + (idx == 0 ? 1 : idx);
        return;
    }
    const int cw = w - 1;
    if (rem < (long long)delta * cw) {                          // the first delta chains: column tiles only
        c = (int)(rem / cw);
        i = jj + 1 + (int)(rem - (long long)c * cw);
        return;
    }
    const long long r2 = rem - (long long)delta * cw;
    if (r2 < (long long)(C - delta) * w) {                      // column tiles of chain delta + g, then the diagonal tile of chain g
        const int gq = (int)(r2 / w), idx = (int)(r2 - (long long)gq * w);
        if (idx < cw) { c = delta + gq; i = jj + 1 + idx; }
        else { c = gq; i = jj + 1; j = jj + 1; }
        return;
    }
    c = C - delta + (int)(r2 - (long long)(C - delta) * w);     // the remaining diagonal tiles
    i = jj + 1;
    j = jj + 1;
}

// One 128 x 16 box of both operands: 2 chunk pairs x (4 + (8 - NTLO) LDS.128, 2 x 4 x (8 - NTLO) DMMA) per warp.  NTLO > 0 skips
// the first n-tiles (the S W^T pass: W is lower triangular, column block nt of the warp needs p <= its last column only).
// NTHI >= 0 instead keeps, for the m-tile mt, only the n-tiles nt <= NTHI + mt (a 32 x 64 block that the diagonal of a
// diagonal tile crosses: everything right of it is never used).
template <int NTLO, int NTHI = 8>
__device__ __forceinline__ void compute_box(double (&acc)[4][8][2], const uint8_t* __restrict__ sa, const uint8_t* __restrict__ sb,
                                            const int xo0, const int xo1)
{
    constexpr int NTE = (NTHI + 3 < 7) ? NTHI + 4 : 8;         // n-tiles any m-tile needs
#pragma unroll
    for (int jj = 0; jj < 2; ++jj) {
        const int xo = jj ? xo1 : xo0;
        double2 af[4], bf[8];
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) af[mt] = *reinterpret_cast<const double2*>(sa + mt * 1024 + xo);
#pragma unroll
        for (int nt = NTLO; nt < NTE; ++nt) bf[nt] = *reinterpret_cast<const double2*>(sb + nt * 1024 + xo);
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
#pragma unroll
            for (int nt = NTLO; nt < NTE; ++nt)
                if (nt <= NTHI + mt) dmma884(acc[mt][nt][0], acc[mt][nt][1], af[mt].x, bf[nt].x);
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
#pragma unroll
            for (int nt = NTLO; nt < NTE; ++nt)
                if (nt <= NTHI + mt) dmma884(acc[mt][nt][0], acc[mt][nt][1], af[mt].y, bf[nt].y);
    }
}

// box B8 (16 columns p = 16 B8 ..) of the S W^T pass for the warp column half wn: X[., cc] needs p <= cc
template <int B8>
__device__ __forceinline__ void trsm_box(double (&acc)[4][8][2], const int wn, const uint8_t* sa, const uint8_t* sb, const int xo0,
                                         const int xo1)
{
    if (wn == 0) {
        if constexpr (B8 < 4) compute_box<2 * B8>(acc, sa, sb, xo0, xo1);        // columns 0..63: p < 64 only
    } else {
        if constexpr (B8 < 4) compute_box<0>(acc, sa, sb, xo0, xo1);
        else compute_box<2 * (B8 - 4)>(acc, sa, sb, xo0, xo1);
    }
}

// LATENCY = true: the instance for factorisations with few tiles per column (one chain of moderate size), where the
// diagonal tiles are the critical path: its factoring warp defers the rank-1 update (warp_chol_deferred).
template <bool LATENCY>
__global__ void __launch_bounds__(NTHREADS, 1) k_potrf_tiles(const __grid_constant__ CUtensorMap tmA,
                                                             const __grid_constant__ CUtensorMap tmW, const TileArgs a)
{
    extern __shared__ uint8_t smem_raw[];
    // full[0..S), empty[S..2S), S-stored, diagonal-tile-done, ticket queue full[QD], ticket queue empty[QD]
    __shared__ __align__(8) uint64_t sBar[2 * STAGES + 2 + 2 * QD];
    __shared__ unsigned sQ[QD];
    __shared__ int sFail;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const uint32_t ring = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* ring_g = smem_raw + (ring - smem_u32(smem_raw));
    const uint32_t bar_full = smem_u32(&sBar[0]), bar_empty = smem_u32(&sBar[STAGES]), bar_s = smem_u32(&sBar[2 * STAGES]),
                   bar_d = smem_u32(&sBar[2 * STAGES + 1]), bar_qf = smem_u32(&sBar[2 * STAGES + 2]),
                   bar_qe = smem_u32(&sBar[2 * STAGES + 2 + QD]);

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, NCONS / 32); }
        mbar_init(bar_s, NCONS);
        mbar_init(bar_d, NCONS / 32);
        for (int s = 0; s < QD; ++s) { mbar_init(bar_qf + 8 * s, 1); mbar_init(bar_qe + 8 * s, NCONS / 32); }
        mbar_fence_init();
    }
    __syncthreads();

    const int M = a.M, T = a.T;
    const int64_t ld = a.ld;

    // Register budget: 384 threads cap the kernel at 168 registers per thread (each of the 4 sub-partitions holds 3
    // warps); the producer warpgroup hands its share to the 8 consumer warps (64 accumulators + fragments) with
    // setmaxnreg.  The two roles run SEPARATE tile loops from here to the end of the kernel (ptxas allocates registers per
    // region) and talk through mbarriers only: the producer draws the tickets, publishes them in a 2-deep queue and runs
    // AHEAD of the consumers (the next tile's first stages are in flight while the current tile is still in its epilogue);
    // it only stops behind a diagonal tile, whose factorisation uses the ring as scratch.
    if (warp >= NCONS / 32) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(REGS_PRODUCER));
        if (warp != NCONS / 32 || lane != 0) return;
        // ================================== producer: one thread feeds the ring ==================================
        uint32_t git = 0, sphase = 0, dphase = 0;      // ring stages issued, uses of the S-stored / diagonal-done barriers
        for (uint32_t n = 0;; ++n) {
            const unsigned tk = atomicAdd(a.ticket, 1u) - a.ticket_base;
            const uint32_t qs = n % QD;
            if (n >= QD) mbar_wait(bar_qe + 8 * qs, ((n / QD) - 1) & 1);
            sQ[qs] = tk;
            mbar_arrive(bar_qf + 8 * qs);              // release: the consumers read sQ after their wait
            if (tk >= a.total) break;
            int i, j, c;
            decode_ticket(tk, a.C, T, a.nsm, j, c, i);
            const bool diag = (i == j);
            const int KT = j * SPB;                    // ring stages of the K loop
            int* flags_c = a.flags + (size_t)c * T * T;
            const int tm0 = i * TB, tn0 = j * TB;
            auto acquire_slot = [&](uint32_t G) {
                const uint32_t sl = G % STAGES;
                if (G >= STAGES) mbar_wait(bar_empty + 8 * sl, ((G / STAGES) - 1) & 1);
                return sl;
            };
            int ready = 0;                             // 128-column blocks known to be final in rows i and j
            if (j > 0 && ld_acquire_gpu(flags_c + (size_t)i * T + j - 1) == a.epoch &&
                ld_acquire_gpu(flags_c + (size_t)j * T + j - 1) == a.epoch) {
                ready = j;                             // tile (., j-1) final => every (., k < j-1) it read is final too
                fence_proxy_async();
            }
            for (int kb = 0; kb < j; ++kb) {
                if (kb >= ready) {
                    wait_flag(flags_c + (size_t)i * T + kb, a.epoch, a.err);
                    if (!diag) wait_flag(flags_c + (size_t)j * T + kb, a.epoch, a.err);
                    fence_proxy_async();               // the acquired tiles are read through the async proxy (TMA)
                }
                for (int s4 = 0; s4 < SPB; ++s4) {
                    const uint32_t G = git + kb * SPB + s4, sl = acquire_slot(G);
                    const uint32_t dst = ring + sl * STAGE_BYTES, fb = bar_full + 8 * sl;
                    const int k0 = kb * TB + s4 * BK;
                    mbar_expect_tx(fb, diag ? 2 * BOX_BYTES : 4 * BOX_BYTES);
                    tma_tile_3d(dst, &tmA, k0, tm0, c, fb);
                    tma_tile_3d(dst + BOX_BYTES, &tmA, k0 + BOXK, tm0, c, fb);
                    if (!diag) {
                        tma_tile_3d(dst + 2 * BOX_BYTES, &tmA, k0, tn0, c, fb);
                        tma_tile_3d(dst + 3 * BOX_BYTES, &tmA, k0 + BOXK, tn0, c, fb);
                    }
                }
            }
            git += (uint32_t)KT;
            if (!diag) {
                mbar_wait(bar_s, sphase & 1);          // the consumers have stored S (generic proxy) ...
                ++sphase;
                fence_proxy_async();                   // ... which is now read back through TMA
                wait_flag(flags_c + (size_t)j * T + j, a.epoch, a.err);     // L_jj and W_j are final
                fence_proxy_async();
                for (int s4 = 0; s4 < SPB; ++s4) {
                    const uint32_t G = git + s4, sl = acquire_slot(G);
                    const uint32_t dst = ring + sl * STAGE_BYTES, fb = bar_full + 8 * sl;
                    mbar_expect_tx(fb, 4 * BOX_BYTES);
                    tma_tile_3d(dst, &tmA, tn0 + s4 * BK, tm0, c, fb);                          // S[rows i][p]
                    tma_tile_3d(dst + BOX_BYTES, &tmA, tn0 + s4 * BK + BOXK, tm0, c, fb);
                    tma_tile_2d(dst + 2 * BOX_BYTES, &tmW, s4 * BK, (c * T + j) * TB, fb);      // W_j[cc][p]
                    tma_tile_2d(dst + 3 * BOX_BYTES, &tmW, s4 * BK + BOXK, (c * T + j) * TB, fb);
                }
                git += SPB;
            } else {
                mbar_wait(bar_d, dphase & 1);          // the ring is scratch until the diagonal tile is finished
                ++dphase;
            }
        }
        return;
    }

    // ====================================== consumers: 8 warps, warp tile 32 x 64 ======================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(REGS_CONSUMER));
    // fragment addressing inside a 128 x 16 box: row r at r * 128 bytes, logical 16-byte chunk q at (q ^ (r & 7)) * 16
    const int xo0 = ((2 * t) ^ g) * 16, xo1 = ((2 * t + 1) ^ g) * 16;
    const int wm_off = warp & 3, wn_off = (warp >> 2) & 1;
    // Diagonal tiles need the lower triangle only: of the eight 32 x 64 warp blocks two lie above the diagonal, two are
    // full and four are crossed by it (10 or 26 of their 32 DMMA tiles are needed).  The six blocks are dealt to the warps
    // so that every sub-partition (warp & 3) gets the same work: {A, F}, {B, E}, {C}, {D} = 36, 36, 32, 32 DMMA tiles per k-step
    // (all eight blocks on their home warps would cost 64).  pattern 0: idle, 1: n-tile <= m-tile, 2: n-tile <= m-tile + 4, 3: full.
    const int wm_dg = (warp < 4) ? warp : (warp == 4 ? 3 : 2), wn_dg = (warp == 4 || warp == 5) ? 1 : 0;
    const int pat_dg = (warp == 0 || warp == 5) ? 1 : (warp == 1 || warp == 4) ? 2 : (warp < 4) ? 3 : 0;
    uint32_t git = 0;                                  // ring stages consumed so far
    for (uint32_t n = 0;; ++n) {
        const uint32_t qs = n % QD;
        mbar_wait(bar_qf + 8 * qs, (n / QD) & 1);
        const unsigned tk = sQ[qs];
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_qe + 8 * qs);
        if (tk >= a.total) break;
        int i, j, c;
        decode_ticket(tk, a.C, T, a.nsm, j, c, i);
        const bool diag = (i == j);
        const int KT = j * SPB;
        double* A = a.A + (size_t)c * a.stride;
        int* flags_c = a.flags + (size_t)c * T * T;
        const int tm0 = i * TB, tn0 = j * TB;
        const int wm = diag ? wm_dg : wm_off, wn = diag ? wn_dg : wn_off;       // this warp's 32 x 64 block of the tile
        const int offA = (wm * 32 + g) * 128, offB = (wn * 64 + g) * 128;
        const bool warp_active = !diag || pat_dg != 0;
        double acc[4][8][2];
        if (warp_active) {
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const int gi = tm0 + wm * 32 + mt * 8 + g;
                const double* crow = A + (size_t)gi * ld;
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    const int gj = tn0 + wn * 64 + nt * 8 + 2 * t;
                    double c0 = 0.0, c1 = 0.0;
                    if (gi < M) {
                        if (gj + 1 <= gi) {
                            const double2 cv = *reinterpret_cast<const double2*>(crow + gj);
                            c0 = cv.x; c1 = cv.y;
                        } else if (gj <= gi) {
                            c0 = crow[gj];
                        }
                    }
                    acc[mt][nt][0] = -c0;
                    acc[mt][nt][1] = -c1;
                }
            }
        }
        // K loop; pc = std::integral_constant of the block pattern (3 = all 32 DMMA tiles)
        auto k_loop = [&](auto pc, const int b_off) {
            constexpr int NTHI = (decltype(pc)::value == 1) ? 0 : (decltype(pc)::value == 2) ? 4 : 8;
            for (int kt = 0; kt < KT; ++kt) {
                const uint32_t G = git + kt, sl = G % STAGES;
                mbar_wait(bar_full + 8 * sl, (G / STAGES) & 1);
                if constexpr (decltype(pc)::value != 0) {
                    const uint8_t* sa = ring_g + sl * STAGE_BYTES + offA;
                    const uint8_t* sb = ring_g + sl * STAGE_BYTES + b_off + offB;
                    compute_box<0, NTHI>(acc, sa, sb, xo0, xo1);
                    compute_box<0, NTHI>(acc, sa + BOX_BYTES, sb + BOX_BYTES, xo0, xo1);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_empty + 8 * sl);
            }
        };
        if (!diag) k_loop(std::integral_constant<int, 3>{}, 2 * BOX_BYTES);
        else if (pat_dg == 3) k_loop(std::integral_constant<int, 3>{}, 0);          // B operand = the A boxes (rows j = rows i)
        else if (pat_dg == 2) k_loop(std::integral_constant<int, 2>{}, 0);
        else if (pat_dg == 1) k_loop(std::integral_constant<int, 1>{}, 0);
        else k_loop(std::integral_constant<int, 0>{}, 0);
        git += (uint32_t)KT;

        if (!diag) {
            // ---- S = D_ij - sum  ->  global (in place), read back as the A operand of  L_ij = S W_j^T ----
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const int gi = tm0 + wm * 32 + mt * 8 + g;
                if (gi >= M) continue;
                double* crow = A + (size_t)gi * ld;
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    const int gj = tn0 + wn * 64 + nt * 8 + 2 * t;           // gj + 1 < tn0 + 128 <= tm0 <= gi
                    *reinterpret_cast<double2*>(crow + gj) = make_double2(-acc[mt][nt][0], -acc[mt][nt][1]);
                }
            }
            fence_proxy_async();
            mbar_arrive(bar_s);
#pragma unroll
            for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;
            // X[r][cc] = sum_{p <= cc} S[r][p] W[cc][p], W lower triangular: zero blocks are skipped per 16 x 8 box
            auto trsm_stage = [&](auto s4c) {
                constexpr int S4 = decltype(s4c)::value;
                const uint32_t G = git + S4, sl = G % STAGES;
                mbar_wait(bar_full + 8 * sl, (G / STAGES) & 1);
                const uint8_t* sa = ring_g + sl * STAGE_BYTES + offA;
                const uint8_t* sb = ring_g + sl * STAGE_BYTES + 2 * BOX_BYTES + offB;
                trsm_box<2 * S4>(acc, wn, sa, sb, xo0, xo1);
                trsm_box<2 * S4 + 1>(acc, wn, sa + BOX_BYTES, sb + BOX_BYTES, xo0, xo1);
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_empty + 8 * sl);
            };
            trsm_stage(std::integral_constant<int, 0>{});
            trsm_stage(std::integral_constant<int, 1>{});
            trsm_stage(std::integral_constant<int, 2>{});
            trsm_stage(std::integral_constant<int, 3>{});
            git += SPB;
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const int gi = tm0 + wm * 32 + mt * 8 + g;
                if (gi >= M) continue;
                double* crow = A + (size_t)gi * ld;
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    const int gj = tn0 + wn * 64 + nt * 8 + 2 * t;
                    *reinterpret_cast<double2*>(crow + gj) = make_double2(acc[mt][nt][0], acc[mt][nt][1]);
                }
            }
            __threadfence();
            fence_proxy_async();
            cons_sync();
            if (tid == 0) st_release_gpu(flags_c + (size_t)i * T + j, a.epoch);
        } else {
            // ---- diagonal tile: S -> shared memory, L_jj = chol(S) and W_j = L_jj^-1 as 64 + 64 -------------
            cons_sync();                                          // every warp is done with the ring
            double* S11 = reinterpret_cast<double*>(ring_g);
            double* S21 = S11 + 64 * potf2::SLDP;
            double* S22 = S21 + 64 * potf2::SLDP;
            double* W11 = S22 + 64 * potf2::SLDP;
            double* W22 = W11 + 64 * potf2::SLDP;
            double* sCol = W22 + 64 * potf2::SLDP;
            double* sRinv = sCol + 64;
            const int nloc = min(TB, M - tn0);                    // rows / columns of the block that exist
            for (int idx = tid; idx < 64 * potf2::SLDP; idx += NCONS) { W11[idx] = 0.0; W22[idx] = 0.0; }
            if (warp_active) {
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    const int R = wm * 32 + mt * 8 + g;
#pragma unroll
                    for (int nt = 0; nt < 8; ++nt)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int Cc = wn * 64 + nt * 8 + 2 * t + e;
                            double v = (Cc <= R) ? -acc[mt][nt][e] : 0.0;
                            if (R >= nloc || Cc >= nloc) v = (R == Cc) ? 1.0 : 0.0;       // identity padding (ragged tile)
                            double* dst = (R < 64) ? S11 + R * potf2::SLDP + Cc
                                                   : (Cc < 64 ? S21 + (R - 64) * potf2::SLDP + Cc : S22 + (R - 64) * potf2::SLDP + (Cc - 64));
                            if (R >= 64 || Cc < 64) *dst = v;
                        }
                }
            }
            if (tid == 0) sFail = 0;
            cons_sync();
            const int g64r = 16 * (warp & 3), g64c = 32 * (warp >> 2);     // gemm64 output block of this warp
            double o[2][4][2];
#pragma unroll 1
            for (int hh = 0; hh < 2; ++hh) {
                double* Sb = hh ? S22 : S11;
                double* Wb = hh ? W22 : W11;
                const int nrem = nloc - 64 * hh;
                potf2::block64<LATENCY>(Sb, Wb, sCol, sRinv, (nrem > potf2::HB) ? 2 : 1, lane, warp, tn0 + 64 * hh, &sFail, [] { cons_sync(); });
                if (hh == 0) {
                    potf2::gemm64(S21, W11, false, warp, lane, o);             // L21 = S21 W11^T
                    cons_sync();
#pragma unroll
                    for (int mm = 0; mm < 2; ++mm)
#pragma unroll
                        for (int nn = 0; nn < 4; ++nn) {
                            const int r = g64r + 8 * mm + g, cc = g64c + 8 * nn + 2 * t;
                            S21[r * potf2::SLDP + cc] = o[mm][nn][0];
                            S21[r * potf2::SLDP + cc + 1] = o[mm][nn][1];
                            const int gi = tn0 + 64 + r;
                            if (gi < M) *reinterpret_cast<double2*>(A + (size_t)gi * ld + tn0 + cc) = make_double2(o[mm][nn][0], o[mm][nn][1]);
                        }
                    cons_sync();
                    potf2::gemm64(S21, S21, false, warp, lane, o);             // S22 -= L21 L21^T (lower part)
#pragma unroll
                    for (int mm = 0; mm < 2; ++mm)
#pragma unroll
                        for (int nn = 0; nn < 4; ++nn)
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int r = g64r + 8 * mm + g, cc = g64c + 8 * nn + 2 * t + e;
                                if (cc <= r && 64 + r < nloc) S22[r * potf2::SLDP + cc] -= o[mm][nn][e];
                            }
                    cons_sync();
                }
            }
            potf2::gemm64(S21, W11, true, warp, lane, o);                      // Tm = L21 W11
            cons_sync();
#pragma unroll
            for (int mm = 0; mm < 2; ++mm)
#pragma unroll
                for (int nn = 0; nn < 4; ++nn) {
                    const int r = g64r + 8 * mm + g, cc = g64c + 8 * nn + 2 * t;
                    S21[r * potf2::SLDP + cc] = o[mm][nn][0];
                    S21[r * potf2::SLDP + cc + 1] = o[mm][nn][1];
                }
            cons_sync();
            potf2::gemm64(W22, S21, true, warp, lane, o);                      // W21 = -W22 Tm
            double* Wg = a.Wbuf + ((size_t)c * T + j) * TB * TB;
#pragma unroll
            for (int mm = 0; mm < 2; ++mm)
#pragma unroll
                for (int nn = 0; nn < 4; ++nn) {
                    const int r = g64r + 8 * mm + g, cc = g64c + 8 * nn + 2 * t;
                    *reinterpret_cast<double2*>(Wg + (size_t)(64 + r) * TB + cc) = make_double2(-o[mm][nn][0], -o[mm][nn][1]);
                }
            // L11, L22 -> the matrix (lower triangle only); W11, 0, W22 -> Wbuf
            for (int idx = tid; idx < 64 * 64; idx += NCONS) {
                const int r = idx >> 6, cc = idx & 63;
                if (cc <= r) {
                    if (tn0 + r < M) A[(size_t)(tn0 + r) * ld + tn0 + cc] = S11[r * potf2::SLDP + cc];
                    if (tn0 + 64 + r < M) A[(size_t)(tn0 + 64 + r) * ld + tn0 + 64 + cc] = S22[r * potf2::SLDP + cc];
                }
                Wg[(size_t)r * TB + cc] = W11[r * potf2::SLDP + cc];
                Wg[(size_t)r * TB + 64 + cc] = 0.0;
                Wg[(size_t)(64 + r) * TB + 64 + cc] = W22[r * potf2::SLDP + cc];
            }
            __threadfence();
            fence_proxy_async();
            cons_sync();
            if (tid == 0) {
                if (sFail != 0 && a.info != nullptr && a.info[c] == 0) a.info[c] = sFail;
                st_release_gpu(flags_c + (size_t)j * T + j, a.epoch);
            }
            if (lane == 0) mbar_arrive(bar_d);                    // the ring may be refilled
        }
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;           // a driver entry point, not library state
    if (fn == nullptr) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

}  // namespace

size_t bdk_potrf_tiles_scratch_bytes(const bd_ctx* ctx)
{
    const size_t T = (size_t)(ctx->M + TB - 1) / TB;
    return sizeof(double) * (size_t)ctx->C * T * TB * TB;
}

size_t bdk_potrf_tiles_flag_words(const bd_ctx* ctx)
{
    const size_t T = (size_t)(ctx->M + TB - 1) / TB;
    return (size_t)ctx->C * T * T;
}

int bdk_potrf_tiles(bd_ctx* ctx, double* A, int64_t ld, int64_t stride, int32_t* info)
{
    const int M = ctx->M, C = ctx->C, T = (M + TB - 1) / TB;
    const uint64_t total64 = (uint64_t)C * T * (T + 1) / 2;
    if (total64 + 1024 > 0xffffffffull || (uint64_t)C * T * TB > 0x7fffffffull) return BD_ERR_ALLOC;
    if (ctx->tile_flags == nullptr) {                 // first factorisation of this context (flags are allocated last)
        if (ctx->tile_W == nullptr) BD_CUDA(ctx, cudaMalloc(&ctx->tile_W, bdk_potrf_tiles_scratch_bytes(ctx)));
        const size_t fb = sizeof(int) * ((size_t)C * T * T + 2);
        int* flags = nullptr;
        BD_CUDA(ctx, cudaMalloc(&flags, fb));
        cudaError_t e0 = cudaMemsetAsync(flags, 0, fb, ctx->stream);
        if (e0 != cudaSuccess) { cudaFree(flags); ctx->last_cuda = e0; return BD_ERR_CUDA; }
        ctx->tile_flags = flags;
        ctx->tile_epoch = 0;
        ctx->tile_ticket_base = 0;
        BD_CUDA(ctx, cudaFuncSetAttribute(k_potrf_tiles<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TILE_SMEM));
        BD_CUDA(ctx, cudaFuncSetAttribute(k_potrf_tiles<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TILE_SMEM));
    }
    EncodeTiledFn enc = encode_fn();
    if (enc == nullptr) { ctx->last_cuda = cudaErrorNotSupported; return BD_ERR_CUDA; }
    if (ctx->tile_mapA_ptr != A || ctx->tile_mapA_ld != ld || ctx->tile_mapA_stride != stride) {
        static_assert(sizeof(CUtensorMap) == sizeof(ctx->tile_maps[0]), "tensor map storage");
        CUtensorMap* mA = reinterpret_cast<CUtensorMap*>(&ctx->tile_maps[0]);
        CUtensorMap* mW = reinterpret_cast<CUtensorMap*>(&ctx->tile_maps[1]);
        // columns beyond M read as zero (the ragged last tile column), rows beyond M likewise
        const cuuint64_t dimA[3] = {(cuuint64_t)M, (cuuint64_t)M, (cuuint64_t)C};
        const cuuint64_t strA[2] = {(cuuint64_t)ld * 8, (cuuint64_t)stride * 8};
        const cuuint32_t boxA[3] = {BOXK, TB, 1}, es3[3] = {1, 1, 1};
        CUresult r1 = enc(mA, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, A, dimA, strA, boxA, es3, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        const cuuint64_t dimW[2] = {(cuuint64_t)TB, (cuuint64_t)C * T * TB};
        const cuuint64_t strW[1] = {(cuuint64_t)TB * 8};
        const cuuint32_t boxW[2] = {BOXK, TB}, es2[2] = {1, 1};
        CUresult r2 = enc(mW, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, ctx->tile_W, dimW, strW, boxW, es2, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r1 != CUDA_SUCCESS || r2 != CUDA_SUCCESS) { ctx->last_cuda = cudaErrorInvalidValue; return BD_ERR_CUDA; }
        ctx->tile_mapA_ptr = A; ctx->tile_mapA_ld = ld; ctx->tile_mapA_stride = stride;
    }
    TileArgs a;
    a.A = A; a.ld = ld; a.stride = stride; a.M = M; a.C = C; a.T = T; a.nsm = ctx->num_sms;
    a.Wbuf = ctx->tile_W;
    a.flags = ctx->tile_flags;
    a.epoch = ++ctx->tile_epoch;
    a.ticket = reinterpret_cast<unsigned*>(ctx->tile_flags + (size_t)C * T * T);
    a.err = ctx->tile_flags + (size_t)C * T * T + 1;
    a.ticket_base = ctx->tile_ticket_base;
    a.total = (unsigned)total64;
    a.info = info;
    const unsigned grid = (a.total < (unsigned)ctx->num_sms) ? a.total : (unsigned)ctx->num_sms;
    ctx->tile_ticket_base += a.total + grid;          // every CTA's producer draws exactly one ticket beyond the last tile
    const CUtensorMap& mapA = *reinterpret_cast<const CUtensorMap*>(&ctx->tile_maps[0]);
    const CUtensorMap& mapW = *reinterpret_cast<const CUtensorMap*>(&ctx->tile_maps[1]);
    // few tiles per column (C T / 2 on average, against num_sms CTAs): the diagonal tiles are the critical path
    if ((int64_t)C * T <= 2 * ctx->num_sms && T <= 64)
        BD_LAUNCH(ctx, k_potrf_tiles<true>, dim3(grid), dim3(NTHREADS), TILE_SMEM, mapA, mapW, a);
    else
        BD_LAUNCH(ctx, k_potrf_tiles<false>, dim3(grid), dim3(NTHREADS), TILE_SMEM, mapA, mapW, a);
    return 0;
}

// =================================================================================================
// bd_cholesky_noalloc -- the tile Cholesky for callers that cannot allocate (CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc).  Same kernel (k_potrf_tiles), but its scratch -- the inverse diagonal blocks W, the
// ready flags, the ticket counter and the error word -- lives in ONE file-scope device array of fixed size instead of
// the context's cudaMalloc'ed buffers.  No context is needed: the caller passes the matrices, the sizes and the stream.
//   limit: n_chains * ceil(M / 128) <= BD_NOALLOC_MAX_TILE_ROWS (32), e.g. one chain of M <= 4096, 2 of M <= 2048, 8 of
//          M <= 512, 32 of M <= 128.  The array is 4 MB + 4.2 KB; every GPU that loads libbd holds it until exit.
//   Every call shares the array: calls that overlap on the GPU (two streams, two host threads) RACE; serialise them.
//   The array keeps the last call's contents, so flags, ticket counter and error word are cleared on the stream at the
//   start of every call (W needs no clearing: every block that is read has been written by this call's diagonal tiles).
// In host code `g_noalloc_scratch` is only a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
// =================================================================================================
namespace {

constexpr int NOALLOC_MAX_TILE_ROWS = 32;                                          // C * T
constexpr size_t NOALLOC_W_BYTES = (size_t)NOALLOC_MAX_TILE_ROWS * TB * TB * sizeof(double);            // 4 MB
constexpr size_t NOALLOC_FLAG_WORDS = (size_t)NOALLOC_MAX_TILE_ROWS * NOALLOC_MAX_TILE_ROWS + 2;         // C T^2 <= (C T)^2, + ticket, error
constexpr size_t NOALLOC_BYTES = NOALLOC_W_BYTES + ((NOALLOC_FLAG_WORDS * sizeof(int) + 255) / 256) * 256;

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

struct NoAllocDevice {
    bool ready;
    unsigned char* scratch;      // device address of g_noalloc_scratch on this device
    int num_sms;
};
constexpr int NOALLOC_MAX_DEVICES = 64;
NoAllocDevice g_noalloc_dev[NOALLOC_MAX_DEVICES];     // set-up record per device (address of the symbol, SM count)
std::mutex g_noalloc_mutex;

// once per device, with that device current
int noalloc_setup(int dev, NoAllocDevice** out)
{
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    NoAllocDevice& d = g_noalloc_dev[dev];
    if (!d.ready) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || p == nullptr) return BD_ERR_CUDA;
        if (cudaFuncSetAttribute(k_potrf_tiles<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TILE_SMEM) != cudaSuccess) return BD_ERR_CUDA;
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return BD_ERR_CUDA;
        d.scratch = static_cast<unsigned char*>(p);
        d.num_sms = sms;
        d.ready = true;
    }
    *out = &d;
    return 0;
}

}  // namespace

extern "C" int bd_cholesky_noalloc(double* DL_dev, int32_t M, int32_t n_chains, int64_t ld, int64_t chain_stride,
                                   int32_t* info_dev, void* cuda_stream)
{
    if (DL_dev == nullptr || (reinterpret_cast<uintptr_t>(DL_dev) % 16) != 0) return -1;
    if (M < 1) return -2;
    if (n_chains < 1) return -3;
    if (ld < M || (ld % 2) != 0) return -4;
    if (chain_stride < ld * (int64_t)M || (chain_stride % 2) != 0) return -5;
    const int C = n_chains, T = (M + TB - 1) / TB;
    if ((int64_t)C * T > NOALLOC_MAX_TILE_ROWS) return BD_ERR_TOO_LARGE;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NOALLOC_MAX_DEVICES) return BD_ERR_CUDA;
    NoAllocDevice* d = nullptr;
    int rc = noalloc_setup(dev, &d);
    if (rc != 0) return rc;
    EncodeTiledFn enc = encode_fn();
    if (enc == nullptr) return BD_ERR_CUDA;

    double* Wbuf = reinterpret_cast<double*>(d->scratch);
    int* flags = reinterpret_cast<int*>(d->scratch + NOALLOC_W_BYTES);
    const size_t nflags = (size_t)C * T * T;                       // <= (C T)^2 <= NOALLOC_FLAG_WORDS - 2

    CUtensorMap mA, mW;                                            // host objects, passed to the kernel by value
    const cuuint64_t dimA[3] = {(cuuint64_t)M, (cuuint64_t)M, (cuuint64_t)C};
    const cuuint64_t strA[2] = {(cuuint64_t)ld * 8, (cuuint64_t)chain_stride * 8};
    const cuuint32_t boxA[3] = {BOXK, TB, 1}, es3[3] = {1, 1, 1};
    if (enc(&mA, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, DL_dev, dimA, strA, boxA, es3, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return BD_ERR_CUDA;
    const cuuint64_t dimW[2] = {(cuuint64_t)TB, (cuuint64_t)C * T * TB};
    const cuuint64_t strW[1] = {(cuuint64_t)TB * 8};
    const cuuint32_t boxW[2] = {BOXK, TB}, es2[2] = {1, 1};
    if (enc(&mW, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, Wbuf, dimW, strW, boxW, es2, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return BD_ERR_CUDA;

    // the array keeps the last call's contents: flags, ticket counter and error word start at zero
    if (cudaMemsetAsync(flags, 0, sizeof(int) * (nflags + 2), stream) != cudaSuccess) return BD_ERR_CUDA;
    if (info_dev != nullptr && cudaMemsetAsync(info_dev, 0, sizeof(int32_t) * (size_t)C, stream) != cudaSuccess) return BD_ERR_CUDA;

    TileArgs a;
    a.A = DL_dev; a.ld = ld; a.stride = chain_stride; a.M = M; a.C = C; a.T = T; a.nsm = d->num_sms;
    a.Wbuf = Wbuf;
    a.flags = flags;
    a.epoch = 1;
    a.ticket = reinterpret_cast<unsigned*>(flags + nflags);
    a.err = flags + nflags + 1;
    a.ticket_base = 0;
    a.total = (unsigned)((int64_t)C * T * (T + 1) / 2);
    a.info = info_dev;
    const unsigned grid = (a.total < (unsigned)d->num_sms) ? a.total : (unsigned)d->num_sms;
    k_potrf_tiles<false><<<dim3(grid), dim3(NTHREADS), TILE_SMEM, stream>>>(mA, mW, a);
    return (cudaGetLastError() == cudaSuccess) ? 0 : BD_ERR_CUDA;
}
