// chain_step.cu -- the whole per-timestep hot path (a0-a8) for SHORT chains (M = 3(N+1) <= 320) in ONE
// persistent kernel: one CTA owns one chain for all requested time steps; positions, forces, drift,
// noise and the Brownian displacement live in shared memory; the RPY tensor D is never stored.
//
// Cholesky (Eq. 10) is blocked LEFT-looking over column panels of NBP = 8*NT columns:
//   (a) the CTA generates the panel's block column of D pair by pair (Eqs. 7-9, :106-112) into a
//       shared-memory tile;
//   (b) S = D_panel - L[rows, :k0] L[panel, :k0]^T with FP64 tensor-core DMMA (m8n8k4): every warp owns
//       m-tiles (8 rows) mt = warp, warp+8, ...  L lives in global/L2 in a FRAGMENT-MAJOR layout
//       Lg[(col/4)][row][col%4]: for one k-group (4 columns) the fragments of ALL rows >= k0 are one
//       contiguous byte range, so a single TMA bulk copy (cp.async.bulk + mbarrier) per k-group feeds
//       the A fragments of every warp and the B fragments (the panel rows) through a 4-stage
//       shared-memory ring; each DMMA fragment is then one conflict-free 256-byte warp load;
//   (c) the NBP x NBP diagonal block is factored in registers by G x G threads (3x3 each), one named
//       barrier per pivot, and its inverse W = L_kk^-1 is accumulated by the same elimination steps;
//   (d) rows below the panel: X = S W^T, again DMMA, skipping the zero blocks of W; X is written to Lg
//       for the later panels and folded into y += X dW immediately (Eq. 6, :102), so L is never
//       re-read for the matvec.
// Finished rows of L are never needed again (left-looking), so the working set in L2 is small and
// stays resident while the CTA moves on to its next chain.
// After the last panel the CTA applies the semi-implicit rod update (Eqs. 14, 17, 15, :139-160).
#include <type_traits>

#include "bd_internal.cuh"
#include "block_ops.cuh"
#include "philox.cuh"
#include "tma.cuh"
#include "warp_chol.cuh"

namespace {

constexpr int CS_THREADS = 256;
constexpr int CS_WARPS = 8;
constexpr int CS_MTW = 5;                 // m-tiles per warp  -> M <= 8*8*5 = 320
constexpr int CS_MAXM = 8 * CS_WARPS * CS_MTW;
constexpr int CS_KG = 2;                  // k-groups per ring stage: one mbarrier round trip (~90 cycles) per CS_KG k-groups
constexpr int CS_STAGES = 2;              // ring stages

struct ChainStepParams {
    int N, C;
    double b, hstar, a_s, inv_a, inv_b, dt;
    SpringLaw sl;
    double kap[9];
    uint64_t seed, chain0, first_step;
    int n_steps, noise_kind;
    double* r;            // [C][Nb][3], updated in place
    double* scratch;      // per-CTA L storage, fragment-major, MP*MP doubles each
    int64_t scratch_stride;
    int32_t* info;        // [C]
};

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}
template <int NT>
__global__ void __launch_bounds__(CS_THREADS, (NT <= 3) ? 2 : 1) k_chain_step(ChainStepParams P)
{
    constexpr int NBP = 8 * NT;            // panel width (columns)
    constexpr int NQP = NBP / 4;           // k-groups per panel
    constexpr int PB = NBP / 3;            // beads per panel
    constexpr int WS = NBP + 4;            // row stride of W (conflict-free B fragments)

    const int N = P.N, Nb = N + 1, M = 3 * Nb;
    const int MP = (M + 7) & ~7, nmt = MP >> 3;
    const int MT4 = (MP + 1) * 4;          // tile k-group stride in doubles ((MP+1) rows: spreads banks)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;

    extern __shared__ __align__(128) double sm[];
    const int slot_d = (max(MP - NBP, NBP) * 4 + 15) & ~15;     // ring slot: rows k0..MP-1 of one k-group, k0 >= NBP
    const int slot_s = CS_KG * slot_d;                          // one ring stage = CS_KG k-groups
    double* ring = sm;                                          // [CS_STAGES][CS_KG][slot_d]   operand ring (TMA destination)
    double* tile = ring + CS_STAGES * slot_s;                   // [NQP][MP+1][4]  panel block column, fragment-major
    double* winv = tile + (size_t)NQP * MT4;                    // [NBP][WS] inverse of the diagonal block
    double* sR = winv + NBP * WS;                               // [MP] positions
    double* sF = sR + MP;                                       // [MP] bead forces (later: unshifted new positions)
    double* sV = sF + MP;                                       // [MP] drift D.F
    double* sY = sV + MP;                                       // [MP] L.dW
    double* sDW = sY + MP;                                      // [MP + NBP] Brownian increments, zero padded
    double* sCol = sDW + MP + NBP;                              // [2][32] column broadcast buffer of warp_chol
    double* sScan = sCol + 64;                                  // [96]
    double* sRinv = sScan + 96;                                 // [32] 1 / L_kk of the current diagonal block
    __shared__ int sFail;
    __shared__ __align__(8) uint64_t sBar[2 * CS_STAGES];       // full[0..S), empty[S..2S)

    auto TIDX = [&](int r, int c) { return (c >> 2) * MT4 + r * 4 + (c & 3); };

    double* Lg = P.scratch + (size_t)blockIdx.x * P.scratch_stride;
    // (A triangular Lg -- rows >= 4 (col / 4) only, 110 MB instead of 219 MB for the 296 resident CTAs of c2, all of it in
    // L2 -- was measured in round 2: 6 % SLOWER (9.77e5 against 1.04e6 chain-steps/s): the offset arithmetic costs more than
    // the DRAM spill, which is not the limiter at 0.37 TB/s.)
    const uint32_t bar_full = smem_u32(&sBar[0]), bar_empty = smem_u32(&sBar[CS_STAGES]);
    const uint32_t ring_u32 = smem_u32(ring);
    if (tid == 0) {
        for (int s = 0; s < CS_STAGES; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, CS_WARPS); }
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t git = 0;                      // global k-group counter (ring position / barrier parity), same in all threads

    for (int c = blockIdx.x; c < P.C; c += gridDim.x) {
        double* rg = P.r + (size_t)c * M;
        for (int i = tid; i < MP; i += CS_THREADS) sR[i] = (i < M) ? rg[i] : 0.0;
        int chain_info = 0;
        __syncthreads();

        for (int s = 0; s < P.n_steps; ++s) {
            const uint64_t step = P.first_step + (uint64_t)s;
            // ---- a1: tensions -> net bead forces (Eq. 3, Eq. 1/22) ---------------------------------
            for (int j = tid; j <= N; j += CS_THREADS) {
                double Tl[3] = {0, 0, 0}, Tr[3] = {0, 0, 0};
#pragma unroll
                for (int side = 0; side < 2; ++side) {
                    const int k = j - 1 + side;
                    if (k < 0 || k >= N) continue;
                    const double qx = sR[3 * k + 3] - sR[3 * k], qy = sR[3 * k + 4] - sR[3 * k + 1], qz = sR[3 * k + 5] - sR[3 * k + 2];
                    const double q = sqrt(qx * qx + qy * qy + qz * qz);
                    const double cf = spring_coeff(P.sl, q);
                    double* T = side ? Tr : Tl;
                    T[0] = cf * qx; T[1] = cf * qy; T[2] = cf * qz;
                }
                sF[3 * j] = Tr[0] - Tl[0]; sF[3 * j + 1] = Tr[1] - Tl[1]; sF[3 * j + 2] = Tr[2] - Tl[2];
            }
            // ---- a0: Brownian increments ------------------------------------------------------------
            for (int p = tid; 2 * p < MP + NBP; p += CS_THREADS) {
                double w0 = 0.0, w1 = 0.0;
                if (2 * p < M) brownian_pair(P.seed, (uint32_t)p, P.chain0 + (uint64_t)c, step, P.noise_kind, P.dt, w0, w1);
                sDW[2 * p] = w0;
                if (2 * p + 1 < MP + NBP) sDW[2 * p + 1] = (2 * p + 1 < M) ? w1 : 0.0;
            }
            for (int i = tid; i < MP; i += CS_THREADS) sY[i] = 0.0;
            if (tid == 0) sFail = 0;
            __syncthreads();

            // ---- a2 + a3 + a5: left-looking blocked Cholesky with on-the-fly D and fused y = L dW ------
            for (int k0 = 0; k0 < M; k0 += NBP) {
                const int pw = min(NBP, M - k0);               // panel width (multiple of 3)
                const int jb0 = k0 / 3, npb = pw / 3, nrb = Nb - jb0;
                const int nq = k0 >> 2;
                const uint32_t stage_bytes = (uint32_t)(MP - k0) * 32u;
                // operand ring prologue: the first CS_STAGES-1 k-groups of this panel (thread 0 = producer)
                // k-groups per ring stage: as many as fit into a stage (sized for CS_KG k-groups of the longest panel) and
                // divide nq (a multiple of 6) -- one mbarrier round trip (~90 cycles) then covers 2, 3 or 6 k-groups
                const int sub_d = (MP - k0) * 4;                // doubles of one k-group (rows k0 .. MP-1)
                const int kg = (6 * sub_d <= slot_s) ? 6 : (3 * sub_d <= slot_s) ? 3 : CS_KG;
                const int nqs = nq / kg;                        // stages of this panel
                auto produce = [&](int qs, uint32_t Gs) {       // thread 0: stage qs of this panel -> ring slot Gs % S
                    const uint32_t sl = Gs % CS_STAGES;
                    if (Gs >= CS_STAGES) mbar_wait(bar_empty + 8 * sl, ((Gs / CS_STAGES) - 1) & 1);
                    mbar_expect_tx(bar_full + 8 * sl, kg * stage_bytes);
                    for (int h = 0; h < kg; ++h)
                        tma_bulk_g2s(ring_u32 + (sl * slot_s + h * sub_d) * 8, Lg + ((size_t)(qs * kg + h) * MP + k0) * 4, stage_bytes,
                                     bar_full + 8 * sl);
                };
                if (tid == 0) {
                    for (int q = 0; q < CS_STAGES - 1 && q < nqs; ++q) produce(q, git + q);
                }
                // (a) block column of D: pairs (row bead jb0+ib, panel bead jb0+jb)
                for (int p = tid; p < nrb * PB; p += CS_THREADS) {
                    const int ib = p / PB, jb = p - ib * PB;
                    double blk[3][3];
                    if (jb >= npb) {
#pragma unroll
                        for (int kk = 0; kk < 3; ++kk)
#pragma unroll
                            for (int l = 0; l < 3; ++l) blk[kk][l] = 0.0;
                    } else {
                        const int i = jb0 + ib, j = jb0 + jb;
                        double cI = 1.0, cRR = 0.0, d[3] = {0.0, 0.0, 0.0};
                        if (i != j) {
                            d[0] = (sR[3 * i] - sR[3 * j]) * P.inv_b; d[1] = (sR[3 * i + 1] - sR[3 * j + 1]) * P.inv_b;
                            d[2] = (sR[3 * i + 2] - sR[3 * j + 2]) * P.inv_b;
                            rpy_coeffs(d[0] * d[0] + d[1] * d[1] + d[2] * d[2], P.hstar, P.a_s, P.inv_a, cI, cRR);
                        }
#pragma unroll
                        for (int kk = 0; kk < 3; ++kk)
#pragma unroll
                            for (int l = 0; l < 3; ++l) blk[kk][l] = cRR * d[kk] * d[l] + ((kk == l) ? cI : 0.0);
                    }
#pragma unroll
                    for (int kk = 0; kk < 3; ++kk)
#pragma unroll
                        for (int l = 0; l < 3; ++l) tile[TIDX(3 * ib + kk, 3 * jb + l)] = blk[kk][l];
                }
                for (int q = tid; q < (MP - M) * NBP; q += CS_THREADS)          // padding rows M..MP-1
                    tile[TIDX(M - k0 + q / NBP, q % NBP)] = 0.0;
                __syncthreads();

                // (b) S = D - L[rows, :k0] L[panel, :k0]^T, operands from the TMA ring
                double acc[CS_MTW][NT][2];
                bool act[CS_MTW];
#pragma unroll
                for (int i = 0; i < CS_MTW; ++i) {
                    const int mt = warp + CS_WARPS * i;
                    act[i] = (mt < nmt) && (8 * mt >= k0);
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) acc[i][nt][0] = acc[i][nt][1] = 0.0;
                }
                {
                    // m-tiles below k0 are retired: the active ones are i >= imin.  A predicated-off DMMA still
                    // occupies the tensor pipe (measured), so the loop is specialised per imin with real branches.
                    const int a_off = (8 * warp - k0 + g) * 4 + t;             // + i*256 doubles per m-tile step
                    const int b_off = g * 4 + t;                               // + nt*32
                    auto gemm = [&](auto i0c) {
                        constexpr int I0 = decltype(i0c)::value;
                        for (int q = 0; q < nqs; ++q) {
                            const uint32_t G_ = git + q, sl = G_ % CS_STAGES;
                            mbar_wait(bar_full + 8 * sl, (G_ / CS_STAGES) & 1);
                            // refill first (stage q + S - 1 goes where stage q - 1 was): the copy flies during this stage's DMMAs
                            if (tid == 0 && q + CS_STAGES - 1 < nqs) produce(q + CS_STAGES - 1, G_ + CS_STAGES - 1);
                            if constexpr (I0 < CS_MTW) {
                                for (int h = 0; h < kg; ++h) {
                                    const double* st = ring + (size_t)sl * slot_s + h * sub_d;
                                    double af[CS_MTW], bf[NT];
#pragma unroll
                                    for (int nt = 0; nt < NT; ++nt) bf[nt] = st[b_off + nt * 32];
#pragma unroll
                                    for (int i = I0; i < CS_MTW; ++i) af[i] = (i + 1 < CS_MTW || act[i]) ? st[a_off + i * (8 * CS_WARPS * 4)] : 0.0;
#pragma unroll
                                    for (int i = I0; i < CS_MTW; ++i) {
                                        if (i + 1 == CS_MTW && !act[i]) continue;  // only the last slot can lie beyond nmt
#pragma unroll
                                        for (int nt = 0; nt < NT; ++nt) dmma(acc[i][nt][0], acc[i][nt][1], af[i], bf[nt]);
                                    }
                                }
                            }
                            __syncwarp();
                            if (lane == 0) mbar_arrive(bar_empty + 8 * sl);    // this warp is done with the slot
                        }
                    };
                    int imin = 0;
#pragma unroll
                    for (int i = 0; i < CS_MTW; ++i)
                        if (8 * (warp + CS_WARPS * i) < k0) imin = i + 1;
                    // slots below the last one are always inside the matrix when active (nmt > 8*(CS_MTW-1) is not
                    // guaranteed for short chains, so fall back to "nothing active" when this warp has no tile at all)
                    if (imin < CS_MTW && !act[imin]) imin = CS_MTW;
                    if (imin < CS_MTW - 1 && !act[CS_MTW - 2]) {
                        // short chain: fewer than CS_MTW-1 slots in use -> generic predicated path is cheap enough
                        for (int q = 0; q < nqs; ++q) {
                            const uint32_t G_ = git + q, sl = G_ % CS_STAGES;
                            mbar_wait(bar_full + 8 * sl, (G_ / CS_STAGES) & 1);
                            if (tid == 0 && q + CS_STAGES - 1 < nqs) produce(q + CS_STAGES - 1, G_ + CS_STAGES - 1);
                            for (int h = 0; h < kg; ++h) {
                                const double* st = ring + (size_t)sl * slot_s + h * sub_d;
                                double bf[NT];
#pragma unroll
                                for (int nt = 0; nt < NT; ++nt) bf[nt] = st[b_off + nt * 32];
#pragma unroll
                                for (int i = 0; i < CS_MTW; ++i) {
                                    if (!act[i]) continue;
                                    const double af = st[a_off + i * (8 * CS_WARPS * 4)];
#pragma unroll
                                    for (int nt = 0; nt < NT; ++nt) dmma(acc[i][nt][0], acc[i][nt][1], af, bf[nt]);
                                }
                            }
                            __syncwarp();
                            if (lane == 0) mbar_arrive(bar_empty + 8 * sl);
                        }
                    } else {
                        switch (imin) {
                            case 0: gemm(std::integral_constant<int, 0>{}); break;
                            case 1: gemm(std::integral_constant<int, 1>{}); break;
                            case 2: gemm(std::integral_constant<int, 2>{}); break;
                            case 3: gemm(std::integral_constant<int, 3>{}); break;
                            case 4: gemm(std::integral_constant<int, 4>{}); break;
                            default: gemm(std::integral_constant<int, CS_MTW>{}); break;
                        }
                    }
                    git += (uint32_t)nqs;
                }
#pragma unroll
                for (int i = 0; i < CS_MTW; ++i)
                    if (act[i]) {
                        const int rr = 8 * (warp + CS_WARPS * i) - k0 + g;
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            double2* tp = reinterpret_cast<double2*>(tile + TIDX(rr, 8 * nt + 2 * t));
                            double2 dv = *tp;
                            dv.x -= acc[i][nt][0];
                            dv.y -= acc[i][nt][1];
                            *tp = dv;
                        }
                    }
                __syncthreads();

                // (c) diagonal block, warp 0: L_kk (back into the tile) and W = L_kk^-1 (-> winv), one row per lane,
                //     registers + shuffles (warp_chol.cuh): ~100 cycles per pivot instead of a CTA barrier and a
                //     division per pivot.  Warps 1..7 meanwhile compute this panel's slice of the drift v = D F
                //     (a4, Eq. 6 second term; D blocks recomputed from positions, Eqs. 7-9), which nothing in the
                //     factorisation depends on.
                const int nrows = min(NBP, MP - k0);                           // rows of the block that exist (ragged last panel)
                if (warp == 0) {
                    double x[NBP];
#pragma unroll
                    for (int j = 0; j < NBP; ++j) {
                        double val = (lane == j) ? 1.0 : 0.0;                   // identity padding (ragged last panel)
                        if (lane < pw && j < pw) val = tile[TIDX(max(lane, j), min(lane, j))];
                        x[j] = (lane < NBP) ? val : 0.0;
                    }
                    const bool row_ok = lane < nrows;
                    __syncwarp();
                    const int f = warp_chol<NBP, 4>(x, lane, sCol, sRinv, 1, [&](int k, double l) {
                        if (row_ok) tile[TIDX(lane, k)] = (lane >= k) ? l : 0.0;
                    });
                    if (lane == 0 && f != 0 && sFail == 0) sFail = k0 + f;
                } else if (warp == 1) {
                    // W = L_kk^-1 (-> winv) by forward substitution, 4 pivots behind warp 0 (named barriers 1..6)
                    warp_inverse<NBP, 4, WS>(lane, nrows, sRinv, winv, 1, [&](int k, int j) { return tile[TIDX(k, j)]; });
                } else {
                    const int npan = (M + NBP - 1) / NBP, bps = (Nb + npan - 1) / npan;
                    const int ib0 = (k0 / NBP) * bps, ib1 = min(ib0 + bps, Nb);
                    for (int i = ib0 + warp - 2; i < ib1; i += CS_WARPS - 2) {
                        const double xi = sR[3 * i], yi = sR[3 * i + 1], zi = sR[3 * i + 2];
                        double s0 = 0, s1 = 0, s2 = 0;
                        for (int j = lane; j < Nb; j += 32) {
                            const double fx = sF[3 * j], fy = sF[3 * j + 1], fz = sF[3 * j + 2];
                            if (j == i) { s0 += fx; s1 += fy; s2 += fz; continue; }
                            const double dx = (xi - sR[3 * j]) * P.inv_b, dy = (yi - sR[3 * j + 1]) * P.inv_b, dz = (zi - sR[3 * j + 2]) * P.inv_b;
                            double cI, cRR;
                            rpy_coeffs(dx * dx + dy * dy + dz * dz, P.hstar, P.a_s, P.inv_a, cI, cRR);
                            const double dot = cRR * (dx * fx + dy * fy + dz * fz);
                            s0 += cI * fx + dot * dx; s1 += cI * fy + dot * dy; s2 += cI * fz + dot * dz;
                        }
                        s0 = warp_sum(s0); s1 = warp_sum(s1); s2 = warp_sum(s2);
                        if (lane == 0) { sV[3 * i] = s0; sV[3 * i + 1] = s1; sV[3 * i + 2] = s2; }
                    }
                }
                __syncthreads();

                // (d) rows below the panel: X = S W^T (DMMA, zero blocks of W skipped); panel rows: L_kk.
                //     X -> Lg (fragment-major) and y += X dW.
                //     The fragments of W are the same for every m-tile of the warp: loaded once per panel.
                double wf[2 * NT][NT];
#pragma unroll
                for (int qq = 0; qq < 2 * NT; ++qq)
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) wf[qq][nt] = (qq <= 2 * nt + 1) ? winv[(8 * nt + g) * WS + 4 * qq + t] : 0.0;
#pragma unroll
                for (int i = 0; i < CS_MTW; ++i) {
                    if (!act[i]) continue;
                    const int mt = warp + CS_WARPS * i;
                    const int rr = 8 * mt - k0 + g;
                    double x[NT][2];
                    if (8 * mt >= k0 + NBP) {
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) x[nt][0] = x[nt][1] = 0.0;
#pragma unroll
                        for (int qq = 0; qq < 2 * NT; ++qq) {
                            const double af = tile[qq * MT4 + rr * 4 + t];
#pragma unroll
                            for (int nt = 0; nt < NT; ++nt)
                                if (qq <= 2 * nt + 1) dmma(x[nt][0], x[nt][1], af, wf[qq][nt]);
                        }
                    } else {
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) {
                            const double2 lv = *reinterpret_cast<const double2*>(tile + TIDX(rr, 8 * nt + 2 * t));
                            x[nt][0] = lv.x; x[nt][1] = lv.y;
                        }
                    }
                    double part = 0.0;
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) {
                        part += x[nt][0] * sDW[k0 + 8 * nt + 2 * t] + x[nt][1] * sDW[k0 + 8 * nt + 2 * t + 1];
                        // columns >= MP (ragged last panel) do not exist in Lg: k-group q >= MP/4 would land in the
                        // NEXT CTA's scratch (rows 8mt.. of its k-groups 0, 1) and corrupt a chain in flight there
                        if (k0 + 8 * nt >= MP) continue;
                        const int q = (k0 >> 2) + 2 * nt + (t >> 1);
                        *reinterpret_cast<double2*>(Lg + ((size_t)q * MP + 8 * mt + g) * 4 + 2 * (t & 1)) = make_double2(x[nt][0], x[nt][1]);
                    }
                    part += __shfl_xor_sync(0xffffffffu, part, 1);
                    part += __shfl_xor_sync(0xffffffffu, part, 2);
                    if (t == 0) sY[8 * mt + g] += part;
                }
                fence_proxy_async();                                          // Lg stores (generic proxy) before later TMA reads
                __syncthreads();
            }

            // ---- a6-a8: semi-implicit rod update, position rebuild, centre of mass -> 0 ----------------
            const int fail = sFail;
            if (fail != 0) {
                if (chain_info == 0) chain_info = fail;
                __syncthreads();
                continue;                                          // reading A10: state unchanged
            }
            bool bad = false;
            {
                double carry[3] = {0.0, 0.0, 0.0}, sum[3] = {0.0, 0.0, 0.0};
                for (int base = 0; base < N; base += CS_THREADS) {
                    const int k = base + tid;
                    double q[3] = {0.0, 0.0, 0.0};
                    if (k < N) {
                        double ra[3], rb[3], Y[3];
#pragma unroll
                        for (int d = 0; d < 3; ++d) { ra[d] = sR[3 * k + d]; rb[d] = sR[3 * k + 3 + d]; }
                        const double Q[3] = {rb[0] - ra[0], rb[1] - ra[1], rb[2] - ra[2]};
                        const double qn = sqrt(Q[0] * Q[0] + Q[1] * Q[1] + Q[2] * Q[2]);
                        const double tc = spring_coeff(P.sl, qn);
#pragma unroll
                        for (int d = 0; d < 3; ++d) {
                            const double fa = P.kap[3 * d] * ra[0] + P.kap[3 * d + 1] * ra[1] + P.kap[3 * d + 2] * ra[2];
                            const double fb = P.kap[3 * d] * rb[0] + P.kap[3 * d + 1] * rb[1] + P.kap[3 * d + 2] * rb[2];
                            const double ua = P.dt * (fa + sV[3 * k + d]) + sY[3 * k + d];
                            const double ub = P.dt * (fb + sV[3 * k + 3 + d]) + sY[3 * k + 3 + d];
                            Y[d] = Q[d] + (ub - ua) + 2.0 * P.dt * (tc * Q[d]);
                        }
                        const double Yn = sqrt(Y[0] * Y[0] + Y[1] * Y[1] + Y[2] * Y[2]);
                        const double scale = implicit_length(P.sl, Yn) / Yn;
                        if (!(Yn > 0.0) || !isfinite(scale)) bad = true;
                        q[0] = Y[0] * scale; q[1] = Y[1] * scale; q[2] = Y[2] * scale;
                    }
                    block_scan3(q[0], q[1], q[2], sScan, carry);
                    if (k < N) {
                        sF[3 * k + 3] = q[0]; sF[3 * k + 4] = q[1]; sF[3 * k + 5] = q[2];
                        sum[0] += q[0]; sum[1] += q[1]; sum[2] += q[2];
                    }
                }
                double cm[3];
                for (int d = 0; d < 3; ++d) cm[d] = block_sum(sum[d], sScan) / (double)Nb;
                const int anybad = __syncthreads_or((int)bad || !isfinite(cm[0]) || !isfinite(cm[1]) || !isfinite(cm[2]));
                if (anybad) {
                    if (chain_info == 0) chain_info = M + 1;
                } else {
                    for (int i = tid; i < Nb; i += CS_THREADS) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) sR[3 * i + d] = ((i == 0) ? 0.0 : sF[3 * i + d]) - cm[d];
                    }
                }
                __syncthreads();
            }
        }
        for (int i = tid; i < M; i += CS_THREADS) rg[i] = sR[i];
        if (tid == 0 && chain_info != 0 && P.info[c] == 0) P.info[c] = chain_info;
        __syncthreads();
    }
}

template <int NT>
size_t chain_step_smem(int M)
{
    const int NBP = 8 * NT, MP = (M + 7) & ~7;
    const size_t slot_d = ((size_t)(MP - NBP > NBP ? MP - NBP : NBP) * 4 + 15) & ~(size_t)15;
    return sizeof(double) * (CS_STAGES * CS_KG * slot_d + (size_t)(NBP / 4) * (MP + 1) * 4 + (size_t)NBP * (NBP + 4) + 4 * (size_t)MP +
                             (MP + NBP) + 64 + 96 + 32);
}

}  // namespace

bool bdk_chain_step_supported(const bd_ctx* ctx) { return ctx->M <= CS_MAXM; }

// persistent launch: one CTA per chain slot; each CTA needs MP*MP doubles of L scratch taken from the
// caller's workspace.
int bdk_chain_step(bd_ctx* ctx, double* r, uint64_t first_step, int n_steps)
{
    constexpr int NT = 3;
    const size_t smem = chain_step_smem<NT>(ctx->M);
    if (!ctx->attr_chain) {
        BD_CUDA(ctx, cudaFuncSetAttribute(k_chain_step<NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        ctx->attr_chain = true;
    }
    int per_sm = 0;
    BD_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_chain_step<NT>, CS_THREADS, smem));
    if (per_sm < 1) return BD_ERR_CUDA;
    const int MP = (ctx->M + 7) & ~7;
    ChainStepParams P;
    P.N = ctx->N; P.C = ctx->C;
    P.b = ctx->p.b; P.hstar = ctx->p.hstar; P.a_s = ctx->p.a / ctx->p.b; P.inv_a = ctx->p.b / ctx->p.a; P.inv_b = 1.0 / ctx->p.b;
    P.sl = make_spring_law(ctx->p); P.dt = ctx->p.dt;
    for (int i = 0; i < 9; ++i) P.kap[i] = ctx->p.kappa[i];
    P.seed = ctx->p.seed; P.chain0 = ctx->p.chain_id0; P.first_step = first_step;
    P.n_steps = n_steps; P.noise_kind = ctx->p.noise_kind;
    P.r = r; P.scratch = ctx->ws; P.info = ctx->info;
    P.scratch_stride = (int64_t)MP * MP;
    int grid = ctx->num_sms * per_sm;
    if (grid > ctx->C) grid = ctx->C;
    BD_LAUNCH(ctx, k_chain_step<NT>, dim3(grid), dim3(CS_THREADS), smem, P);
    return 0;
}
