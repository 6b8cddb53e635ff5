// update.cu -- O(N) stages of the hot path: initial walk, spring tensions / bead forces (a1),
// HI drift v = D F recomputed from positions (a4), and the semi-implicit rod update with position
// rebuild (a6-a8).  Citations: /root/reference/PAPER.md lines.
#include "bd_internal.cuh"
#include "philox.cuh"
#include "block_ops.cuh"

namespace {

constexpr int kUpdThreads = 256;

// Rebuild positions from link vectors held one per thread per chunk: p_0 = 0, p_{k+1} = p_k + Q_k,
// written unshifted to `tmp`, then shifted so that the centre of mass is 0 and written to r_out
// (reading A8).  link(k, Q) must return the k-th link vector.
template <class LinkFn>
__device__ void rebuild_positions(int N, double* tmp, double* r_out, double* s_buf, bool& bad, LinkFn link)
{
    double carry[3] = {0.0, 0.0, 0.0};
    double sum[3] = {0.0, 0.0, 0.0};
    for (int base = 0; base < N; base += blockDim.x) {
        const int k = base + threadIdx.x;
        double q[3] = {0.0, 0.0, 0.0};
        if (k < N) link(k, q);
        block_scan3(q[0], q[1], q[2], s_buf, carry);
        if (k < N) {
            tmp[3 * (k + 1) + 0] = q[0]; tmp[3 * (k + 1) + 1] = q[1]; tmp[3 * (k + 1) + 2] = q[2];
            sum[0] += q[0]; sum[1] += q[1]; sum[2] += q[2];
        }
    }
    double cm[3];
    for (int d = 0; d < 3; ++d) cm[d] = block_sum(sum[d], s_buf) / (double)(N + 1);
    const int anybad = __syncthreads_or((int)bad || !isfinite(cm[0]) || !isfinite(cm[1]) || !isfinite(cm[2]));
    bad = anybad != 0;
    if (bad) return;
    for (int i = threadIdx.x; i <= N; i += blockDim.x) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double p = (i == 0) ? 0.0 : tmp[3 * i + d];
            r_out[3 * i + d] = p - cm[d];
        }
    }
}

// -------------------------------------------------------------------------------------------------
// Initial conformation: freely jointed walk, link k from Philox purpose 1, pair k, step 0:
// z = 2 u1 - 1, phi = 2 pi u2, Q = b (s cos phi, s sin phi, z), s = sqrt(1 - z^2)   (reading A13).
__global__ void __launch_bounds__(kUpdThreads) k_init_walk(int N, double b, uint64_t seed, uint64_t chain0,
                                                           double* __restrict__ tmp_all, double* __restrict__ r_all)
{
    __shared__ double s_buf[96];
    const int c = blockIdx.x;
    const size_t M = 3 * (size_t)(N + 1);
    bool bad = false;
    rebuild_positions(N, tmp_all + c * M, r_all + c * M, s_buf, bad, [&](int k, double* q) {
        Philox2 u = philox_uniform_pair(seed, (uint32_t)k, chain0 + (uint64_t)c, 0ull, 1u);
        const double z = 2.0 * u.u1 - 1.0;
        double sn, cs;
        sincos(6.283185307179586 * u.u2, &sn, &cs);
        const double s = sqrt(1.0 - z * z);
        q[0] = b * (s * cs); q[1] = b * (s * sn); q[2] = b * z;
    });
}

// -------------------------------------------------------------------------------------------------
// a1: T_k = K (|Q_k| - b)/|Q_k| Q_k (Eq. 3, :76);  F_0 = T_0, F_j = T_j - T_{j-1}, F_N = -T_{N-1}
// (Eq. 1 net spring term :68, Eq. 22 :235).  One thread per bead j computes T_{j-1} and T_j.
__device__ __forceinline__ void tension(const double* __restrict__ r, int k, const SpringLaw& sl, double T[3])
{
    const double qx = r[3 * k + 3] - r[3 * k], qy = r[3 * k + 4] - r[3 * k + 1], qz = r[3 * k + 5] - r[3 * k + 2];
    const double q = sqrt(qx * qx + qy * qy + qz * qz);
    const double c = spring_coeff(sl, q);
    T[0] = c * qx; T[1] = c * qy; T[2] = c * qz;
}

__global__ void __launch_bounds__(256) k_forces(int N, int nblk, SpringLaw sl, const double* __restrict__ r_all,
                                                double* __restrict__ T_all, double* __restrict__ F_all)
{
    const int c = blockIdx.x / nblk;                       // chain and block both on grid.x
    const int j = (blockIdx.x - c * nblk) * blockDim.x + threadIdx.x;
    if (j > N) return;
    const double* r = r_all + (size_t)c * 3 * (N + 1);
    double Tl[3] = {0, 0, 0}, Tr[3] = {0, 0, 0};
    if (j > 0) tension(r, j - 1, sl, Tl);
    if (j < N) tension(r, j, sl, Tr);
    if (T_all != nullptr && j < N) {
        double* T = T_all + (size_t)c * 3 * N;
        T[3 * j] = Tr[0]; T[3 * j + 1] = Tr[1]; T[3 * j + 2] = Tr[2];
    }
    if (F_all != nullptr) {
        double* F = F_all + (size_t)c * 3 * (N + 1);
        F[3 * j] = Tr[0] - Tl[0]; F[3 * j + 1] = Tr[1] - Tl[1]; F[3 * j + 2] = Tr[2] - Tl[2];
    }
}

// a4: v_i = sum_j D_ij F_j (Eq. 6 second term, :102) with D_ij recomputed from positions (Eqs. 7-9),
// so D is never read for the drift.  One warp per bead i, lanes stride over j.
__global__ void __launch_bounds__(256) k_drift(int N, int nblk, double hstar, double a_s, double inv_a, double inv_b,
                                               const double* __restrict__ r_all, const double* __restrict__ F_all,
                                               double* __restrict__ v_all)
{
    const int c = blockIdx.x / nblk;
    const int Nb = N + 1;
    const int i = (blockIdx.x - c * nblk) * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= Nb) return;
    const int lane = threadIdx.x & 31;
    const double* r = r_all + (size_t)c * 3 * Nb;
    const double* F = F_all + (size_t)c * 3 * Nb;
    const double xi = r[3 * i], yi = r[3 * i + 1], zi = r[3 * i + 2];
    double s0 = 0, s1 = 0, s2 = 0;
    for (int j = lane; j < Nb; j += 32) {
        const double fx = F[3 * j], fy = F[3 * j + 1], fz = F[3 * j + 2];
        if (j == i) { s0 += fx; s1 += fy; s2 += fz; continue; }          // Eq. 7: D_ii = I
        const double dx = (xi - r[3 * j]) * inv_b, dy = (yi - r[3 * j + 1]) * inv_b, dz = (zi - r[3 * j + 2]) * inv_b;
        double cI, cRR;
        rpy_coeffs(dx * dx + dy * dy + dz * dz, hstar, a_s, inv_a, cI, cRR);
        const double dot = cRR * (dx * fx + dy * fy + dz * fz);
        s0 += cI * fx + dot * dx; s1 += cI * fy + dot * dy; s2 += cI * fz + dot * dz;
    }
    s0 = warp_sum(s0); s1 = warp_sum(s1); s2 = warp_sum(s2);
    if (lane == 0) {
        double* v = v_all + (size_t)c * 3 * Nb;
        v[3 * i] = s0; v[3 * i + 1] = s1; v[3 * i + 2] = s2;
    }
}

// -------------------------------------------------------------------------------------------------
// a6-a8.  u_i = dt (kappa r_i + v_i) + y_i                 (Eq. 6 x dt; Eq. 5 :86)
//         Y_k = Q_k + (u_{k+1} - u_k) + 2 dt T_k           (Eq. 14 :139, reading A7)
//         |Q'_k| = (2 dt K b + |Y_k|)/(2 dt K + 1)         (Eq. 17 :154)
//         Q'_k = Y_k |Q'_k| / |Y_k|                        (Eq. 15 :144, recipe :156-160)
//         r'_0 = 0, r'_{k+1} = r'_k + Q'_k, centre of mass -> 0 (reading A8)
// One CTA per chain.  A chain whose factorisation failed in THIS step (info_step != 0) or whose update is
// non-finite keeps its positions for this step (reading A10); its first failure code is kept in info_sticky.
struct UpdParams { double dt; SpringLaw sl; double kap[9]; };

__global__ void __launch_bounds__(kUpdThreads) k_update(int N, UpdParams P, const double* __restrict__ r_all,
                                                        const double* __restrict__ v_all, const double* __restrict__ y_all,
                                                        const int32_t* __restrict__ info_step, int32_t* __restrict__ info_sticky,
                                                        double* __restrict__ tmp_all, double* r_out_all)
{
    __shared__ double s_buf[96];
    const int c = blockIdx.x;
    const size_t M = 3 * (size_t)(N + 1);
    const double* r = r_all + c * M;
    const double* v = v_all + c * M;
    const double* y = y_all + c * M;
    double* r_out = r_out_all + c * M;
    bool bad = false;
    const int32_t code_in = (info_step != nullptr) ? info_step[c] : 0;       // this step's factorisation failure, if any
    const bool skip = code_in != 0;
    if (!skip) {
        rebuild_positions(N, tmp_all + c * M, r_out, s_buf, bad, [&](int k, double* q) {
            double ra[3], rb[3], Y[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) { ra[d] = r[3 * k + d]; rb[d] = r[3 * k + 3 + d]; }
            const double Qx = rb[0] - ra[0], Qy = rb[1] - ra[1], Qz = rb[2] - ra[2];
            const double qn = sqrt(Qx * Qx + Qy * Qy + Qz * Qz);
            const double tc = spring_coeff(P.sl, qn);                   // Eq. 3 (or Eq. 4)
            const double Q[3] = {Qx, Qy, Qz};
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const double fa = P.kap[3 * d] * ra[0] + P.kap[3 * d + 1] * ra[1] + P.kap[3 * d + 2] * ra[2];
                const double fb = P.kap[3 * d] * rb[0] + P.kap[3 * d + 1] * rb[1] + P.kap[3 * d + 2] * rb[2];
                const double ua = P.dt * (fa + v[3 * k + d]) + y[3 * k + d];
                const double ub = P.dt * (fb + v[3 * k + 3 + d]) + y[3 * k + 3 + d];
                Y[d] = Q[d] + (ub - ua) + 2.0 * P.dt * (tc * Q[d]);
            }
            const double Yn = sqrt(Y[0] * Y[0] + Y[1] * Y[1] + Y[2] * Y[2]);
            const double scale = implicit_length(P.sl, Yn) / Yn;        // Eq. 17, then Eq. 15
            if (!(Yn > 0.0) || !isfinite(scale)) bad = true;
            q[0] = Y[0] * scale; q[1] = Y[1] * scale; q[2] = Y[2] * scale;
        });
    }
    if (skip || bad) {
        if (r_out != r)
            for (int i = threadIdx.x; i < (int)M; i += blockDim.x) r_out[i] = r[i];
        // first failure of the chain since the last reset: failing pivot row, or M + 1 for a non-finite update
        if (threadIdx.x == 0 && info_sticky != nullptr && info_sticky[c] == 0) info_sticky[c] = skip ? code_in : (int32_t)M + 1;
    }
}

}  // namespace

int bdk_init_random_walk(bd_ctx* ctx, double* r, uint64_t init_seed)
{
    BD_LAUNCH(ctx, k_init_walk, dim3(ctx->C), dim3(kUpdThreads), 0, ctx->N, ctx->p.b, init_seed, ctx->p.chain_id0,
              ctx->tmp, r);
    return 0;
}

int bdk_drift(bd_ctx* ctx, const double* r, double* T, double* F, double* v)
{
    double* Fbuf = (F != nullptr) ? F : ctx->F;
    if (T != nullptr || F != nullptr || v != nullptr)
        BD_LAUNCH(ctx, k_forces, dim3((unsigned)((int64_t)((ctx->Nb + 255) / 256) * ctx->C)), dim3(256), 0, ctx->N, (ctx->Nb + 255) / 256,
                  make_spring_law(ctx->p), r, T, Fbuf);
    if (v != nullptr)
        BD_LAUNCH(ctx, k_drift, dim3((unsigned)((int64_t)((ctx->Nb + 7) / 8) * ctx->C)), dim3(256), 0, ctx->N, (ctx->Nb + 7) / 8, ctx->p.hstar,
                  ctx->p.a / ctx->p.b, ctx->p.b / ctx->p.a, 1.0 / ctx->p.b, r, Fbuf, v);
    return 0;
}

int bdk_update(bd_ctx* ctx, const double* r, const double* v, const double* y, const int32_t* info_step,
               int32_t* info_sticky, double* r_out)
{
    UpdParams P;
    P.dt = ctx->p.dt; P.sl = make_spring_law(ctx->p);
    for (int i = 0; i < 9; ++i) P.kap[i] = ctx->p.kappa[i];
    BD_LAUNCH(ctx, k_update, dim3(ctx->C), dim3(kUpdThreads), 0, ctx->N, P, r, v, y, info_step, info_sticky, ctx->tmp, r_out);
    return 0;
}
