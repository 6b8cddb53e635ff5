// observables.cu -- a9: per-chain and ensemble observables (Eqs. 25-29).
//   0 R^2 = |r_N - r_0|^2 (Eq. 25), 1..3 its x,y,z parts (Eq. 26), 4 Rg^2 (Eq. 27),
//   5..10 S = sum_k T_k (x) Q_k: xx yy zz xy xz yz (Eq. 28 without N delta; N_1 = S_xx - S_yy, Eq. 29),
//   11 mean_k (|Q_k|-b)^2, 12 max_k ||Q_k|-b|.
// One CTA per chain with warp-shuffle reductions; the ensemble sums are reduced by a second,
// single-CTA kernel in a fixed order (deterministic, no atomics).
#include "bd_internal.cuh"

namespace {

constexpr int kObsThreads = 256;

__global__ void __launch_bounds__(kObsThreads) k_obs_chain(int N, SpringLaw sl, const double* __restrict__ r_all,
                                                           double* __restrict__ per_chain)
{
    __shared__ double s_red[kObsThreads / 32][12];
    __shared__ double s_cm[3];
    const int c = blockIdx.x, Nb = N + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double* r = r_all + (size_t)c * 3 * Nb;
    // pass 1: centre of mass
    double acc[12];
#pragma unroll
    for (int e = 0; e < 12; ++e) acc[e] = 0.0;
    for (int i = threadIdx.x; i < Nb; i += blockDim.x) { acc[0] += r[3 * i]; acc[1] += r[3 * i + 1]; acc[2] += r[3 * i + 2]; }
#pragma unroll
    for (int d = 0; d < 3; ++d) acc[d] = warp_sum(acc[d]);
    if (lane == 0) { s_red[warp][0] = acc[0]; s_red[warp][1] = acc[1]; s_red[warp][2] = acc[2]; }
    __syncthreads();
    if (threadIdx.x < 3) {
        double t = 0;
        for (int w = 0; w < kObsThreads / 32; ++w) t += s_red[w][threadIdx.x];
        s_cm[threadIdx.x] = t / (double)Nb;
    }
    __syncthreads();
    const double cx = s_cm[0], cy = s_cm[1], cz = s_cm[2];
    // pass 2: Rg^2, stress sums, rod-length deviation
    double rg = 0, sxx = 0, syy = 0, szz = 0, sxy = 0, sxz = 0, syz = 0, dev2 = 0, devmax = 0;
    for (int i = threadIdx.x; i < Nb; i += blockDim.x) {
        const double x = r[3 * i] - cx, y = r[3 * i + 1] - cy, z = r[3 * i + 2] - cz;
        rg += x * x + y * y + z * z;
        if (i < N) {
            const double qx = r[3 * i + 3] - r[3 * i], qy = r[3 * i + 4] - r[3 * i + 1], qz = r[3 * i + 5] - r[3 * i + 2];
            const double q = sqrt(qx * qx + qy * qy + qz * qz);
            const double t = spring_coeff(sl, q);                 // Eq. 3 (or Eq. 4): T = t Q
            const double b = sl.b;
            sxx += t * qx * qx; syy += t * qy * qy; szz += t * qz * qz;
            sxy += t * qx * qy; sxz += t * qx * qz; syz += t * qy * qz;
            const double dv = q - b;
            dev2 += dv * dv;
            devmax = fmax(devmax, fabs(dv));
        }
    }
    double vals[9] = {rg, sxx, syy, szz, sxy, sxz, syz, dev2, devmax};
    __syncthreads();
#pragma unroll
    for (int e = 0; e < 8; ++e) vals[e] = warp_sum(vals[e]);
    vals[8] = warp_max(vals[8]);
    if (lane == 0)
        for (int e = 0; e < 9; ++e) s_red[warp][e] = vals[e];
    __syncthreads();
    if (threadIdx.x == 0) {
        double t[9];
        for (int e = 0; e < 9; ++e) t[e] = 0.0;
        for (int w = 0; w < kObsThreads / 32; ++w) {
            for (int e = 0; e < 8; ++e) t[e] += s_red[w][e];
            t[8] = fmax(t[8], s_red[w][8]);
        }
        double* o = per_chain + (size_t)c * BD_NOBS;
        const double ex = r[3 * N] - r[0], ey = r[3 * N + 1] - r[1], ez = r[3 * N + 2] - r[2];
        o[1] = ex * ex; o[2] = ey * ey; o[3] = ez * ez;
        o[0] = o[1] + o[2] + o[3];
        o[4] = t[0] / (double)Nb;
        for (int e = 0; e < 6; ++e) o[5 + e] = t[1 + e];
        o[11] = t[7] / (double)N;
        o[12] = t[8];
    }
}

// ensemble[0][o] = sum_c per_chain[c][o], ensemble[1][o] = sum_c per_chain[c][o]^2; warp o.
__global__ void __launch_bounds__(BD_NOBS * 32) k_obs_ensemble(int C, const double* __restrict__ per_chain,
                                                               double* __restrict__ ensemble)
{
    const int o = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double s = 0, s2 = 0;
    for (int c = lane; c < C; c += 32) {
        const double x = per_chain[(size_t)c * BD_NOBS + o];
        s += x; s2 += x * x;
    }
    s = warp_sum(s); s2 = warp_sum(s2);
    if (lane == 0) { ensemble[o] = s; ensemble[BD_NOBS + o] = s2; }
}

// fail[0] = number of chains with info != 0, fail[1] = first such chain or -1
__global__ void __launch_bounds__(256) k_count_failures(int C, const int32_t* __restrict__ info, int32_t* __restrict__ fail)
{
    __shared__ int s_cnt, s_first;
    if (threadIdx.x == 0) { s_cnt = 0; s_first = 0x7fffffff; }
    __syncthreads();
    int cnt = 0, first = 0x7fffffff;
    for (int c = threadIdx.x; c < C; c += blockDim.x)
        if (info[c] != 0) { cnt += 1; first = min(first, c); }
    atomicAdd(&s_cnt, cnt);
    atomicMin(&s_first, first);
    __syncthreads();
    if (threadIdx.x == 0) { fail[0] = s_cnt; fail[1] = (s_first == 0x7fffffff) ? -1 : s_first; }
}

// End-to-end vectors R_c = r_N - r_0 (Eq. 25's vector), one thread per chain.
__global__ void __launch_bounds__(256) k_end_to_end(int N, int C, const double* __restrict__ r_all, double* __restrict__ R_all)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    const double* r = r_all + (size_t)c * 3 * (N + 1);
#pragma unroll
    for (int d = 0; d < 3; ++d) R_all[3 * (size_t)c + d] = r[3 * N + d] - r[d];
}

// Autocorrelation sums of the end-to-end vector against a stored origin R0 (the relaxation time is the
// decay time of this function): out = { sum_c R.R0, sum_c (R.R0)^2, sum_c R0.R0 }.  ONE CTA, fixed summation order
// (deterministic, no atomics): the sums are 3 doubles per sampling instant.
__global__ void __launch_bounds__(256) k_autocorr(int N, int C, const double* __restrict__ r_all, const double* __restrict__ R0_all,
                                                  double* __restrict__ out)
{
    __shared__ double s_red[8][3];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    for (int c = threadIdx.x; c < C; c += blockDim.x) {
        const double* r = r_all + (size_t)c * 3 * (N + 1);
        const double* R0 = R0_all + 3 * (size_t)c;
        double dot = 0.0, n0 = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double Rd = r[3 * N + d] - r[d];
            dot += Rd * R0[d];
            n0 += R0[d] * R0[d];
        }
        a0 += dot; a1 += dot * dot; a2 += n0;
    }
    a0 = warp_sum(a0); a1 = warp_sum(a1); a2 = warp_sum(a2);
    if (lane == 0) { s_red[warp][0] = a0; s_red[warp][1] = a1; s_red[warp][2] = a2; }
    __syncthreads();
    if (threadIdx.x < 3) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += s_red[w][threadIdx.x];
        out[threadIdx.x] = t;
    }
}

}  // namespace

int bdk_end_to_end(bd_ctx* ctx, const double* r, double* R)
{
    BD_LAUNCH(ctx, k_end_to_end, dim3((ctx->C + 255) / 256), dim3(256), 0, ctx->N, ctx->C, r, R);
    return 0;
}

int bdk_autocorr(bd_ctx* ctx, const double* r, const double* R0, double* out)
{
    BD_LAUNCH(ctx, k_autocorr, dim3(1), dim3(256), 0, ctx->N, ctx->C, r, R0, out);
    return 0;
}

int bdk_observables(bd_ctx* ctx, const double* r, double* per_chain, double* ensemble)
{
    double* pc = (per_chain != nullptr) ? per_chain : ctx->obs;
    BD_LAUNCH(ctx, k_obs_chain, dim3(ctx->C), dim3(kObsThreads), 0, ctx->N, make_spring_law(ctx->p), r, pc);
    if (ensemble != nullptr) BD_LAUNCH(ctx, k_obs_ensemble, dim3(1), dim3(BD_NOBS * 32), 0, ctx->C, pc, ensemble);
    return 0;
}

int bdk_count_failures(bd_ctx* ctx, const int32_t* info)
{
    BD_LAUNCH(ctx, k_count_failures, dim3(1), dim3(256), 0, ctx->C, info, ctx->fail);
    return 0;
}
