// bd_internal.cuh -- context, launch helpers and small device utilities shared by the libbd kernels.
// (Nothing here is shared with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/bd.h"

struct bd_ctx {
    bd_params p;            // resolved parameters (a, K filled in)
    int32_t N, Nb, M, C;
    cudaStream_t stream;
    int64_t ws_ld;          // leading dimension used by bd_step's own storage
    int64_t ws_stride;      // doubles between chains in the workspace
    double* ws;             // caller-owned D/L storage (bd_set_workspace)
    size_t ws_bytes;
    // O(C*M) scratch, library-owned
    double* T;              // [C][N][3]
    double* F;              // [C][Nb][3]
    double* v;              // [C][M]
    double* y;              // [C][M]
    double* dW;             // [C][M]
    double* Winv;           // [C][NB_INNER*NB_INNER] inverse of the current diagonal block
    int32_t* info;          // [C] sticky: first failure of every chain since the last reset (bd_last_info)
    int32_t* info_step;     // [C] failures of the current time step only (staged bd_step; reading A10: a chain is retried every step)
    int32_t* fail;          // [2]: count, first chain
    double* obs;            // [C][BD_NOBS] + [2][BD_NOBS]
    double* tmp;            // [C][M] unshifted positions inside the update / init kernels
    double* r_own;          // [C][M] device positions for bd_step_host
    int64_t launches;
    // stage timing (bd_profile): (BD_NSTAGES+1) events per profiled step
    cudaEvent_t* ev;
    int32_t ev_cap_steps, ev_steps, prof_on;
    int32_t* ev_nsteps;     // time steps covered by each profiled record
    int32_t path;           // bd_set_path
    cudaError_t last_cuda;
    int num_sms;
    bool attr_potrf, attr_chain;   // cudaFuncSetAttribute done for this context's device (no process-wide statics)
    // tile Cholesky (potrf_tiles.cu): inverse diagonal blocks, ready flags (+ ticket counter, error word), tensor maps
    int32_t chol_algo;             // bd_set_cholesky: 0 auto, 1 multi-launch recursive (potrf.cu), 2 persistent tile kernel
    double* tile_W;
    int* tile_flags;
    int tile_epoch;
    unsigned tile_ticket_base;
    const void* tile_mapA_ptr;
    int64_t tile_mapA_ld, tile_mapA_stride;
    struct alignas(64) { unsigned char bytes[128]; } tile_maps[2];
};

#define BD_NB_INNER 64      // width of the diagonal block factored by potf2 (one CTA per chain)

#define BD_CUDA(ctx, call)                                  \
    do {                                                    \
        cudaError_t e__ = (call);                           \
        if (e__ != cudaSuccess) {                           \
            (ctx)->last_cuda = e__;                         \
            return BD_ERR_CUDA;                             \
        }                                                   \
    } while (0)

// every kernel launch goes through this so that bd_launch_count is exact
#define BD_LAUNCH(ctx, kernel, grid, block, smem, ...)                          \
    do {                                                                        \
        kernel<<<(grid), (block), (smem), (ctx)->stream>>>(__VA_ARGS__);        \
        (ctx)->launches += 1;                                                   \
        cudaError_t e__ = cudaGetLastError();                                   \
        if (e__ != cudaSuccess) {                                               \
            (ctx)->last_cuda = e__;                                             \
            return BD_ERR_CUDA;                                                 \
        }                                                                       \
    } while (0)

// ---- stage entry points implemented in the .cu files (host side) -------------------------------
int bdk_init_random_walk(bd_ctx* ctx, double* r, uint64_t init_seed);
int bdk_assemble(bd_ctx* ctx, const double* r, double* D, int64_t ld, int64_t stride, int full);
int bdk_potrf(bd_ctx* ctx, double* A, int64_t ld, int64_t stride, int32_t* info);            // dispatch on chol_algo
int bdk_potrf_launches(bd_ctx* ctx, double* A, int64_t ld, int64_t stride, int32_t* info);   // potrf.cu
int bdk_potrf_tiles(bd_ctx* ctx, double* A, int64_t ld, int64_t stride, int32_t* info);      // potrf_tiles.cu
size_t bdk_potrf_tiles_scratch_bytes(const bd_ctx* ctx);
size_t bdk_potrf_tiles_flag_words(const bd_ctx* ctx);      // ready flags [C][T][T]; then the ticket counter and the error word
int bdk_noise(bd_ctx* ctx, uint64_t step, double* dW);
int bdk_trmv(bd_ctx* ctx, const double* L, int64_t ld, int64_t stride, const double* dW, double* y);
int bdk_drift(bd_ctx* ctx, const double* r, double* T, double* F, double* v);
int bdk_update(bd_ctx* ctx, const double* r, const double* v, const double* y, const int32_t* info_step,
               int32_t* info_sticky, double* r_out);
int bdk_observables(bd_ctx* ctx, const double* r, double* per_chain, double* ensemble);
int bdk_end_to_end(bd_ctx* ctx, const double* r, double* R);
int bdk_autocorr(bd_ctx* ctx, const double* r, const double* R0, double* out);
int bdk_count_failures(bd_ctx* ctx, const int32_t* info);
bool bdk_chain_step_supported(const bd_ctx* ctx);
int bdk_chain_step(bd_ctx* ctx, double* r, uint64_t first_step, int n_steps);

// ---- device helpers ------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}
__device__ __forceinline__ double warp_max(double x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(0xffffffffu, x, o));
    return x;
}

// Spring law of the connectors (a1, a7).  kind 0: Fraenkel rod, T = K (|Q| - b)/|Q| Q (Eq. 3);
// kind 1: Cohen-Pade spring, |T| = (3 x - x^3)/(1 - x^2) / b with x = |Q| / (nu b) (Eq. 4, :78-82, alpha = 3, beta = 1;
// DESIGN.md reading B4 for the units).
struct SpringLaw {
    int kind;
    double K, b, dt;
    double inv_L, L, inv_b, c;       // kind 1: L = nu b (full extension), c = 2 dt / (nu b^2)
};
inline SpringLaw make_spring_law(const bd_params& p)
{
    SpringLaw s;
    s.kind = p.spring_kind; s.K = p.K; s.b = p.b; s.dt = p.dt;
    s.L = (p.spring_kind == 1) ? p.nu * p.b : 1.0;
    s.inv_L = 1.0 / s.L; s.inv_b = 1.0 / p.b;
    s.c = (p.spring_kind == 1) ? 2.0 * p.dt / (p.nu * p.b * p.b) : 0.0;
    return s;
}
// tension = spring_coeff(q) * Q, q = |Q|
__device__ __forceinline__ double spring_coeff(const SpringLaw& s, double q)
{
    if (s.kind == 1) {
        const double x = q * s.inv_L;
        return ((3.0 * x - x * x * x) / (1.0 - x * x)) * s.inv_b / q;
    }
    return s.K * (q - s.b) / q;
}
// semi-implicit link length |Q'| from |Y|: Eq. 17 (:154) for the rod; for the Cohen-Pade spring the root in [0, 1) of
// (1 + c) x^3 - y x^2 - (1 + 3c) x + y = 0 (Eq. 13 written with Eq. 4; f(0) = y >= 0, f(1) = -2c < 0), bracketed by
// bisection and finished by Newton steps that are kept inside the bracket.
__device__ __forceinline__ double implicit_length(const SpringLaw& s, double Yn)
{
    if (s.kind == 1) {
        const double y = Yn * s.inv_L, c = s.c;
        double lo = 0.0, hi = 1.0;
        auto f = [&](double x) { return ((1.0 + c) * x - y) * x * x - (1.0 + 3.0 * c) * x + y; };
        for (int it = 0; it < 40; ++it) {
            const double x = 0.5 * (lo + hi);
            if (f(x) > 0.0) lo = x; else hi = x;
        }
        double x = 0.5 * (lo + hi);
        for (int it = 0; it < 3; ++it) {
            const double df = (3.0 * (1.0 + c) * x - 2.0 * y) * x - (1.0 + 3.0 * c);
            const double xn = x - f(x) / df;
            if (xn > lo && xn < hi) x = xn;
        }
        return x * s.L;
    }
    const double tdk = 2.0 * s.dt * s.K;
    return (tdk * s.b + Yn) / (tdk + 1.0);
}

// RPY off-diagonal block coefficients (Eqs. 8-9): block = cI*I + cRR*Rv Rv^T with
// Rv = (r_i - r_j)/b, a_s = a/b, inv_a = 1/a_s.  One rsqrt, no divisions: 1/R = rsqrt(R^2).
__device__ __forceinline__ void rpy_coeffs(double R2, double hstar, double a_s, double inv_a, double& cI, double& cRR)
{
    if (R2 >= 4.0 * a_s * a_s) {                                   // Eq. 8, R >= 2a
        double iR = rsqrt(R2);
        double iR2 = iR * iR;
        double pre = 0.75 * hstar * iR;
        double a2 = a_s * a_s * iR2;
        cI = pre * (1.0 + (2.0 / 3.0) * a2);
        cRR = pre * (1.0 - 2.0 * a2) * iR2;
    } else {                                                       // Eq. 9, R < 2a (finite at R -> 0)
        double pre = 0.375 * hstar * inv_a;
        double iR = (R2 > 0.0) ? rsqrt(R2) : 0.0;
        double R = R2 * iR;
        cI = pre * (8.0 / 3.0 - 0.75 * R * inv_a);
        cRR = pre * 0.25 * iR * inv_a;
    }
}
