// api.cu -- the C ABI of include/bd.h: argument checking and stage sequencing only; every step of
// the path runs in the kernels of assemble.cu / potrf.cu / brownian.cu / update.cu / observables.cu.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "bd_internal.cuh"

namespace {

inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

bool layout_ok(const bd_ctx* ctx, const void* p, int64_t ld, int64_t stride)
{
    return p != nullptr && ld >= ctx->M && (ld % 2) == 0 && stride >= ld * (int64_t)ctx->M && (stride % 2) == 0 &&
           (reinterpret_cast<uintptr_t>(p) % 16) == 0;
}

}  // namespace

// bd_create can fail before a context exists: its CUDA error is kept per calling thread for bd_strerror.  Every other
// CUDA error lives in the context (bd_last_error).
static thread_local cudaError_t tl_create_cuda = cudaSuccess;

// a3 dispatch: the persistent tile kernel unless its O(C M) scratch (128 x 128 inverse blocks) would be unreasonably large
int bdk_potrf(bd_ctx* ctx, double* A, int64_t ld, int64_t stride, int32_t* info)
{
    const bool tiles = (ctx->chol_algo == 2) || (ctx->chol_algo == 0 && bdk_potrf_tiles_scratch_bytes(ctx) <= ((size_t)4 << 30));
    return tiles ? bdk_potrf_tiles(ctx, A, ld, stride, info) : bdk_potrf_launches(ctx, A, ld, stride, info);
}

extern "C" {

int bd_create(const bd_params* params, void* cuda_stream, bd_ctx** out)
{
    if (params == nullptr) return -1;
    if (out == nullptr) return -3;
    *out = nullptr;
    bd_params p = *params;
    if (p.n_rods < 1 || p.n_chains < 1) return -1;
    if (!(p.b > 0.0) || !(p.hstar >= 0.0) || !(p.dt > 0.0) || !std::isfinite(p.b) || !std::isfinite(p.hstar) || !std::isfinite(p.dt))
        return -1;
    if (!(p.a > 0.0)) p.a = p.hstar * p.b;                 // reading A3: a = h* b
    if (p.hstar == 0.0 && !(p.a > 0.0)) p.a = p.b;         // free draining: a is irrelevant, keep it finite
    if (p.hstar * p.b > p.a * (1.0 + 1e-12)) return -1;    // h*/a > 1: D not guaranteed positive definite (A3)
    if (!(p.K > 0.0)) p.K = 1.0 / p.dt;                    // reading A6: K* dt = 1
    if (p.noise_kind != 0 && p.noise_kind != 1) return -1;
    if (p.spring_kind != 0 && p.spring_kind != 1) return -1;
    if (p.spring_kind == 1 && !(p.nu > 0.0 && std::isfinite(p.nu))) return -1;
    for (int i = 0; i < 9; ++i)
        if (!std::isfinite(p.kappa[i])) return -1;
    if ((int64_t)3 * ((int64_t)p.n_rods + 1) > (int64_t)1 << 20) return -1;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        tl_create_cuda = cudaGetLastError();
        return BD_ERR_CUDA;                               // no host fallback, by design
    }
    bd_ctx* ctx = new (std::nothrow) bd_ctx();
    if (ctx == nullptr) return BD_ERR_ALLOC;
    std::memset(ctx, 0, sizeof(*ctx));
    ctx->p = p;
    ctx->N = p.n_rods;
    ctx->Nb = p.n_rods + 1;
    ctx->M = 3 * ctx->Nb;
    ctx->C = p.n_chains;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->ws_ld = round_up(ctx->M, 16);
    ctx->ws_stride = ctx->ws_ld * round_up(ctx->M, 8);
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        tl_create_cuda = cudaGetLastError();
        delete ctx;
        return BD_ERR_CUDA;
    }
    ctx->num_sms = prop.multiProcessorCount;
    const size_t CM = (size_t)ctx->C * ctx->M;
    struct { void** p; size_t bytes; } allocs[] = {
        {(void**)&ctx->T, sizeof(double) * (size_t)ctx->C * 3 * ctx->N},
        {(void**)&ctx->F, sizeof(double) * CM},
        {(void**)&ctx->v, sizeof(double) * CM},
        {(void**)&ctx->y, sizeof(double) * CM},
        {(void**)&ctx->dW, sizeof(double) * CM},
        {(void**)&ctx->tmp, sizeof(double) * CM},
        {(void**)&ctx->r_own, sizeof(double) * CM},
        {(void**)&ctx->info, sizeof(int32_t) * (size_t)ctx->C},
        {(void**)&ctx->info_step, sizeof(int32_t) * (size_t)ctx->C},
        {(void**)&ctx->fail, sizeof(int32_t) * 2},
        {(void**)&ctx->obs, sizeof(double) * ((size_t)ctx->C + 2) * BD_NOBS},
        {(void**)&ctx->Winv, sizeof(double) * (size_t)ctx->C * BD_NB_INNER * BD_NB_INNER},
    };
    for (auto& al : allocs) {
        cudaError_t e = cudaMalloc(al.p, al.bytes);
        if (e != cudaSuccess) {
            tl_create_cuda = e;
            bd_destroy(ctx);
            return BD_ERR_CUDA;
        }
    }
    cudaError_t e = cudaMemsetAsync(ctx->info, 0, sizeof(int32_t) * (size_t)ctx->C, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) {
        tl_create_cuda = e;
        bd_destroy(ctx);
        return BD_ERR_CUDA;
    }
    *out = ctx;
    return 0;
}

int bd_destroy(bd_ctx* ctx)
{
    if (ctx == nullptr) return -1;
    cudaStreamSynchronize(ctx->stream);
    void* ptrs[] = {ctx->T, ctx->F, ctx->v, ctx->y, ctx->dW, ctx->tmp, ctx->r_own, ctx->info, ctx->info_step, ctx->fail, ctx->obs, ctx->Winv,
                    ctx->tile_W, ctx->tile_flags};
    for (void* q : ptrs)
        if (q != nullptr) cudaFree(q);
    if (ctx->ev != nullptr) {
        for (int i = 0; i < ctx->ev_cap_steps * (BD_NSTAGES + 1); ++i)
            if (ctx->ev[i] != nullptr) cudaEventDestroy(ctx->ev[i]);
        std::free(ctx->ev);
        std::free(ctx->ev_nsteps);
    }
    delete ctx;
    return 0;
}

size_t bd_workspace_bytes(const bd_ctx* ctx)
{
    if (ctx == nullptr) return 0;
    return sizeof(double) * (size_t)ctx->C * (size_t)ctx->ws_stride;
}

int bd_set_workspace(bd_ctx* ctx, void* ws_dev, size_t bytes)
{
    if (ctx == nullptr) return -1;
    if (ws_dev == nullptr || (reinterpret_cast<uintptr_t>(ws_dev) % 16) != 0) return -2;
    if (bytes < bd_workspace_bytes(ctx)) return -3;
    ctx->ws = static_cast<double*>(ws_dev);
    ctx->ws_bytes = bytes;
    return 0;
}

int bd_set_flow(bd_ctx* ctx, const double kappa_host[9])
{
    if (ctx == nullptr) return -1;
    if (kappa_host == nullptr) return -2;
    for (int i = 0; i < 9; ++i)
        if (!std::isfinite(kappa_host[i])) return -2;
    for (int i = 0; i < 9; ++i) ctx->p.kappa[i] = kappa_host[i];
    return 0;
}

int bd_init_random_walk(bd_ctx* ctx, double* r_dev, uint64_t init_seed)
{
    if (ctx == nullptr) return -1;
    if (r_dev == nullptr) return -2;
    return bdk_init_random_walk(ctx, r_dev, init_seed);
}

int bd_assemble_hi(bd_ctx* ctx, const double* r_dev, double* D_dev, int64_t ld, int64_t chain_stride, int32_t full)
{
    if (ctx == nullptr) return -1;
    if (r_dev == nullptr) return -2;
    if (D_dev == nullptr || (reinterpret_cast<uintptr_t>(D_dev) % 16) != 0) return -3;
    if (ld < ctx->M || (ld % 2) != 0) return -4;
    if (chain_stride < ld * (int64_t)ctx->M || (chain_stride % 2) != 0) return -5;
    return bdk_assemble(ctx, r_dev, D_dev, ld, chain_stride, full != 0);
}

int bd_cholesky(bd_ctx* ctx, double* DL_dev, int64_t ld, int64_t chain_stride, int32_t* info_dev)
{
    if (ctx == nullptr) return -1;
    if (DL_dev == nullptr || (reinterpret_cast<uintptr_t>(DL_dev) % 16) != 0) return -2;
    if (ld < ctx->M || (ld % 2) != 0) return -3;
    if (chain_stride < ld * (int64_t)ctx->M || (chain_stride % 2) != 0) return -4;
    int32_t* info = (info_dev != nullptr) ? info_dev : ctx->info;
    BD_CUDA(ctx, cudaMemsetAsync(info, 0, sizeof(int32_t) * (size_t)ctx->C, ctx->stream));
    return bdk_potrf(ctx, DL_dev, ld, chain_stride, info);
}

int bd_set_cholesky(bd_ctx* ctx, int32_t algo)
{
    if (ctx == nullptr) return -1;
    if (algo < 0 || algo > 2) return -2;
    ctx->chol_algo = algo;
    return 0;
}

int bd_noise(bd_ctx* ctx, uint64_t step, double* dW_dev)
{
    if (ctx == nullptr) return -1;
    if (dW_dev == nullptr) return -3;
    return bdk_noise(ctx, step, dW_dev);
}

int bd_brownian(bd_ctx* ctx, const double* L_dev, int64_t ld, int64_t chain_stride, uint64_t step,
                const double* dW_dev_or_null, double* y_dev)
{
    if (ctx == nullptr) return -1;
    if (!layout_ok(ctx, L_dev, ld, chain_stride)) return (L_dev == nullptr) ? -2 : ((ld < ctx->M || ld % 2) ? -3 : -4);
    if (y_dev == nullptr) return -7;
    const double* dW = dW_dev_or_null;
    if (dW == nullptr) {
        int rc = bdk_noise(ctx, step, ctx->dW);
        if (rc != 0) return rc;
        dW = ctx->dW;
    }
    return bdk_trmv(ctx, L_dev, ld, chain_stride, dW, y_dev);
}

int bd_drift(bd_ctx* ctx, const double* r_dev, double* T_dev, double* F_dev, double* v_dev)
{
    if (ctx == nullptr) return -1;
    if (r_dev == nullptr) return -2;
    return bdk_drift(ctx, r_dev, T_dev, F_dev, v_dev);
}

int bd_update(bd_ctx* ctx, const double* r_dev, const double* v_dev, const double* y_dev, double* r_out_dev)
{
    if (ctx == nullptr) return -1;
    if (r_dev == nullptr) return -2;
    if (v_dev == nullptr) return -3;
    if (y_dev == nullptr) return -4;
    if (r_out_dev == nullptr) return -5;
    return bdk_update(ctx, r_dev, v_dev, y_dev, nullptr, ctx->info, r_out_dev);   // a non-finite update is recorded in the sticky info
}

int bd_step(bd_ctx* ctx, double* r_dev, uint64_t first_step, int32_t n_steps)
{
    if (ctx == nullptr) return -1;
    if (r_dev == nullptr) return -2;
    if (n_steps < 0) return -4;
    if (ctx->ws == nullptr) return BD_ERR_WORKSPACE;
    BD_CUDA(ctx, cudaMemsetAsync(ctx->info, 0, sizeof(int32_t) * (size_t)ctx->C, ctx->stream));
    const bool fused = (ctx->path == 2) || (ctx->path == 0 && bdk_chain_step_supported(ctx));
    if (fused) {
        if (n_steps == 0) return 0;
        cudaEvent_t* ev = nullptr;
        if (ctx->prof_on && ctx->ev_steps < ctx->ev_cap_steps) {
            ctx->ev_nsteps[ctx->ev_steps] = -n_steps;                       // negative: fused record
            ev = ctx->ev + (size_t)(ctx->ev_steps++) * (BD_NSTAGES + 1);
            BD_CUDA(ctx, cudaEventRecord(ev[0], ctx->stream));
        }
        int rc = bdk_chain_step(ctx, r_dev, first_step, n_steps);          // a0-a8, all steps, one launch
        if (rc != 0) return rc;
        if (ev != nullptr) BD_CUDA(ctx, cudaEventRecord(ev[1], ctx->stream));
        return 0;
    }
    for (int32_t s = 0; s < n_steps; ++s) {
        int rc;
        cudaEvent_t* ev = nullptr;
        if (ctx->prof_on && ctx->ev_steps < ctx->ev_cap_steps) {
            ctx->ev_nsteps[ctx->ev_steps] = 1;
            ev = ctx->ev + (size_t)(ctx->ev_steps++) * (BD_NSTAGES + 1);
        }
#define BD_MARK(i) do { if (ev != nullptr) BD_CUDA(ctx, cudaEventRecord(ev[i], ctx->stream)); } while (0)
        // reading A10: a failed chain keeps its positions FOR THAT STEP and is tried again in the next one (as the fused
        // kernel and the oracle do): failures of this step go to info_step, the first failure of a chain stays in info
        BD_CUDA(ctx, cudaMemsetAsync(ctx->info_step, 0, sizeof(int32_t) * (size_t)ctx->C, ctx->stream));
        BD_MARK(0);
        if ((rc = bdk_drift(ctx, r_dev, nullptr, ctx->F, ctx->v)) != 0) return rc;                       // a1, a4
        BD_MARK(1);
        if ((rc = bdk_assemble(ctx, r_dev, ctx->ws, ctx->ws_ld, ctx->ws_stride, 0)) != 0) return rc;     // a2
        BD_MARK(2);
        if ((rc = bdk_potrf(ctx, ctx->ws, ctx->ws_ld, ctx->ws_stride, ctx->info_step)) != 0) return rc;  // a3
        BD_MARK(3);
        if ((rc = bdk_noise(ctx, first_step + (uint64_t)s, ctx->dW)) != 0) return rc;                    // a0
        BD_MARK(4);
        if ((rc = bdk_trmv(ctx, ctx->ws, ctx->ws_ld, ctx->ws_stride, ctx->dW, ctx->y)) != 0) return rc;  // a5
        BD_MARK(5);
        if ((rc = bdk_update(ctx, r_dev, ctx->v, ctx->y, ctx->info_step, ctx->info, r_dev)) != 0) return rc;  // a6-a8
        BD_MARK(6);
#undef BD_MARK
    }
    return 0;
}

int bd_set_path(bd_ctx* ctx, int32_t path)
{
    if (ctx == nullptr) return -1;
    if (path < 0 || path > 2) return -2;
    if (path == 2 && !bdk_chain_step_supported(ctx)) return -2;
    ctx->path = path;
    return 0;
}

int bd_observables(bd_ctx* ctx, const double* r_dev, double* per_chain_dev, double* ensemble_dev)
{
    if (ctx == nullptr) return -1;
    if (r_dev == nullptr) return -2;
    return bdk_observables(ctx, r_dev, per_chain_dev, ensemble_dev);
}

int bd_end_to_end(bd_ctx* ctx, const double* r_dev, double* R_dev)
{
    if (ctx == nullptr) return -1;
    if (r_dev == nullptr) return -2;
    if (R_dev == nullptr) return -3;
    return bdk_end_to_end(ctx, r_dev, R_dev);
}

int bd_autocorr(bd_ctx* ctx, const double* r_dev, const double* R0_dev, double* out_dev)
{
    if (ctx == nullptr) return -1;
    if (r_dev == nullptr) return -2;
    if (R0_dev == nullptr) return -3;
    if (out_dev == nullptr) return -4;
    return bdk_autocorr(ctx, r_dev, R0_dev, out_dev);
}

int bd_last_info(bd_ctx* ctx, int32_t* n_failed_chains, int32_t* first_failed_chain)
{
    if (ctx == nullptr) return -1;
    int rc = bdk_count_failures(ctx, ctx->info);
    if (rc != 0) return rc;
    int32_t h[2] = {0, -1};
    int32_t tile_err = 0;
    BD_CUDA(ctx, cudaMemcpyAsync(h, ctx->fail, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    if (ctx->tile_flags != nullptr)                      // error word of the tile Cholesky (after its flags and ticket counter)
        BD_CUDA(ctx, cudaMemcpyAsync(&tile_err, ctx->tile_flags + bdk_potrf_tiles_flag_words(ctx) + 1, sizeof(int32_t),
                                     cudaMemcpyDeviceToHost, ctx->stream));
    BD_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (tile_err != 0) return BD_ERR_INTERNAL;
    if (n_failed_chains != nullptr) *n_failed_chains = h[0];
    if (first_failed_chain != nullptr) *first_failed_chain = h[1];
    return 0;
}

int bd_step_host(bd_ctx* ctx, double* r_host, uint64_t first_step, int32_t n_steps, double* ensemble_host)
{
    if (ctx == nullptr) return -1;
    if (r_host == nullptr) return -2;
    const size_t bytes = sizeof(double) * (size_t)ctx->C * ctx->M;
    BD_CUDA(ctx, cudaMemcpyAsync(ctx->r_own, r_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    int rc = bd_step(ctx, ctx->r_own, first_step, n_steps);
    if (rc != 0) return rc;
    double* ens = ctx->obs + (size_t)ctx->C * BD_NOBS;
    if ((rc = bdk_observables(ctx, ctx->r_own, ctx->obs, ens)) != 0) return rc;
    BD_CUDA(ctx, cudaMemcpyAsync(r_host, ctx->r_own, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    if (ensemble_host != nullptr)
        BD_CUDA(ctx, cudaMemcpyAsync(ensemble_host, ens, sizeof(double) * 2 * BD_NOBS, cudaMemcpyDeviceToHost, ctx->stream));
    BD_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return 0;
}

int bd_profile(bd_ctx* ctx, int32_t enable)
{
    if (ctx == nullptr) return -1;
    if (enable && ctx->ev == nullptr) {
        const int cap = 1024;
        ctx->ev = static_cast<cudaEvent_t*>(std::calloc((size_t)cap * (BD_NSTAGES + 1), sizeof(cudaEvent_t)));
        if (ctx->ev == nullptr) return BD_ERR_ALLOC;
        for (int i = 0; i < cap * (BD_NSTAGES + 1); ++i) BD_CUDA(ctx, cudaEventCreate(&ctx->ev[i]));
        ctx->ev_nsteps = static_cast<int32_t*>(std::calloc((size_t)cap, sizeof(int32_t)));
        if (ctx->ev_nsteps == nullptr) return BD_ERR_ALLOC;
        ctx->ev_cap_steps = cap;
    }
    ctx->prof_on = enable ? 1 : 0;
    ctx->ev_steps = 0;
    return 0;
}

int bd_stage_ms(bd_ctx* ctx, double ms_host[BD_NSTAGES], int64_t* steps_host)
{
    if (ctx == nullptr) return -1;
    if (ms_host == nullptr) return -2;
    BD_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < BD_NSTAGES; ++i) ms_host[i] = 0.0;
    int64_t nsteps = 0;
    for (int s = 0; s < ctx->ev_steps; ++s) {
        cudaEvent_t* ev = ctx->ev + (size_t)s * (BD_NSTAGES + 1);
        if (ctx->ev_nsteps[s] < 0) {                                        // fused record: one interval
            float ms = 0.f;
            BD_CUDA(ctx, cudaEventElapsedTime(&ms, ev[0], ev[1]));
            ms_host[BD_NSTAGES - 1] += (double)ms;
            nsteps += -ctx->ev_nsteps[s];
            continue;
        }
        for (int i = 0; i < BD_NSTAGES - 1; ++i) {
            float ms = 0.f;
            BD_CUDA(ctx, cudaEventElapsedTime(&ms, ev[i], ev[i + 1]));
            ms_host[i] += (double)ms;
        }
        nsteps += 1;
    }
    if (steps_host != nullptr) *steps_host = nsteps;
    ctx->ev_steps = 0;
    return 0;
}

int64_t bd_launch_count(const bd_ctx* ctx) { return (ctx == nullptr) ? 0 : ctx->launches; }

const char* bd_last_error(const bd_ctx* ctx)
{
    if (ctx == nullptr) return "no context";
    return (ctx->last_cuda == cudaSuccess) ? "no CUDA error recorded" : cudaGetErrorString(ctx->last_cuda);
}

const char* bd_strerror(int code)
{
    switch (code) {
        case 0: return "success";
        case BD_ERR_CUDA: return (tl_create_cuda != cudaSuccess) ? cudaGetErrorString(tl_create_cuda) : "CUDA runtime error (bd_last_error(ctx) gives the text)";
        case BD_ERR_WORKSPACE: return "bd_step needs a workspace: call bd_set_workspace first";
        case BD_ERR_ALLOC: return "host allocation failed";
        case BD_ERR_TOO_LARGE: return "bd_cholesky_noalloc: n_chains * ceil(M / 128) exceeds 32 (its fixed 4 MB scratch); use bd_cholesky";
        case BD_ERR_INTERNAL: return "internal error: a dependency wait inside the tile Cholesky timed out";
        default: break;
    }
    if (code < 0 && code > -20) return "invalid argument (index = -code)";
    return "unknown error";
}

}  // extern "C"
