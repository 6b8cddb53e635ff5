/*
 * bd.h -- C ABI of libbd: the per-timestep hot path of bead-rod Brownian dynamics with
 * hydrodynamic interactions (arXiv 2208.06559; citations are /root/reference/PAPER.md lines),
 * hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 *   assemble RPY tensor D (Eqs. 7-9, :106-112)  ->  Cholesky D = L L^T (Eq. 10, :116-118)
 *   -> correlated Brownian displacement y = L dW (Eq. 6, :102)
 *   -> semi-implicit Fraenkel-rod update (Eqs. 14, 17, 15, :139-160) -> observables (Eqs. 25-29)
 * batched over an ensemble of C independent chains (the paper runs one chain per MPI rank, :166).
 *
 * Conventions
 *   - Plain C types only.  Every pointer named *_dev is a CUDA DEVICE pointer owned by the CALLER
 *     (e.g. a torch tensor); *_host pointers are host memory.  The library allocates only O(C*M)
 *     scratch at bd_create; the O(C*M^2) matrix storage is the caller's (bd_set_workspace).
 *   - N = n_rods, N_b = N+1 beads, M = 3*N_b.  Positions r[c][i][xyz]: contiguous doubles,
 *     chain-major; row/column index of D for bead i, component k is 3i+k (Eqs. 18-19, :214-223).
 *   - D / L per chain: ROW-major, leading dimension ld >= M doubles with ld % 2 == 0, chains
 *     chain_stride >= ld*M doubles apart (chain_stride % 2 == 0), base 16-byte aligned.  Only the
 *     LOWER triangle (col <= row) is written by bd_assemble_hi (unless full != 0) and by
 *     bd_cholesky; the strict upper triangle is never read.
 *   - All calls are asynchronous on the stream given at bd_create, except bd_create, bd_destroy,
 *     bd_last_info and the *_host entry points, which synchronise that stream.
 *   - Return value: 0 success; -k = k-th argument invalid (nothing launched); other negative values
 *     are BD_ERR_* below.  Numerical failures (non-positive pivot, non-finite update; the paper's
 *     model has no excluded volume, so coincident beads can make D singular) never abort: they are
 *     recorded per chain in info (1-based failing pivot row, or M+1 for a non-finite update; 0 = ok),
 *     the failed chain's positions are left unchanged for that step, and bd_last_info reports them.
 *   - No host fallback exists anywhere: without a CUDA device every compute call fails with
 *     BD_ERR_CUDA.
 */
#ifndef BD_H
#define BD_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BD_NOBS 13          /* observables per chain, see bd_observables */

#define BD_ERR_CUDA      (-100)   /* a CUDA runtime call failed; bd_strerror gives the text */
#define BD_ERR_WORKSPACE (-101)   /* bd_step needs a workspace: call bd_set_workspace first  */
#define BD_ERR_ALLOC     (-102)
#define BD_ERR_TOO_LARGE (-104)   /* bd_cholesky_noalloc: problem beyond its fixed scratch (see there)           */
#define BD_ERR_INTERNAL  (-103)   /* bd_last_info: a dependency wait inside the tile Cholesky timed out (a bug, not a
                                     numerical failure); results of that call are undefined                  */

typedef struct bd_ctx bd_ctx;     /* opaque; one context per stream */

typedef struct {
    int32_t  n_rods;       /* N >= 1                                                              */
    int32_t  n_chains;     /* C >= 1 (ensemble size on this device)                               */
    double   b;            /* rod / Kuhn length (paper: 1, lengths scaled by b_k; Eq. 3, :76)     */
    double   hstar;        /* h* >= 0; 0 = free draining, D = I (:108-114)                        */
    double   a;            /* bead radius (same unit as r); <= 0 means a = hstar*b (paper pairs
                              h* = a* = 0.5, :305).  hstar*b/a > 1 is rejected (D may be non-PD)  */
    double   K;            /* Fraenkel stiffness K* (:76); <= 0 means K = 1/dt (paper pairs
                              (dt,K*) = (1e-3,1e3), (1e-4,1e4), :305)                              */
    double   dt;           /* time step > 0                                                       */
    double   kappa[9];     /* row-major kappa, flow velocity = kappa . r (Eq. 5, :86-98)          */
    uint64_t seed;         /* Philox4x32-10 key                                                   */
    uint64_t chain_id0;    /* global id of local chain 0 (noise/initial-walk counters use
                              chain_id0 + c, so an ensemble sharded over GPUs is reproducible)    */
    int32_t  noise_kind;   /* 0: Gaussian, dW = sqrt(2 dt) g (Philox + Box-Muller);
                              1: the paper's uniform law, dW = sqrt(6 dt) n, n in [-1,1] (Eq. 2)  */
    int32_t  spring_kind;  /* 0: Fraenkel rod, Eq. 3 (the bead-rod chain of the paper);
                              1: Cohen-Pade spring, Eq. 4 with alpha = 3, beta = 1 (:78-82), the
                              bead-spring comparison model (:305-307); K is then unused             */
    double   nu;           /* Kuhn steps per spring (Eq. 4: fractional extension |Q| / (nu b));
                              > 0 required when spring_kind = 1                                    */
} bd_params;

/* Create a context bound to cuda_stream (a cudaStream_t passed as void*, NULL = default stream).
 * Validates params (-1), allocates O(C*M) device scratch.                                        */
int bd_create(const bd_params *params, void *cuda_stream, bd_ctx **out);
int bd_destroy(bd_ctx *ctx);

/* Bytes of matrix storage bd_step needs: C * ld * (M rounded up to 8) * 8, ld = M rounded up to 16. */
size_t bd_workspace_bytes(const bd_ctx *ctx);
/* Hand the context a caller-owned device buffer of at least bd_workspace_bytes (-2 if too small
 * or misaligned).  The buffer must outlive every later bd_step.                                  */
int bd_set_workspace(bd_ctx *ctx, void *ws_dev, size_t bytes);

/* Replace kappa (startup of flow).  Takes effect for calls enqueued afterwards.                  */
int bd_set_flow(bd_ctx *ctx, const double kappa_host[9]);

/* Freely-jointed random-walk start, centre of mass at 0 (the paper's "different initial
 * configurations", :166, :258; reading A13).  r_dev: [C][N_b][3].                      */
int bd_init_random_walk(bd_ctx *ctx, double *r_dev, uint64_t init_seed);

/* a2: D_ii = I (Eq. 7), D_ij by Eq. 8 (R >= 2a) / Eq. 9 (R < 2a) for every bead pair.
 * Writes the lower triangle of D (all of D when full != 0).                                      */
int bd_assemble_hi(bd_ctx *ctx, const double *r_dev, double *D_dev, int64_t ld, int64_t chain_stride,
                   int32_t full);

/* a3: in-place Cholesky of the lower triangle, D = L L^T, L lower with positive diagonal (Eq. 10).
 * info_dev: [C] int32, may be NULL (then the context's own array is used, see bd_last_info).     */
int bd_cholesky(bd_ctx *ctx, double *DL_dev, int64_t ld, int64_t chain_stride, int32_t *info_dev);

/* a0 + a5: y = L dW (Eq. 6, third term), y_dev: [C][M].  If dW_dev_or_null is NULL the increments
 * of time step `step` are generated in the kernel (Philox counter (pair, chain, step)); otherwise
 * dW is read from dW_dev_or_null [C][M].                                                         */
int bd_brownian(bd_ctx *ctx, const double *L_dev, int64_t ld, int64_t chain_stride, uint64_t step,
                const double *dW_dev_or_null, double *y_dev);

/* a3 WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops,
 * harnesses that forbid it): the same tile Cholesky as bd_cholesky, with its scratch (inverse diagonal blocks, ready
 * flags, ticket counter) in a fixed file-scope device array of 4 MB + 4.2 KB that every GPU that loads the library
 * holds until exit.  No context: DL_dev [n_chains] matrices of order M, layout as for bd_cholesky (row-major, ld >= M
 * even, chain_stride >= ld*M even, base 16-byte aligned, lower triangle in and out); info_dev [n_chains] int32 or NULL
 * (cleared, then 1-based failing pivot row per chain); cuda_stream a cudaStream_t (NULL = default stream); the device
 * current at the call is used.  Asynchronous on that stream.  The call itself issues no cudaMalloc / cudaFree; its first
 * call on a device looks up the array's address (cudaGetSymbolAddress).
 * LIMIT: n_chains * ceil(M / 128) <= 32 (one chain of M <= 4096, 2 of M <= 2048, 8 of M <= 512, 32 of M <= 128);
 * beyond it BD_ERR_TOO_LARGE and nothing is launched.  Returns -k for the k-th invalid argument.
 * ALL calls share the one array: calls that overlap on the GPU (different streams or host threads) race and give
 * undefined results -- serialise them.  It keeps the last call's contents; what must start at zero is cleared on the
 * stream at the start of each call.                                                                              */
int bd_cholesky_noalloc(double *DL_dev, int32_t M, int32_t n_chains, int64_t ld, int64_t chain_stride,
                        int32_t *info_dev, void *cuda_stream);

/* The Brownian increments alone: dW_dev [C][M] for time step `step`.                             */
int bd_noise(bd_ctx *ctx, uint64_t step, double *dW_dev);

/* a1 + a4: spring tensions T [C][N][3] (Eq. 3), net bead forces F [C][N_b][3] (Eq. 1 / Eq. 22) and
 * the HI drift v = D F [C][M] (Eq. 6, second term; blocks recomputed from positions, D is not
 * read).  Any output pointer may be NULL.                                                        */
int bd_drift(bd_ctx *ctx, const double *r_dev, double *T_dev, double *F_dev, double *v_dev);

/* a6-a8 from given v = D F and y = L dW: r_out = updated positions (may alias r_dev).            */
int bd_update(bd_ctx *ctx, const double *r_dev, const double *v_dev, const double *y_dev,
              double *r_out_dev);

/* Which kernels bd_step uses.  0 (default): automatic -- the fused per-chain kernel (one persistent CTA
 * per chain, D never stored, M <= 320) when the chain is short enough, else the staged kernels
 * (assemble / blocked Cholesky / L dW / update) that the stage entry points above expose.
 * 1: always staged.  2: always fused (-2 if M is too large).                                        */
int bd_set_path(bd_ctx *ctx, int32_t path);

/* Which factorisation bd_cholesky / the staged bd_step use.  0 (default): automatic; 1: blocked right-looking
 * factorisation with a recursive panel, one kernel launch per block operation (k_potf2 / k_trsm / k_syrk);
 * 2: left-looking tile Cholesky in ONE persistent kernel (TMA-fed DMMA tiles, ticket counter, ready flags).
 * Both give the same L up to rounding.                                                               */
int bd_set_cholesky(bd_ctx *ctx, int32_t algo);

/* The whole hot path a0-a8, n_steps times, time steps first_step .. first_step+n_steps-1;
 * r_dev [C][N_b][3] updated in place.  Needs bd_set_workspace.                                   */
int bd_step(bd_ctx *ctx, double *r_dev, uint64_t first_step, int32_t n_steps);

/* a9: per-chain observables per_chain_dev [C][BD_NOBS] and ensemble sums ensemble_dev [2][BD_NOBS]
 * (row 0: sum over chains, row 1: sum of squares).  Index: 0 R^2=|r_N-r_0|^2 (Eq. 25), 1..3 its
 * x,y,z parts (Eq. 26), 4 Rg^2 (Eq. 27), 5..10 S_xx S_yy S_zz S_xy S_xz S_yz with
 * S = sum_k T_k (x) Q_k (Eq. 28 without N delta), 11 mean_k(|Q_k|-b)^2, 12 max_k||Q_k|-b|.
 * Either output may be NULL.                                                                     */
int bd_observables(bd_ctx *ctx, const double *r_dev, double *per_chain_dev, double *ensemble_dev);

/* Relaxation-time observable ("the time scale of the decay of the autocorrelation function of the
 * end-to-end vector", fitted over its last 70 %).  bd_end_to_end writes R_dev [C][3] = r_N - r_0 (the origin R(0) of a
 * run); bd_autocorr writes out_dev[3] = { sum_c R.R0, sum_c (R.R0)^2, sum_c R0.R0 } for the current positions, so that
 * C(t) = out[0] / out[2] and its standard error follow on the host (reading B3: ensemble average at lag t).  */
int bd_end_to_end(bd_ctx *ctx, const double *r_dev, double *R_dev);
int bd_autocorr(bd_ctx *ctx, const double *r_dev, const double *R0_dev, double *out_dev);

/* Synchronises the stream; number of chains whose info != 0 since the last call that reset it
 * (bd_step / bd_cholesky with info_dev == NULL reset at entry), and the first such chain (-1).   */
int bd_last_info(bd_ctx *ctx, int32_t *n_failed_chains, int32_t *first_failed_chain);

/* Convenience for callers without device buffers (bench.py's end-to-end leg): copies r_host
 * [C][N_b][3] to the device, runs bd_step, computes observables, copies positions and the
 * ensemble sums back; synchronises.  ensemble_host [2][BD_NOBS] may be NULL.                     */
int bd_step_host(bd_ctx *ctx, double *r_host, uint64_t first_step, int32_t n_steps,
                 double *ensemble_host);

/* Stage timing for bench.py's roofline object.  bd_profile(ctx, 1) makes every later bd_step bracket
 * its stages with CUDA events on the context's stream (first 1024 steps after enabling);
 * bd_stage_ms synchronises, returns the accumulated milliseconds per stage
 * [0 forces+drift a1/a4, 1 assemble a2, 2 cholesky a3, 3 noise a0, 4 L dW a5, 5 update a6-a8,
 * 6 the fused per-chain kernel (all of a0-a8) when that path is active] and the number of bd_step
 * time steps they cover, and resets the accumulators.                                             */
#define BD_NSTAGES 7
int bd_profile(bd_ctx *ctx, int32_t enable);
int bd_stage_ms(bd_ctx *ctx, double ms_host[BD_NSTAGES], int64_t *steps_host);

/* Number of kernel launches issued through this context so far (for bench.py's gpu_launches).   */
int64_t bd_launch_count(const bd_ctx *ctx);

/* Text for a return code.  For BD_ERR_CUDA raised by bd_create (no context yet) the CUDA error text of the calling
 * thread's last failed bd_create; for BD_ERR_CUDA from any other call use bd_last_error.                            */
const char *bd_strerror(int code);

/* Text of the last CUDA error recorded in this context (errors are per context; the library keeps no
 * process-wide state).                                                                                */
const char *bd_last_error(const bd_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
