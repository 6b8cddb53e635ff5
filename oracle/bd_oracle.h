/*
 * bd_oracle.h -- CPU ORACLE (test infrastructure, NOT the product path).
 *
 * Plain, slow, double-precision restatement of the per-timestep hot path of
 * bead-rod Brownian dynamics with hydrodynamic interactions, written from
 * /root/reference/PAPER.md (arXiv 2208.06559) equation by equation.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * constant generator with the CUDA library (include/bd.h,
 * paper_2208_06559_b200/csrc/).
 *
 * Notation (zero based): N rods, N_b = N+1 beads, M = 3*N_b.
 *   r[i][xyz]     bead positions, contiguous doubles, i = 0..N
 *   Q_k           = r_{k+1} - r_k               (link vector, k = 0..N-1)
 *   T_k           tension of spring k           (paper's F^S_i, Eq. 3)
 *   F_j           net spring force on bead j    (Eq. 1 / Eq. 22)
 *   D             M x M diffusion tensor, row-major, row 3i+k, col 3j+l (Eqs. 18-19)
 *   L  (= sigma)  lower Cholesky factor, D = L L^T (Eq. 10)
 *
 * Parity pins: every function below is pinned by tests/test_oracle_*.py
 * (closed forms, known-answer vectors, invariants, LAPACK special cases, brute
 * force).  No function here is "parity unpinned".
 */
#ifndef BD_ORACLE_H
#define BD_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_NOBS 13

typedef struct {
    int32_t  n_rods;      /* N >= 1 */
    double   b;           /* rod (Kuhn) length; paper: 1 (Eq. 3)            */
    double   hstar;       /* h*                                        */
    double   a;           /* bead radius, same length unit as r           */
    double   K;           /* Fraenkel stiffness K*                          */
    double   dt;          /* time step                                    */
    double   kappa[9];    /* row-major, v = kappa . r (Eq. 5)            */
    uint64_t seed;        /* Philox key                                                  */
    int32_t  noise_kind;  /* 0 Gaussian sqrt(2dt) g ; 1 uniform sqrt(6dt) n (Eq. 2)      */
    int32_t  spring_kind; /* 0 Fraenkel rod (Eq. 3) ; 1 Cohen-Pade spring (Eq. 4)        */
    double   nu;          /* Kuhn steps per spring (Eq. 4: r^ = |Q| / (nu b)); kind 1    */
} orc_params;

/* optional per-step intermediates; any pointer may be NULL */
typedef struct {
    double *T;   /* [N][3]   */
    double *F;   /* [N_b][3] */
    double *D;   /* [M][M]   */
    double *L;   /* [M][M] (strict upper = 0) */
    double *dW;  /* [M] */
    double *v;   /* [M]  D.F  */
    double *y;   /* [M]  L.dW */
    double *u;   /* [M]  explicit displacement */
    double *Y;   /* [N][3] Eq. 14 */
} orc_trace;

/* --- noise (BASELINE.json north_star: Philox4x32-10 + Box-Muller) ------------------------ */
void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_u01(uint64_t x);
void   orc_noise_counter(uint32_t p, uint64_t chain, uint64_t step, uint32_t purpose, uint32_t ctr[4]);
void   orc_normals(uint64_t seed, uint64_t chain, uint64_t step, int32_t M, double *g);
void   orc_uniforms_pm1(uint64_t seed, uint64_t chain, uint64_t step, int32_t M, double *n);
void   orc_noise_dW(const orc_params *p, uint64_t chain, uint64_t step, double *dW);

/* --- initial conformation (freely jointed random walk) ---------------------------------- */
void   orc_init_random_walk(int32_t n_rods, double b, uint64_t init_seed, uint64_t chain, double *r);

/* --- forces ------------------------------------------------------------------------------ */
/* spring law: T = orc_spring_coeff(p, |Q|) * Q  (Eq. 3, or Eq. 4 with alpha = 3, beta = 1)      */
double orc_spring_coeff(const orc_params *p, double q);
/* semi-implicit link length |Q'| from |Y| (Eq. 17 for the Fraenkel rod; for the Cohen-Pade spring
 * the root in [0, nu b) of Eq. 13 written with Eq. 4 -- a cubic, reading B4)          */
double orc_implicit_length(const orc_params *p, double Yn);
void   orc_spring_tensions(const orc_params *p, const double *r, double *T);
void   orc_bead_forces(int32_t n_rods, const double *T, double *F);

/* --- HI tensor ---------------------------------------------------------------------------- */
void   orc_rpy_block(const orc_params *p, const double *ri, const double *rj, double B[9]);
void   orc_assemble(const orc_params *p, const double *r, double *D /* [M][M] */);

/* --- Cholesky ---------------------------------------------------------------------------- */
int32_t orc_cholesky(int32_t M, const double *A, double *L);

/* --- matvecs ------------------------------------------------------------------------------ */
void   orc_symv(int32_t M, const double *D, const double *x, double *v);
void   orc_trmv_lower(int32_t M, const double *L, const double *x, double *y);
void   orc_drift_onthefly(const orc_params *p, const double *r, const double *F, double *v);

/* --- update ------------------------------------------------------------------------------- */
int32_t orc_finish_step(const orc_params *p, const double *r, const double *T, const double *v,
                        const double *y, double *r_out, double *u_out, double *Y_out);

/* one chain, one step.  returns info: 0 ok, k>0 non-positive pivot at row k (1-based),
 * M+1 non-finite update.  On failure r_out = r_in.                                        */
int32_t orc_step(const orc_params *p, uint64_t chain, uint64_t step, const double *r_in,
                 double *r_out, orc_trace *tr);

/* C chains [chain0, chain0+C), n_steps steps from first_step, r updated in place,
 * info[C] sticky first failure.  OpenMP over chains only.  returns #failed chains.        */
int32_t orc_step_ensemble(const orc_params *p, int32_t C, uint64_t chain0, uint64_t first_step,
                          int32_t n_steps, double *r, int32_t *info);

/* --- observables -------------------------------------------------------------------------- */
void   orc_observables_chain(const orc_params *p, const double *r, double obs[ORC_NOBS]);
void   orc_observables(const orc_params *p, int32_t C, const double *r,
                       double *per_chain /* [C][ORC_NOBS] */, double *ensemble /* [2][ORC_NOBS] */);

/* end-to-end vectors R[C][3] = r_N - r_0 and their autocorrelation sums against R0:
 * out = { sum_c R.R0, sum_c (R.R0)^2, sum_c R0.R0 }                                           */
void   orc_end_to_end(int32_t n_rods, int32_t C, const double *r, double *R);
void   orc_autocorr(int32_t n_rods, int32_t C, const double *r, const double *R0, double out[3]);

int32_t orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
