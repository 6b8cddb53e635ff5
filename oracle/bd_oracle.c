/*
 * bd_oracle.c -- CPU ORACLE (test infrastructure, NOT the product path).
 *
 * Straight loops, FP64, round-to-nearest, no FMA contraction
 * (build: gcc -O2 -ffp-contract=off -fopenmp; see oracle/__init__.py).
 * Every function cites the passage of /root/reference/PAPER.md it restates, or
 * the DESIGN.md reading (A1..A20) it takes where the paper is silent.
 * OpenMP is used ONLY to run independent chains side by side
 * (orc_step_ensemble, orc_observables): no blocking, fusion or reordering of
 * the arithmetic of a chain.
 *
 * Shares nothing with paper_2208_06559_b200/csrc/.
 */
#include "bd_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---------------------------------------------------------------------------------------
 * Noise: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) -- fixed by BASELINE.json
 * north_star ("Philox4x32-10 + Box-Muller"); replaces the paper's cuRAND uniform stream
 * (PAPER.md:258).  DESIGN.md reading A5.
 * ------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;   /* key schedule: bump after every round */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 64 random bits -> u in (0,1): u = (2*(x>>12)+1) * 2^-53, exactly representable,
 * never 0 or 1.                                          */
double orc_u01(uint64_t x)
{
    uint64_t k = x >> 12;                              /* 52 bits */
    return (double)(2u * k + 1u) * 0x1.0p-53;
}

/* counter = (p, chain, step_lo32, step_hi28 | purpose<<28); purpose 0 noise, 1 init. */
void orc_noise_counter(uint32_t pidx, uint64_t chain, uint64_t step, uint32_t purpose, uint32_t ctr[4])
{
    ctr[0] = pidx;
    ctr[1] = (uint32_t)chain;
    ctr[2] = (uint32_t)(step & 0xFFFFFFFFu);
    ctr[3] = (uint32_t)((step >> 32) & 0x0FFFFFFFu) | (purpose << 28);
}

static void philox_pair(uint64_t seed, uint32_t pidx, uint64_t chain, uint64_t step, uint32_t purpose,
                        double *u1, double *u2)
{
    uint32_t ctr[4], key[2], w[4];
    orc_noise_counter(pidx, chain, step, purpose, ctr);
    key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
    key[1] = (uint32_t)(seed >> 32);
    orc_philox4x32_10(ctr, key, w);
    uint64_t x1 = ((uint64_t)w[1] << 32) | (uint64_t)w[0];
    uint64_t x2 = ((uint64_t)w[3] << 32) | (uint64_t)w[2];
    *u1 = orc_u01(x1);
    *u2 = orc_u01(x2);
}

/* M standard normals of (chain, step): Box-Muller on pair p = floor(m/2):
 * rho = sqrt(-2 log u1), theta = 2 pi u2, g_{2p} = rho cos theta, g_{2p+1} = rho sin theta. */
void orc_normals(uint64_t seed, uint64_t chain, uint64_t step, int32_t M, double *g)
{
    for (int32_t pidx = 0; 2 * pidx < M; ++pidx) {
        double u1, u2;
        philox_pair(seed, (uint32_t)pidx, chain, step, 0u, &u1, &u2);
        double rho = sqrt(-2.0 * log(u1));
        double theta = 6.283185307179586 * u2;
        g[2 * pidx] = rho * cos(theta);
        if (2 * pidx + 1 < M) g[2 * pidx + 1] = rho * sin(theta);
    }
}

/* the paper's own law: components uniform in [-1,1] (Eq. 2). n = 2u - 1. */
void orc_uniforms_pm1(uint64_t seed, uint64_t chain, uint64_t step, int32_t M, double *n)
{
    for (int32_t pidx = 0; 2 * pidx < M; ++pidx) {
        double u1, u2;
        philox_pair(seed, (uint32_t)pidx, chain, step, 0u, &u1, &u2);
        n[2 * pidx] = 2.0 * u1 - 1.0;
        if (2 * pidx + 1 < M) n[2 * pidx + 1] = 2.0 * u2 - 1.0;
    }
}

/* dW: the Brownian increment such that cov(L dW) = 2 D dt.
 * Gaussian: dW = sqrt(2 dt) g.   Uniform (Eq. 2 x dt): dW = dt sqrt(6/dt) n = sqrt(6 dt) n,
 * var(n) = 1/3 -> same second moment.                             */
void orc_noise_dW(const orc_params *p, uint64_t chain, uint64_t step, double *dW)
{
    int32_t M = 3 * (p->n_rods + 1);
    if (p->noise_kind == 1) {
        orc_uniforms_pm1(p->seed, chain, step, M, dW);
        double s = sqrt(6.0 * p->dt);
        for (int32_t m = 0; m < M; ++m) dW[m] = s * dW[m];
    } else {
        orc_normals(p->seed, chain, step, M, dW);
        double s = sqrt(2.0 * p->dt);
        for (int32_t m = 0; m < M; ++m) dW[m] = s * dW[m];
    }
}

/* ---------------------------------------------------------------------------------------
 * Initial conformation: freely jointed random walk (paper: "different initial
 * configurations" from cuRAND, method not given, PAPER.md:258, :166 -- reading A13).
 * Link k: z = 2 u1 - 1, phi = 2 pi u2, Q_k = b (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z)
 * with Philox purpose 1, counter p = k, step 0.  r_0 = 0, prefix sum, centre of mass -> 0.
 * ------------------------------------------------------------------------------------- */
static void shift_to_centre_of_mass(int32_t n_beads, double *r)
{
    double cm[3] = {0.0, 0.0, 0.0};
    for (int32_t i = 0; i < n_beads; ++i)
        for (int d = 0; d < 3; ++d) cm[d] += r[3 * i + d];
    for (int d = 0; d < 3; ++d) cm[d] = cm[d] / (double)n_beads;
    for (int32_t i = 0; i < n_beads; ++i)
        for (int d = 0; d < 3; ++d) r[3 * i + d] -= cm[d];
}

void orc_init_random_walk(int32_t n_rods, double b, uint64_t init_seed, uint64_t chain, double *r)
{
    r[0] = r[1] = r[2] = 0.0;
    for (int32_t k = 0; k < n_rods; ++k) {
        double u1, u2;
        philox_pair(init_seed, (uint32_t)k, chain, 0u, 1u, &u1, &u2);
        double z = 2.0 * u1 - 1.0;
        double phi = 6.283185307179586 * u2;
        double s = sqrt(1.0 - z * z);
        double Q[3] = { b * (s * cos(phi)), b * (s * sin(phi)), b * z };
        for (int d = 0; d < 3; ++d) r[3 * (k + 1) + d] = r[3 * k + d] + Q[d];
    }
    shift_to_centre_of_mass(n_rods + 1, r);
}

/* ---------------------------------------------------------------------------------------
 * Eq. 3: T_k = K (|Q_k| - b)/|Q_k| Q_k  (paper: b = 1).
 * ------------------------------------------------------------------------------------- */
double orc_spring_coeff(const orc_params *p, double q)
{
    if (p->spring_kind == 1) {
        /* Eq. 4: |F| = (alpha r^ - beta r^^3)/(1 - r^^2), alpha = 3, beta = 1,
         * r^ = |Q|/(nu b) the fractional extension; force in units of kT/b (lengths in b,
         * DESIGN.md reading B4), direction along Q:  T = (|F|/b) Q/|Q|.                      */
        double x = q / (p->nu * p->b);
        double F = (3.0 * x - x * x * x) / (1.0 - x * x);
        return (F / p->b) / q;
    }
    return p->K * (q - p->b) / q;                      /* Eq. 3 */
}

void orc_spring_tensions(const orc_params *p, const double *r, double *T)
{
    for (int32_t k = 0; k < p->n_rods; ++k) {
        double Q[3];
        for (int d = 0; d < 3; ++d) Q[d] = r[3 * (k + 1) + d] - r[3 * k + d];
        double q = sqrt(Q[0] * Q[0] + Q[1] * Q[1] + Q[2] * Q[2]);
        double c = orc_spring_coeff(p, q);
        for (int d = 0; d < 3; ++d) T[3 * k + d] = c * Q[d];
    }
}

/* ---------------------------------------------------------------------------------------
 * Semi-implicit link length.  Eq. 13 with D_ii = I (Eq. 7): Y = Q' + 2 dt T(Q'), T parallel to
 * Q', so |Y| = |Q'| + 2 dt |T(|Q'|)|.
 *  Fraenkel rod (Eq. 3):  |Q'| = (2 dt K b + |Y|)/(2 dt K + 1)                       (Eq. 17)
 *  Cohen-Pade spring (Eq. 4), x = |Q'|/(nu b), y = |Y|/(nu b), c = 2 dt/(nu b^2):
 *      y = x + c (3x - x^3)/(1 - x^2)   <=>   (1 + c) x^3 - y x^2 - (1 + 3c) x + y = 0,
 *  f(0) = y >= 0 and f(1) = -2c < 0: exactly one root in [0, 1) (finite extensibility); found
 *  by plain bisection (200 halvings: to the last bit).  The paper states the scheme for the
 *  Fraenkel spring only and refers to its ref. [27] for the rest (reading B4).
 * ------------------------------------------------------------------------------------- */
double orc_implicit_length(const orc_params *p, double Yn)
{
    if (p->spring_kind == 1) {
        double L = p->nu * p->b;
        double y = Yn / L, c = 2.0 * p->dt / (p->nu * p->b * p->b);
        double lo = 0.0, hi = 1.0;
        for (int it = 0; it < 200; ++it) {
            double x = 0.5 * (lo + hi);
            double f = ((1.0 + c) * x - y) * x * x - (1.0 + 3.0 * c) * x + y;
            if (f > 0.0) lo = x; else hi = x;
        }
        return 0.5 * (lo + hi) * L;
    }
    return (2.0 * p->dt * p->K * p->b + Yn) / (2.0 * p->dt * p->K + 1.0);
}

/* Eq. 1 net spring term (F^S_{i+1} - F^S_i) and Eq. 22:
 * F_0 = T_0, F_j = T_j - T_{j-1}, F_N = -T_{N-1}.                                        */
void orc_bead_forces(int32_t n_rods, const double *T, double *F)
{
    for (int32_t j = 0; j <= n_rods; ++j)
        for (int d = 0; d < 3; ++d) {
            double right = (j < n_rods) ? T[3 * j + d] : 0.0;
            double left = (j > 0) ? T[3 * (j - 1) + d] : 0.0;
            F[3 * j + d] = right - left;
        }
}

/* ---------------------------------------------------------------------------------------
 * Eqs. 8-9, off-diagonal 3x3 block between beads at ri, rj.
 * Lengths in units of b (paper: b = 1).  R_vec = r_i - r_j (reading A2).
 *  R >= 2a : (3h/(4R)) [ (1 + 2a^2/(3R^2)) I + (1 - 2a^2/R^2) RR/R^2 ]          (Eq. 8)
 *  R <  2a : (3h/(4R))(R/(2a)) [ (8/3 - 3R/(4a)) I + (R/(4a)) RR/R^2 ]          (Eq. 9)
 *          = (3h/(8a)) [ (8/3 - 3R/(4a)) I + RR/(4aR) ]   (finite as R -> 0)
 * ------------------------------------------------------------------------------------- */
void orc_rpy_block(const orc_params *p, const double *ri, const double *rj, double B[9])
{
    double Rv[3];
    for (int d = 0; d < 3; ++d) Rv[d] = (ri[d] - rj[d]) / p->b;
    double a = p->a / p->b;
    double h = p->hstar;
    double R2 = Rv[0] * Rv[0] + Rv[1] * Rv[1] + Rv[2] * Rv[2];
    double R = sqrt(R2);
    double cI, cRR;   /* block = cI * I + cRR * Rv Rv^T */
    if (R >= 2.0 * a) {
        double pre = 3.0 * h / (4.0 * R);
        cI = pre * (1.0 + 2.0 * a * a / (3.0 * R2));
        cRR = pre * (1.0 - 2.0 * a * a / R2) / R2;
    } else {
        double pre = 3.0 * h / (8.0 * a);
        cI = pre * (8.0 / 3.0 - 3.0 * R / (4.0 * a));
        cRR = (R > 0.0) ? pre / (4.0 * a * R) : 0.0;
    }
    for (int k = 0; k < 3; ++k)
        for (int l = 0; l < 3; ++l)
            B[3 * k + l] = cRR * Rv[k] * Rv[l] + ((k == l) ? cI : 0.0);
}

/* Eqs. 7, 18-19: D_ii = I; block (i,j) at rows 3i.., cols 3j.. */
void orc_assemble(const orc_params *p, const double *r, double *D)
{
    int32_t nb = p->n_rods + 1, M = 3 * nb;
    for (int32_t i = 0; i < nb; ++i)
        for (int32_t j = 0; j < nb; ++j) {
            double B[9];
            if (i == j) {
                for (int e = 0; e < 9; ++e) B[e] = 0.0;
                B[0] = B[4] = B[8] = 1.0;
            } else {
                orc_rpy_block(p, r + 3 * i, r + 3 * j, B);
            }
            for (int k = 0; k < 3; ++k)
                for (int l = 0; l < 3; ++l)
                    D[(size_t)(3 * i + k) * M + (3 * j + l)] = B[3 * k + l];
        }
}

/* ---------------------------------------------------------------------------------------
 * Eq. 10: D = sigma sigma^T, sigma = L lower, positive diagonal
 * (reading A11).  Cholesky-Banachiewicz, row by row.  Reads the lower triangle of A.
 * returns 0, or the 1-based row of the first non-positive (or NaN) pivot (reading A10).
 * ------------------------------------------------------------------------------------- */
int32_t orc_cholesky(int32_t M, const double *A, double *L)
{
    for (int32_t i = 0; i < M; ++i)
        for (int32_t j = 0; j < M; ++j) L[(size_t)i * M + j] = 0.0;
    for (int32_t i = 0; i < M; ++i) {
        for (int32_t j = 0; j < i; ++j) {
            double s = A[(size_t)i * M + j];
            for (int32_t k = 0; k < j; ++k) s -= L[(size_t)i * M + k] * L[(size_t)j * M + k];
            L[(size_t)i * M + j] = s / L[(size_t)j * M + j];
        }
        double s = A[(size_t)i * M + i];
        for (int32_t k = 0; k < i; ++k) s -= L[(size_t)i * M + k] * L[(size_t)i * M + k];
        if (!(s > 0.0)) return i + 1;
        L[(size_t)i * M + i] = sqrt(s);
    }
    return 0;
}

/* Eq. 6 second term: v_i = sum_j D_ij F_j, full matrix, j ascending. */
void orc_symv(int32_t M, const double *D, const double *x, double *v)
{
    for (int32_t i = 0; i < M; ++i) {
        double s = 0.0;
        for (int32_t j = 0; j < M; ++j) s += D[(size_t)i * M + j] * x[j];
        v[i] = s;
    }
}

/* Eq. 6 third term (reading A1): y_i = sum_{j<=i} L_ij dW_j. */
void orc_trmv_lower(int32_t M, const double *L, const double *x, double *y)
{
    for (int32_t i = 0; i < M; ++i) {
        double s = 0.0;
        for (int32_t j = 0; j <= i; ++j) s += L[(size_t)i * M + j] * x[j];
        y[i] = s;
    }
}

/* same v as orc_symv(orc_assemble(r)) without storing D: blocks recomputed, j ascending. */
void orc_drift_onthefly(const orc_params *p, const double *r, const double *F, double *v)
{
    int32_t nb = p->n_rods + 1;
    for (int32_t i = 0; i < nb; ++i) {
        double s[3] = {0.0, 0.0, 0.0};
        for (int32_t j = 0; j < nb; ++j) {
            double B[9];
            if (i == j) {
                for (int e = 0; e < 9; ++e) B[e] = 0.0;
                B[0] = B[4] = B[8] = 1.0;
            } else {
                orc_rpy_block(p, r + 3 * i, r + 3 * j, B);
            }
            for (int k = 0; k < 3; ++k)
                for (int l = 0; l < 3; ++l) s[k] += B[3 * k + l] * F[3 * j + l];
        }
        for (int k = 0; k < 3; ++k) v[3 * i + k] = s[k];
    }
}

/* ---------------------------------------------------------------------------------------
 * Steps 7-10 of DESIGN.md's algorithm:
 *  u_i = dt (kappa r_i + v_i) + y_i                    (Eq. 6 x dt; Eq. 5)
 *  Y_k = Q_k + (u_{k+1} - u_k) + 2 dt T_k              (Eq. 14; reading A7)
 *  |Q'_k| = (2 dt K b + |Y_k|) / (2 dt K + 1)          (Eq. 17)
 *  Q'_k = Y_k |Q'_k| / |Y_k|                           (Eq. 15; recipe :156-160)
 *  r'_0 = 0, r'_{k+1} = r'_k + Q'_k, r' -= mean(r')    (reading A8)
 * returns 0 or M+1 if a non-finite value or |Y_k| = 0 appears (reading A10).
 * ------------------------------------------------------------------------------------- */
int32_t orc_finish_step(const orc_params *p, const double *r, const double *T, const double *v,
                        const double *y, double *r_out, double *u_out, double *Y_out)
{
    int32_t N = p->n_rods, nb = N + 1, M = 3 * nb;
    double *u = (double *)malloc(sizeof(double) * (size_t)M);
    double *rn = (double *)malloc(sizeof(double) * (size_t)M);
    int32_t info = 0;
    for (int32_t i = 0; i < nb; ++i)
        for (int k = 0; k < 3; ++k) {
            double flow = p->kappa[3 * k + 0] * r[3 * i + 0] + p->kappa[3 * k + 1] * r[3 * i + 1] +
                          p->kappa[3 * k + 2] * r[3 * i + 2];
            u[3 * i + k] = p->dt * (flow + v[3 * i + k]) + y[3 * i + k];
        }
    rn[0] = rn[1] = rn[2] = 0.0;
    for (int32_t k = 0; k < N; ++k) {
        double Y[3];
        for (int d = 0; d < 3; ++d) {
            double Q = r[3 * (k + 1) + d] - r[3 * k + d];
            Y[d] = Q + (u[3 * (k + 1) + d] - u[3 * k + d]) + 2.0 * p->dt * T[3 * k + d];
        }
        double Yn = sqrt(Y[0] * Y[0] + Y[1] * Y[1] + Y[2] * Y[2]);
        double qn = orc_implicit_length(p, Yn);          /* Eq. 17 (or the Cohen-Pade cubic) */
        double scale = qn / Yn;
        if (!(Yn > 0.0) || !isfinite(scale)) info = M + 1;
        for (int d = 0; d < 3; ++d) {
            rn[3 * (k + 1) + d] = rn[3 * k + d] + Y[d] * scale;
            if (Y_out) Y_out[3 * k + d] = Y[d];
        }
    }
    shift_to_centre_of_mass(nb, rn);
    for (int32_t m = 0; m < M; ++m)
        if (!isfinite(rn[m])) info = M + 1;
    if (u_out) memcpy(u_out, u, sizeof(double) * (size_t)M);
    if (info == 0) memcpy(r_out, rn, sizeof(double) * (size_t)M);
    else if (r_out != r) memcpy(r_out, r, sizeof(double) * (size_t)M);
    free(u); free(rn);
    return info;
}

/* One chain, one step: DESIGN.md algorithm steps 1-10 in order. */
int32_t orc_step(const orc_params *p, uint64_t chain, uint64_t step, const double *r_in,
                 double *r_out, orc_trace *tr)
{
    int32_t N = p->n_rods, nb = N + 1, M = 3 * nb;
    size_t MM = (size_t)M * (size_t)M;
    double *T = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *F = (double *)malloc(sizeof(double) * (size_t)M);
    double *D = (double *)malloc(sizeof(double) * MM);
    double *L = (double *)malloc(sizeof(double) * MM);
    double *dW = (double *)malloc(sizeof(double) * (size_t)M);
    double *v = (double *)malloc(sizeof(double) * (size_t)M);
    double *y = (double *)malloc(sizeof(double) * (size_t)M);
    int32_t info;

    orc_spring_tensions(p, r_in, T);                 /* 1 */
    orc_bead_forces(N, T, F);                        /* 2 */
    orc_assemble(p, r_in, D);                        /* 3 */
    info = orc_cholesky(M, D, L);                    /* 4 */
    orc_noise_dW(p, chain, step, dW);                /* 5 */
    if (tr) {
        if (tr->T) memcpy(tr->T, T, sizeof(double) * 3 * (size_t)N);
        if (tr->F) memcpy(tr->F, F, sizeof(double) * (size_t)M);
        if (tr->D) memcpy(tr->D, D, sizeof(double) * MM);
        if (tr->L) memcpy(tr->L, L, sizeof(double) * MM);
        if (tr->dW) memcpy(tr->dW, dW, sizeof(double) * (size_t)M);
    }
    if (info == 0) {
        orc_symv(M, D, F, v);                        /* 6 */
        orc_trmv_lower(M, L, dW, y);
        if (tr && tr->v) memcpy(tr->v, v, sizeof(double) * (size_t)M);
        if (tr && tr->y) memcpy(tr->y, y, sizeof(double) * (size_t)M);
        info = orc_finish_step(p, r_in, T, v, y, r_out, tr ? tr->u : NULL, tr ? tr->Y : NULL); /* 7-10 */
    } else if (r_out != r_in) {
        memcpy(r_out, r_in, sizeof(double) * (size_t)M);
    }
    free(T); free(F); free(D); free(L); free(dW); free(v); free(y);
    return info;
}

int32_t orc_step_ensemble(const orc_params *p, int32_t C, uint64_t chain0, uint64_t first_step,
                          int32_t n_steps, double *r, int32_t *info)
{
    int32_t M = 3 * (p->n_rods + 1);
    int32_t failed = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : failed)
    for (int32_t c = 0; c < C; ++c) {
        double *rc = r + (size_t)c * M;
        int32_t first = 0;
        for (int32_t s = 0; s < n_steps; ++s) {
            int32_t e = orc_step(p, chain0 + (uint64_t)c, first_step + (uint64_t)s, rc, rc, NULL);
            if (e != 0 && first == 0) first = e;
        }
        if (info) info[c] = first;
        if (first != 0) failed += 1;
    }
    return failed;
}

/* ---------------------------------------------------------------------------------------
 * Observables per chain (Eqs. 25-29; readings A15, A18):
 *  0 R^2 = |r_N - r_0|^2            (Eq. 25 integrand)
 *  1..3 (x_N-x_0)^2, (y..)^2, (z..)^2 (Eq. 26)
 *  4 Rg^2 = sum_i |r_i - r_cm|^2/(N+1) (Eq. 27 integrand)
 *  5..10 S_xx S_yy S_zz S_xy S_xz S_yz, S = sum_k T_k (x) Q_k (Eq. 28 without N delta)
 *  11 mean_k (|Q_k| - b)^2 ; 12 max_k | |Q_k| - b |      (rod-length check, pin P7)
 * ------------------------------------------------------------------------------------- */
void orc_observables_chain(const orc_params *p, const double *r, double obs[ORC_NOBS])
{
    int32_t N = p->n_rods, nb = N + 1;
    double Re[3], cm[3] = {0, 0, 0};
    for (int d = 0; d < 3; ++d) Re[d] = r[3 * N + d] - r[d];
    obs[1] = Re[0] * Re[0]; obs[2] = Re[1] * Re[1]; obs[3] = Re[2] * Re[2];
    obs[0] = obs[1] + obs[2] + obs[3];
    for (int32_t i = 0; i < nb; ++i)
        for (int d = 0; d < 3; ++d) cm[d] += r[3 * i + d];
    for (int d = 0; d < 3; ++d) cm[d] = cm[d] / (double)nb;
    double rg = 0.0;
    for (int32_t i = 0; i < nb; ++i)
        for (int d = 0; d < 3; ++d) {
            double x = r[3 * i + d] - cm[d];
            rg += x * x;
        }
    obs[4] = rg / (double)nb;
    double S[6] = {0, 0, 0, 0, 0, 0}, dev2 = 0.0, devmax = 0.0;
    for (int32_t k = 0; k < N; ++k) {
        double Q[3], T[3];
        for (int d = 0; d < 3; ++d) Q[d] = r[3 * (k + 1) + d] - r[3 * k + d];
        double q = sqrt(Q[0] * Q[0] + Q[1] * Q[1] + Q[2] * Q[2]);
        double c = orc_spring_coeff(p, q);
        for (int d = 0; d < 3; ++d) T[d] = c * Q[d];
        S[0] += T[0] * Q[0]; S[1] += T[1] * Q[1]; S[2] += T[2] * Q[2];
        S[3] += T[0] * Q[1]; S[4] += T[0] * Q[2]; S[5] += T[1] * Q[2];
        double dv = q - p->b;
        dev2 += dv * dv;
        if (fabs(dv) > devmax) devmax = fabs(dv);
    }
    for (int e = 0; e < 6; ++e) obs[5 + e] = S[e];
    obs[11] = dev2 / (double)N;
    obs[12] = devmax;
}

/* ensemble[0][o] = sum_c obs, ensemble[1][o] = sum_c obs^2 (mean and SE on the host). */
void orc_observables(const orc_params *p, int32_t C, const double *r, double *per_chain, double *ensemble)
{
    int32_t M = 3 * (p->n_rods + 1);
#pragma omp parallel for schedule(static)
    for (int32_t c = 0; c < C; ++c) orc_observables_chain(p, r + (size_t)c * M, per_chain + (size_t)c * ORC_NOBS);
    for (int o = 0; o < 2 * ORC_NOBS; ++o) ensemble[o] = 0.0;
    for (int32_t c = 0; c < C; ++c)
        for (int o = 0; o < ORC_NOBS; ++o) {
            double x = per_chain[(size_t)c * ORC_NOBS + o];
            ensemble[o] += x;
            ensemble[ORC_NOBS + o] += x * x;
        }
}

/* ---------------------------------------------------------------------------------------
 * End-to-end vector and its autocorrelation (the relaxation time is "the time scale of
 * the decay of the autocorrelation function of the end-to-end vector of the chain", fitted over its
 * last 70 %; reading B3: ensemble average at lag t from a common origin,
 * C(t) = <R(t).R(0)> / <R(0).R(0)>).
 *   R_c = r_N - r_0                                          (Eq. 25's vector)
 *   out[0] = sum_c R_c.R0_c, out[1] = sum_c (R_c.R0_c)^2, out[2] = sum_c R0_c.R0_c
 * ------------------------------------------------------------------------------------- */
void orc_end_to_end(int32_t n_rods, int32_t C, const double *r, double *R)
{
    size_t M = 3 * ((size_t)n_rods + 1);
    for (int32_t c = 0; c < C; ++c)
        for (int d = 0; d < 3; ++d) R[3 * (size_t)c + d] = r[c * M + 3 * (size_t)n_rods + d] - r[c * M + d];
}

void orc_autocorr(int32_t n_rods, int32_t C, const double *r, const double *R0, double out[3])
{
    size_t M = 3 * ((size_t)n_rods + 1);
    out[0] = out[1] = out[2] = 0.0;
    for (int32_t c = 0; c < C; ++c) {
        double dot = 0.0, n0 = 0.0;
        for (int d = 0; d < 3; ++d) {
            double Rd = r[c * M + 3 * (size_t)n_rods + d] - r[c * M + d];
            dot += Rd * R0[3 * (size_t)c + d];
            n0 += R0[3 * (size_t)c + d] * R0[3 * (size_t)c + d];
        }
        out[0] += dot;
        out[1] += dot * dot;
        out[2] += n0;
    }
}

int32_t orc_num_threads(void)
{
#ifdef _OPENMP
    return (int32_t)omp_get_max_threads();
#else
    return 1;
#endif
}
