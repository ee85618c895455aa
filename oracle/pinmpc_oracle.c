/*
 * pinmpc_oracle.c — float64 CPU oracle for the batched ADMM-MPC hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct C in double precision.  It shares no
 * code with the CUDA path (paper_2606_05687_b200/csrc) and neither includes the other.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * What it computes (citations: /root/reference/PAPER.md line numbers + SURVEY.md section 8(c)):
 *   the LTV QP of PAPER.md:L142-148, eq. (16)-(17), with C = I, X_k = R^nx:
 *       min  sum_k 1/2 |x_{k+1}-xbar_{k+1}|^2_Q + 1/2 |u_k-ubar_k|^2_R
 *       s.t. x_{k+1} = A_k x_k + B_k u_k + c_k,  x_0 given,  u_k in U_k
 *   iterated by a scaled-form ADMM (Boyd et al. [32]) in the block order of
 *   PAPER.md:L186 eq. (21a)->(21b)->(21c): equality-constrained step, projection, dual update,
 *   stopped after a fixed iteration count.  Readings of the paper:
 *   the dynamics are kept hard inside the equality step (exact time-varying LQR), D2.
 *
 *   O1 orc_assemble      A_k,B_k,c_k of the single-rigid-body model (BASELINE.json config 0;
 *                        the SRB counterpart of PAPER.md:L49-55 eq. (2)-(4))
 *   O2 orc_factor_env    Riccati factorisation of the equality step (analogue of caching
 *                        J_k,H_k "before ADMM iterations")
 *   O3 orc_eqstep_env    equality-constrained step (21a) for given z,y;   orc_solve: the loop
 *   O4 orc_project_stage exact Euclidean projection onto U_k (z-update; sets of
 *                        PAPER.md:L85 eq. (7c) with BASELINE.json's constants)
 *
 * Pins (tests/, -m "not gpu"): O1 closed forms + forward-Euler of the continuous ODE; O2+O3
 * dense KKT solve and an independent numpy Riccati to 1e-9; O4 brute-force face enumeration,
 * hand-derived golden cases, idempotence, non-expansiveness, Moreau; converged iterate vs an
 * independent dense active-set QP solve to 1e-6.  Fixed-iteration outputs at rho = 1 are pinned
 * only transitively ("parity unpinned by the paper": it prints no solver values).
 *
 * Layouts: env-major, row-major, all double.  State x = [Theta(3) p(3) omega(3) v(3) g],
 * control u = [f_0..f_{nw-1} | m_0..m_{nw-1} | fh_0..fh_{nf-1}], each block 3 wide.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NX 13
#define NU_MAX 18

typedef struct {
    int n_wrench, n_force;
    double mu, fz_max, mx_coef, my_coef, mz_coef, hand_fmax;
} orc_layout;

/* ------------------------------------------------------------------------------------------ */
/* O1  assembly                                                                                */
/* ------------------------------------------------------------------------------------------ */
static void inv3(const double *M, double *Mi)
{
    double c00 = M[4] * M[8] - M[5] * M[7], c01 = M[5] * M[6] - M[3] * M[8], c02 = M[3] * M[7] - M[4] * M[6];
    double det = M[0] * c00 + M[1] * c01 + M[2] * c02;
    Mi[0] = c00 / det; Mi[1] = (M[2] * M[7] - M[1] * M[8]) / det; Mi[2] = (M[1] * M[5] - M[2] * M[4]) / det;
    Mi[3] = c01 / det; Mi[4] = (M[0] * M[8] - M[2] * M[6]) / det; Mi[5] = (M[2] * M[3] - M[0] * M[5]) / det;
    Mi[6] = c02 / det; Mi[7] = (M[1] * M[6] - M[0] * M[7]) / det; Mi[8] = (M[0] * M[4] - M[1] * M[3]) / det;
}

static void matmul(int n, int m, int p, const double *X, const double *Y, double *Z)
{   /* Z[n,p] = X[n,m] Y[m,p] */
    for (int i = 0; i < n; i++)
        for (int j = 0; j < p; j++) {
            double a = 0.0;
            for (int l = 0; l < m; l++) a += X[i * m + l] * Y[l * p + j];
            Z[i * p + j] = a;
        }
}

static void matmul_tn(int n, int m, int p, const double *X, const double *Y, double *Z)
{   /* Z[n,p] = X^T Y with X[m,n], Y[m,p] */
    for (int i = 0; i < n; i++)
        for (int j = 0; j < p; j++) {
            double a = 0.0;
            for (int l = 0; l < m; l++) a += X[l * n + i] * Y[l * p + j];
            Z[i * p + j] = a;
        }
}

/* One stage: A[13*13], Bm[13*nu], c[13] from yaw, contact offsets r[nc][3], mass, body inertia,
 * optional external wrench ext = (F_ext, tau_ext).  SURVEY 8(c)-O1. */
void orc_assemble_stage(int nu, int nw, int nf, double dt, double yaw, const double *r, double mass,
                        const double *Ib, const double *ext, double *A, double *Bm, double *c)
{
    double cs = cos(yaw), sn = sin(yaw);
    double Rz[9] = { cs, -sn, 0, sn, cs, 0, 0, 0, 1 };
    double RzT[9] = { cs, sn, 0, -sn, cs, 0, 0, 0, 1 };
    double Ibi[9], T[9], Iwi[9];
    inv3(Ib, Ibi);
    matmul(3, 3, 3, Rz, Ibi, T);
    matmul(3, 3, 3, T, RzT, Iwi);                 /* I_w^{-1} = R_z I_b^{-1} R_z^T */

    memset(A, 0, sizeof(double) * NX * NX);
    memset(Bm, 0, sizeof(double) * NX * nu);
    memset(c, 0, sizeof(double) * NX);
    for (int i = 0; i < NX; i++) A[i * NX + i] = 1.0;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) A[i * NX + 6 + j] = dt * RzT[i * 3 + j];   /* dTheta = R_z^T omega */
    for (int i = 0; i < 3; i++) A[(3 + i) * NX + 9 + i] = dt;                  /* dp = v */
    A[11 * NX + 12] = dt;                                                      /* dv_z += g-state */

    int nc = nw + nf;
    for (int i = 0; i < nc; i++) {
        const double *ri = r + 3 * i;
        double S[9] = { 0, -ri[2], ri[1], ri[2], 0, -ri[0], -ri[1], ri[0], 0 };   /* [r]x */
        double IS[9];
        matmul(3, 3, 3, Iwi, S, IS);
        int fcol = (i < nw) ? 3 * i : 6 * nw + 3 * (i - nw);
        for (int a = 0; a < 3; a++) {
            for (int b = 0; b < 3; b++) Bm[(6 + a) * nu + fcol + b] = dt * IS[a * 3 + b];
            Bm[(9 + a) * nu + fcol + a] = dt / mass;
        }
        if (i < nw) {
            int mcol = 3 * nw + 3 * i;
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++) Bm[(6 + a) * nu + mcol + b] = dt * Iwi[a * 3 + b];
        }
    }
    if (ext) {
        for (int a = 0; a < 3; a++) {
            double t = 0.0;
            for (int b = 0; b < 3; b++) t += Iwi[a * 3 + b] * ext[3 + b];
            c[6 + a] = dt * t;
            c[9 + a] = dt / mass * ext[a];
        }
    }
}

/* Batched O1.  yaw[B,N], foot_r[B,N,nc,3], mass[B], inertia[B,3,3], ext[B,N,6] or NULL. */
void orc_assemble(int B, int N, int nu, int nw, int nf, double dt, const double *yaw, const double *foot_r,
                  const double *mass, const double *inertia, const double *ext,
                  double *A, double *Bm, double *c)
{
    int nc = nw + nf;
    for (long b = 0; b < B; b++)
        for (long k = 0; k < N; k++) {
            long s = b * N + k;
            orc_assemble_stage(nu, nw, nf, dt, yaw[s], foot_r + s * nc * 3, mass[b], inertia + b * 9,
                               ext ? ext + s * 6 : NULL, A + s * NX * NX, Bm + s * NX * nu, c + s * NX);
        }
}

/* ------------------------------------------------------------------------------------------ */
/* O2  factorisation of the equality-constrained step (one env)                                 */
/* ------------------------------------------------------------------------------------------ */
static int cholesky(int n, const double *M, double *L)
{
    memset(L, 0, sizeof(double) * n * n);
    for (int j = 0; j < n; j++) {
        double d = M[j * n + j];
        for (int l = 0; l < j; l++) d -= L[j * n + l] * L[j * n + l];
        if (!(d > 0.0)) return 1;
        L[j * n + j] = sqrt(d);
        for (int i = j + 1; i < n; i++) {
            double a = M[i * n + j];
            for (int l = 0; l < j; l++) a -= L[i * n + l] * L[j * n + l];
            L[i * n + j] = a / L[j * n + j];
        }
    }
    return 0;
}

static void chol_solve(int n, const double *L, const double *b, double *x)
{   /* x = (L L^T)^{-1} b */
    double t[NU_MAX];
    for (int i = 0; i < n; i++) {
        double a = b[i];
        for (int l = 0; l < i; l++) a -= L[i * n + l] * t[l];
        t[i] = a / L[i * n + i];
    }
    for (int i = n - 1; i >= 0; i--) {
        double a = t[i];
        for (int l = i + 1; l < n; l++) a -= L[l * n + i] * x[l];
        x[i] = a / L[i * n + i];
    }
}

/* Riccati recursion:  Rt = R + rho I,  P_N = Q, for k = N-1..0
 *   M_k = Rt + B^T P_{k+1} B,  K_k = M_k^{-1} B^T P_{k+1} A,  Phi_k = A - B K_k,
 *   P_k = [k>=1] Q + A^T P_{k+1} Phi_k (symmetrised),  s_k = P_{k+1} c_k.
 * Outputs K[N,nu,13], L[N,nu,nu] (Cholesky factor of M_k), Phi[N,13,13], s[N,13]; P0[13,13]
 * (P at stage 0 without the [k>=1] Q term, for tests) may be NULL.  Returns nonzero if some M_k
 * is not positive definite. */
int orc_factor_env(int N, int nu, const double *A, const double *Bm, const double *c,
                   const double *Qd, const double *Rd, double rho,
                   double *K, double *L, double *Phi, double *s, double *P0)
{
    double P[NX * NX], PB[NX * NU_MAX], PA[NX * NX], M[NU_MAX * NU_MAX], BtPA[NU_MAX * NX];
    double PPhi[NX * NX], Pn[NX * NX], col[NU_MAX], sol[NU_MAX];
    memset(P, 0, sizeof P);
    for (int i = 0; i < NX; i++) P[i * NX + i] = Qd[i];
    for (int k = N - 1; k >= 0; k--) {
        const double *Ak = A + (long)k * NX * NX, *Bk = Bm + (long)k * NX * nu, *ck = c + (long)k * NX;
        double *Kk = K + (long)k * nu * NX, *Lk = L + (long)k * nu * nu, *Phik = Phi + (long)k * NX * NX;
        matmul(NX, NX, nu, P, Bk, PB);
        matmul_tn(nu, NX, nu, Bk, PB, M);
        for (int i = 0; i < nu; i++) M[i * nu + i] += Rd[i] + rho;
        if (cholesky(nu, M, Lk)) return 1;
        matmul(NX, NX, NX, P, Ak, PA);
        matmul_tn(nu, NX, NX, Bk, PA, BtPA);
        for (int j = 0; j < NX; j++) {
            for (int i = 0; i < nu; i++) col[i] = BtPA[i * NX + j];
            chol_solve(nu, Lk, col, sol);
            for (int i = 0; i < nu; i++) Kk[i * NX + j] = sol[i];
        }
        matmul(NX, nu, NX, Bk, Kk, Phik);
        for (int i = 0; i < NX * NX; i++) Phik[i] = Ak[i] - Phik[i];
        for (int i = 0; i < NX; i++) {
            double a = 0.0;
            for (int j = 0; j < NX; j++) a += P[i * NX + j] * ck[j];
            s[(long)k * NX + i] = a;
        }
        matmul(NX, NX, NX, P, Phik, PPhi);
        matmul_tn(NX, NX, NX, Ak, PPhi, Pn);
        for (int i = 0; i < NX; i++)
            for (int j = 0; j < NX; j++)
                P[i * NX + j] = 0.5 * (Pn[i * NX + j] + Pn[j * NX + i]) + ((k >= 1 && i == j) ? Qd[i] : 0.0);
    }
    if (P0) memcpy(P0, P, sizeof P);
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* O3 steps 1-3  equality-constrained step for given z, y (one env)                             */
/* ------------------------------------------------------------------------------------------ */
/* x_ref[N,13] holds xbar_1..xbar_N; u_ref[N,nu] or NULL; outputs x[N,13] = x_1..x_N, u[N,nu]. */
void orc_eqstep_env(int N, int nu, const double *A, const double *Bm, const double *c,
                    const double *K, const double *L, const double *Phi, const double *s,
                    const double *Qd, const double *Rd, double rho,
                    const double *x0, const double *x_ref, const double *u_ref,
                    const double *z, const double *y, double *x, double *u, double *kappa /*[N,nu] scratch*/)
{
    double p[NX], g[NX], pn[NX], rk[NU_MAX], h[NU_MAX];
    /* step 2: backward vector pass, p = q_N */
    for (int i = 0; i < NX; i++) p[i] = Qd[i] * x_ref[(long)(N - 1) * NX + i];
    for (int k = N - 1; k >= 0; k--) {
        const double *Bk = Bm + (long)k * NX * nu, *Kk = K + (long)k * nu * NX, *Phik = Phi + (long)k * NX * NX;
        /* step 1: r_k = R ubar_k + rho (z_k - y_k) */
        for (int j = 0; j < nu; j++)
            rk[j] = Rd[j] * (u_ref ? u_ref[(long)k * nu + j] : 0.0) + rho * (z[(long)k * nu + j] - y[(long)k * nu + j]);
        for (int i = 0; i < NX; i++) g[i] = p[i] - s[(long)k * NX + i];
        for (int j = 0; j < nu; j++) {
            double a = rk[j];
            for (int i = 0; i < NX; i++) a += Bk[i * nu + j] * g[i];
            h[j] = a;
        }
        chol_solve(nu, L + (long)k * nu * nu, h, kappa + (long)k * nu);
        for (int i = 0; i < NX; i++) {
            double a = (k >= 1) ? Qd[i] * x_ref[(long)(k - 1) * NX + i] : 0.0;     /* q_k = Q xbar_k */
            for (int l = 0; l < NX; l++) a += Phik[l * NX + i] * g[l];
            for (int j = 0; j < nu; j++) a -= Kk[j * NX + i] * rk[j];
            pn[i] = a;
        }
        memcpy(p, pn, sizeof p);
    }
    /* step 3: forward rollout */
    double xk[NX], xn[NX];
    memcpy(xk, x0, sizeof xk);
    for (int k = 0; k < N; k++) {
        const double *Ak = A + (long)k * NX * NX, *Bk = Bm + (long)k * NX * nu, *Kk = K + (long)k * nu * NX;
        double *uk = u + (long)k * nu;
        for (int j = 0; j < nu; j++) {
            double a = kappa[(long)k * nu + j];
            for (int i = 0; i < NX; i++) a -= Kk[j * NX + i] * xk[i];
            uk[j] = a;
        }
        for (int i = 0; i < NX; i++) {
            double a = c[(long)k * NX + i];
            for (int l = 0; l < NX; l++) a += Ak[i * NX + l] * xk[l];
            for (int j = 0; j < nu; j++) a += Bk[i * nu + j] * uk[j];
            xn[i] = a;
        }
        memcpy(x + (long)k * NX, xn, sizeof xn);
        memcpy(xk, xn, sizeof xk);
    }
}

/* ------------------------------------------------------------------------------------------ */
/* O4  exact Euclidean projection onto U_k                                                      */
/* ------------------------------------------------------------------------------------------ */
/* Foot wrench set W = { |f_x|,|f_y| <= mu t, |m_x| <= a_x t, |m_y| <= a_y t, |m_z| <= b t,
 * 0 <= t <= f_max }, t = f_z.  For fixed t the best y_i is the clip to +-w_i t, which leaves
 * the 1-D convex problem  min_t 1/2 (t-t0)^2 + 1/2 sum_i (|y_i| - w_i t)_+^2  on [0, f_max].
 * Its derivative g(t) = (t-t0) - sum_{i: |y_i| > w_i t} w_i (|y_i| - w_i t) is continuous,
 * increasing, piecewise linear with kinks at |y_i|/w_i: walk the sorted kinks to its root. */
void orc_project_wrench(const orc_layout *lay, const double *f, const double *m, double *fo, double *mo)
{
    double yv[5] = { f[0], f[1], m[0], m[1], m[2] };
    double w[5] = { lay->mu, lay->mu, lay->mx_coef, lay->my_coef, lay->mz_coef };
    double t0 = f[2], bp[5];
    int ord[5];
    for (int i = 0; i < 5; i++) {
        bp[i] = (w[i] > 0.0) ? fabs(yv[i]) / w[i] : INFINITY;
        ord[i] = i;
    }
    for (int i = 1; i < 5; i++)                      /* insertion sort of the kinks */
        for (int j = i; j > 0 && bp[ord[j]] < bp[ord[j - 1]]; j--) { int t = ord[j]; ord[j] = ord[j - 1]; ord[j - 1] = t; }
    double tstar = 0.0;
    for (int piece = 0; piece <= 5; piece++) {       /* on piece j the active set is ord[j..4] */
        double num = t0, den = 1.0;
        for (int j = piece; j < 5; j++) { int i = ord[j]; num += w[i] * fabs(yv[i]); den += w[i] * w[i]; }
        double t = num / den;
        double lo = (piece == 0) ? -INFINITY : bp[ord[piece - 1]];
        double hi = (piece == 5) ? INFINITY : bp[ord[piece]];
        if (t >= lo && t <= hi) { tstar = t; break; }
        if (piece == 5) tstar = t;
    }
    double t = tstar < 0.0 ? 0.0 : (tstar > lay->fz_max ? lay->fz_max : tstar);
    double out[5];
    for (int i = 0; i < 5; i++) {
        double lim = w[i] * t;
        out[i] = yv[i] > lim ? lim : (yv[i] < -lim ? -lim : yv[i]);
    }
    fo[0] = out[0]; fo[1] = out[1]; fo[2] = t;
    mo[0] = out[2]; mo[1] = out[3]; mo[2] = out[4];
}

/* z = Proj_{U_k}(v) for one stage; contact[nc] (1 = in contact).  Swing contact => 0;
 * hand (3-D force contact) => componentwise clamp to +-hand_fmax. */
void orc_project_stage(const orc_layout *lay, int nu, const unsigned char *contact, const double *v, double *z)
{
    int nw = lay->n_wrench, nf = lay->n_force;
    (void)nu;
    for (int i = 0; i < nw; i++) {
        const double *f = v + 3 * i, *m = v + 3 * nw + 3 * i;
        double *fo = z + 3 * i, *mo = z + 3 * nw + 3 * i;
        if (contact[i]) orc_project_wrench(lay, f, m, fo, mo);
        else for (int a = 0; a < 3; a++) { fo[a] = 0.0; mo[a] = 0.0; }
    }
    for (int j = 0; j < nf; j++) {
        const double *f = v + 6 * nw + 3 * j;
        double *fo = z + 6 * nw + 3 * j;
        for (int a = 0; a < 3; a++) {
            double q = f[a], lim = lay->hand_fmax;
            fo[a] = !contact[nw + j] ? 0.0 : (q > lim ? lim : (q < -lim ? -lim : q));
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* O3  the ADMM loop (one env)                                                  */
/* ------------------------------------------------------------------------------------------ */
static int solve_env(int N, int nu, const orc_layout *lay, double rho, int iters,
                     double eps_abs, double eps_rel, int check_every,
                     const double *Qd, const double *Rd, const double *A, const double *Bm, const double *c,
                     const double *x0, const double *x_ref, const double *u_ref, const unsigned char *contact,
                     double *x, double *u, double *z, double *y, double *r_prim, double *r_dual, int *iters_done,
                     double *work)
{
    int nc = lay->n_wrench + lay->n_force;
    double *K = work, *L = K + (long)N * nu * NX, *Phi = L + (long)N * nu * nu, *s = Phi + (long)N * NX * NX;
    double *kappa = s + (long)N * NX;
    if (orc_factor_env(N, nu, A, Bm, c, Qd, Rd, rho, K, L, Phi, s, NULL)) return 1;
    double rp = 0.0, rd = 0.0, v[NU_MAX], zn[NU_MAX];
    int done = 0;
    for (int m = 0; m < iters; m++) {
        orc_eqstep_env(N, nu, A, Bm, c, K, L, Phi, s, Qd, Rd, rho, x0, x_ref, u_ref, z, y, x, u, kappa);
        rp = 0.0; rd = 0.0;
        double un = 0.0, znm = 0.0, yn = 0.0;
        for (int k = 0; k < N; k++) {
            double *uk = u + (long)k * nu, *zk = z + (long)k * nu, *yk = y + (long)k * nu;
            for (int j = 0; j < nu; j++) v[j] = uk[j] + yk[j];
            orc_project_stage(lay, nu, contact + (long)k * nc, v, zn);            /* step 4 */
            for (int j = 0; j < nu; j++) {
                yk[j] = yk[j] + uk[j] - zn[j];                                     /* step 5 */
                double a = fabs(uk[j] - zn[j]), b = fabs(zn[j] - zk[j]);           /* step 6 */
                if (a > rp) rp = a;
                if (b > rd) rd = b;
                zk[j] = zn[j];
                if (fabs(uk[j]) > un) un = fabs(uk[j]);
                if (fabs(zn[j]) > znm) znm = fabs(zn[j]);
                if (fabs(yk[j]) > yn) yn = fabs(yk[j]);
            }
        }
        rd *= rho;
        done = m + 1;
        if ((eps_abs > 0.0 || eps_rel > 0.0) && check_every > 0 && done % check_every == 0) {
            double sc = un > znm ? un : znm;
            if (rp <= eps_abs + eps_rel * sc && rd <= eps_abs + eps_rel * rho * yn) break;
        }
    }
    *r_prim = rp; *r_dual = rd; *iters_done = done;
    return 0;
}

/* Full batched solve.  Either A/Bm/c are given ([B,N,13,13],[B,N,13,nu],[B,N,13]; generic LTV)
 * or they are NULL and each env is assembled from (yaw, foot_r, mass, inertia, ext) first.
 * z,y [B,N,nu] are in/out (caller zero-fills for the cold start z0 = y0 = 0).  Outputs x[B,N,13]
 * (x_1..x_N) and u[B,N,nu] of the last equality step, r_prim/r_dual[B], iters_done[B].
 * OpenMP over envs, schedule(static).  Returns the number of envs whose factorisation failed. */
int orc_solve(int B, int N, int nu, const orc_layout *lay, double dt, double rho, int iters,
              double eps_abs, double eps_rel, int check_every, const double *Qd, const double *Rd,
              const double *x0, const double *x_ref, const double *u_ref, const unsigned char *contact,
              const double *A, const double *Bm, const double *c,
              const double *yaw, const double *foot_r, const double *mass, const double *inertia, const double *ext,
              double *x, double *u, double *z, double *y, double *r_prim, double *r_dual, int *iters_done,
              int nthreads)
{
    int nc = lay->n_wrench + lay->n_force, fails = 0;
    long wsz = (long)N * (nu * NX + nu * nu + NX * NX + NX + nu) + (long)N * (NX * NX + NX * nu + NX);
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(static) reduction(+ : fails)
    for (long b = 0; b < B; b++) {
        double *work = (double *)malloc(sizeof(double) * wsz);
        double *As = work + (long)N * (nu * NX + nu * nu + NX * NX + NX + nu);
        double *Bs = As + (long)N * NX * NX, *cs = Bs + (long)N * NX * nu;
        const double *Ab, *Bb, *cb;
        if (A) {
            Ab = A + b * N * NX * NX; Bb = Bm + b * N * NX * nu; cb = c + b * N * NX;
        } else {
            orc_assemble(1, N, nu, lay->n_wrench, lay->n_force, dt, yaw + b * N, foot_r + b * N * nc * 3,
                         mass + b, inertia + b * 9, ext ? ext + b * N * 6 : NULL, As, Bs, cs);
            Ab = As; Bb = Bs; cb = cs;
        }
        fails += solve_env(N, nu, lay, rho, iters, eps_abs, eps_rel, check_every, Qd, Rd, Ab, Bb, cb,
                           x0 + b * NX, x_ref + b * N * NX, u_ref ? u_ref + b * N * nu : NULL,
                           contact + b * N * nc, x + b * N * NX, u + b * N * nu, z + b * N * nu, y + b * N * nu,
                           r_prim + b, r_dual + b, iters_done + b, work);
        free(work);
    }
    return fails;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
