"""float64 oracle of the paper's own stage-local ADMM (pi^n MPC proper) — TEST INFRASTRUCTURE ONLY.

PAPER.md:L152-202, eq. (18)-(22): velocity form, auxiliary copies z_{k+1} = xi_{k+1} and v_k = Bb_k du_k, the
dynamics relaxed with a third dual, closed-form updates that are local to a stage.  Only
tests/ may import this; it shares no code with paper_2606_05687_b200 and never imports it.

One env, generic LTV data A[N,nx,nx], Bm[N,nx,nu], e[N,nx].  Notation of the paper (bars dropped):

  lifted state   xi_k = [x_k ; u_{k-1}] in R^n, n = nx + nu                                   eq. (18)
  Ab_k = [[A_k, B_k],[0, I]],  Bb_k = [B_k ; I],  eb_k = [e_k ; 0]                              eq. (19)
  cost           sum_k 1/2 xi_{k+1}^T Qb xi_{k+1} - qb_k^T xi_{k+1},  Qb = diag(Q, R), qb_k = [Q xbar_{k+1}; R ubar_k]
  J_k = (Bb_k^T Bb_k)^-1 Bb_k^T ;  H_k = (Qb + rho I + rho Ab_{k+1}^T Ab_{k+1})^-1 (k < N-1), (Qb + rho I)^-1 (k = N-1)

  iteration m+1 (every k independently inside a phase):                                        eq. (22)
    du_k      = J_k (v_k - beta_k)
    h_k       = qb_k + rho (z_{k+1} - theta_k) [+ rho Ab_{k+1}^T (z_{k+2} - v_{k+1} - eb_{k+1} + lam_{k+1}), k < N-1]
    xi_{k+1}  = H_k h_k
    gamma_k   = Bb_k du_k + beta_k - Ab_k xi_k - eb_k + lam_k
    gammat_k  = xi_{k+1} + theta_k + Ab_k xi_k + eb_k - lam_k
    z_{k+1}   = Proj_{X x U_k}((2 gammat_k + gamma_k) / 3)
    v_k       = (z_{k+1} + gamma_k) / 2
    theta_k  += xi_{k+1} - z_{k+1} ;  beta_k += Bb_k du_k - v_k ;  lam_k += z_{k+1} - Ab_k xi_k - v_k - eb_k

Readings: the paper prints eb_k inside the Ab_{k+1}^T term of h_k; stationarity of the (20d)
term of stage k+1 requires eb_{k+1} and that is what is used; xi_0 = [x_0 ; u_{-1}] is data and
never updated (in the gamma terms of stage 0 it enters as a constant); all iterates start at 0; X_k = R^nx, so the
projection acts on the u part only (the set of stage k, since xi_{k+1} carries u_k); no Nesterov acceleration.
"""
from __future__ import annotations

import numpy as np


def lifted(A, Bm, e):
    N, nx, nu = Bm.shape
    n = nx + nu
    Ab = np.zeros((N, n, n)); Bb = np.zeros((N, n, nu)); eb = np.zeros((N, n))
    for k in range(N):
        Ab[k, :nx, :nx] = A[k]; Ab[k, :nx, nx:] = Bm[k]; Ab[k, nx:, nx:] = np.eye(nu)
        Bb[k, :nx] = Bm[k]; Bb[k, nx:] = np.eye(nu)
        eb[k, :nx] = e[k]
    return Ab, Bb, eb


def factors(Ab, Bb, Qb, rho):
    N, n, nu = Bb.shape
    J = np.zeros((N, nu, n)); H = np.zeros((N, n, n))
    for k in range(N):
        J[k] = np.linalg.solve(Bb[k].T @ Bb[k], Bb[k].T)
        M = np.diag(Qb + rho)
        if k < N - 1:
            M = M + rho * Ab[k + 1].T @ Ab[k + 1]
        H[k] = np.linalg.inv(M)
    return J, H


def solve_env(A, Bm, e, Qd, Rd, rho, iters, x0, u_prev, x_ref, u_ref, project_u, state=None):
    """project_u(k, v[nu]) -> Proj_{U_k}(v).  Returns dict(xi[N,n], z[N,n], du[N,nu], v, theta, beta, lam, r_prim).

    xi[k] = xi_{k+1} = [x_{k+1}; u_k].  r_prim = max_k |xi_{k+1} - z_{k+1}|_inf of the last iteration."""
    A = np.asarray(A, dtype=np.float64); Bm = np.asarray(Bm, dtype=np.float64); e = np.asarray(e, dtype=np.float64)
    N, nx, nu = Bm.shape
    n = nx + nu
    Qb = np.concatenate([np.asarray(Qd, dtype=np.float64), np.asarray(Rd, dtype=np.float64)])
    qb = np.concatenate([Qb[:nx] * np.asarray(x_ref, dtype=np.float64), Qb[nx:] * np.asarray(u_ref, dtype=np.float64)], axis=1)
    Ab, Bb, eb = lifted(A, Bm, e)
    J, H = factors(Ab, Bb, Qb, rho)
    xi0 = np.concatenate([np.asarray(x0, dtype=np.float64), np.asarray(u_prev, dtype=np.float64)])
    if state is None:
        z = np.zeros((N, n)); v = np.zeros((N, n)); theta = np.zeros((N, n)); beta = np.zeros((N, n)); lam = np.zeros((N, n))
    else:
        z, v, theta, beta, lam = (np.array(state[k], dtype=np.float64) for k in ("z", "v", "theta", "beta", "lam"))
    xi = np.zeros((N, n)); du = np.zeros((N, nu))
    r_prim = 0.0
    for _ in range(iters):
        # (21a): every k from the previous iterates
        for k in range(N):
            du[k] = J[k] @ (v[k] - beta[k])
            h = qb[k] + rho * (z[k] - theta[k])
            if k < N - 1:
                h = h + rho * Ab[k + 1].T @ (z[k + 1] - v[k + 1] - eb[k + 1] + lam[k + 1])
            xi[k] = H[k] @ h
        # (21b), (21c): every k from the new xi, du
        zn = np.zeros_like(z); vn = np.zeros_like(v)
        for k in range(N):
            xik = xi0 if k == 0 else xi[k - 1]
            Axi = Ab[k] @ xik
            Bdu = Bb[k] @ du[k]
            gamma = Bdu + beta[k] - Axi - eb[k] + lam[k]
            gammat = xi[k] + theta[k] + Axi + eb[k] - lam[k]
            w = (2.0 * gammat + gamma) / 3.0
            zn[k, :nx] = w[:nx]
            zn[k, nx:] = project_u(k, w[nx:])
            vn[k] = 0.5 * (zn[k] + gamma)
            theta[k] = theta[k] + xi[k] - zn[k]
            beta[k] = beta[k] + Bdu - vn[k]
            lam[k] = lam[k] + zn[k] - Axi - vn[k] - eb[k]
        z, v = zn, vn
        r_prim = float(np.max(np.abs(xi - z)))
    return dict(xi=xi, z=z, du=du, v=v, theta=theta, beta=beta, lam=lam, r_prim=r_prim)
