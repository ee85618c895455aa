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
never updated (in the gamma terms of stage 0 it enters as a constant); all iterates start at 0; X_k = R^nx unless a
box is given (x_lo, x_hi), so the projection acts on the u part (the set of stage k, since xi_{k+1} carries u_k) and
clips the x part to the box.

Variable scaling (PAPER.md:L184 leaves rho and the units open; with one scalar rho the iteration stalls on
the SRB problem's units).  `scale_x` (nx positive numbers) and `scale_u` (one positive number) define x = Sx x~,
u = su u~; the iteration above runs on the problem in (x~, u~):
    A~ = Sx^-1 A Sx,  B~ = su Sx^-1 B,  e~ = Sx^-1 e,  Q~ = Sx^2 Q,  R~ = su^2 R,  refs and xi_0 divided by the scales,
    U~_k = U_k / su, projected onto through Proj_{U/s}(v) = Proj_U(s v) / s (one scalar for all inputs keeps the
    projection Euclidean in the scaled variables),
and every returned vector is scaled back.  The limit is the optimum of the same QP; the iterates differ.

Nesterov acceleration with restart (PAPER.md:L210 Remark 3 defers to [23], [27]; neither is in the container).
Reading: "fast ADMM with restart" as published by Goldstein, O'Donoghue, Setzer and Baraniuk (2014),
restated from memory, applied to the block that is updated second and to the scaled duals, w = (z, v, theta, beta, lam):
    iteration m runs (22) from the extrapolated point w^_m and yields w_m;
    c_m = rho (|theta_m - theta^_m|^2 + |beta_m - beta^_m|^2 + |lam_m - lam^_m|^2)
        + rho (|dz|^2 + |dv|^2 + |dz - dv|^2),  dz = z_m - z^_m, dv = v_m - v^_m   (the second block enters (20b), (20c), (20d)
                                                                                   as -z, -v, z - v)
    if c_m < eta c_{m-1}:  a_{m+1} = (1 + sqrt(1 + 4 a_m^2)) / 2,  w^_{m+1} = w_m + (a_m - 1) / a_{m+1} (w_m - w_{m-1})
    else (restart):        a_{m+1} = 1,  w^_{m+1} = w_{m-1},  c_m <- c_{m-1} / eta
with a_1 = 1, c_0 = +inf, w_0 = w^_1 = the start, eta = 0.999; sums over all stages of the env.
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


def solve_env(A, Bm, e, Qd, Rd, rho, iters, x0, u_prev, x_ref, u_ref, project_u, state=None, scale_x=None, scale_u=1.0,
              accel=False, eta=0.999, trace=None, x_lo=None, x_hi=None):
    """project_u(k, v[nu]) -> Proj_{U_k}(v) in the caller's units.  Returns dict(xi[N,n], z[N,n], du[N,nu], v, theta, beta, lam, r_prim[, restarts, c]) in the caller's units.

    xi[k] = xi_{k+1} = [x_{k+1}; u_k].  r_prim = max_k |xi_{k+1} - z_{k+1}|_inf of the last iteration (scaled variables).
    trace: optional list, receives (xi, z) in the caller's units after every iteration.
    x_lo, x_hi [nx] (caller's units, +-inf allowed): the state set X_k of (17) as a box, xi_{k+1} in X_k; the projection of
    (21b) then clips the x part of z (Xb_k = X_k x U_k)."""
    A = np.asarray(A, dtype=np.float64); Bm = np.asarray(Bm, dtype=np.float64); e = np.asarray(e, dtype=np.float64)
    N, nx, nu = Bm.shape
    n = nx + nu
    sx = np.ones(nx) if scale_x is None else np.asarray(scale_x, dtype=np.float64)
    su = float(scale_u)
    S = np.concatenate([sx, np.full(nu, su)])                     # xi = S xi~
    A = A / sx[None, :, None] * sx[None, None, :]
    Bm = Bm / sx[None, :, None] * su
    e = e / sx[None, :]
    Qb = np.concatenate([np.asarray(Qd, dtype=np.float64) * sx ** 2, np.asarray(Rd, dtype=np.float64) * su ** 2])
    qb = np.concatenate([Qb[:nx] * (np.asarray(x_ref, dtype=np.float64) / sx), Qb[nx:] * (np.asarray(u_ref, dtype=np.float64) / su)], axis=1)
    Ab, Bb, eb = lifted(A, Bm, e)
    J, H = factors(Ab, Bb, Qb, rho)
    xi0 = np.concatenate([np.asarray(x0, dtype=np.float64) / sx, np.asarray(u_prev, dtype=np.float64) / su])
    proj = (lambda k, v: project_u(k, su * v) / su) if su != 1.0 else project_u      # Proj_{U/s}(v) = Proj_U(s v) / s
    if state is None:
        z = np.zeros((N, n)); v = np.zeros((N, n)); theta = np.zeros((N, n)); beta = np.zeros((N, n)); lam = np.zeros((N, n))
    else:
        z, v, theta, beta, lam = (np.array(state[k], dtype=np.float64) / S for k in ("z", "v", "theta", "beta", "lam"))
    xi = np.zeros((N, n)); du = np.zeros((N, nu))
    r_prim = 0.0
    names = ("z", "v", "theta", "beta", "lam")
    w_prev = dict(z=z.copy(), v=v.copy(), theta=theta.copy(), beta=beta.copy(), lam=lam.copy())      # w_{m-1}
    alpha, c_prev, restarts, c_hist, margin = 1.0, np.inf, 0, [], np.inf
    for _ in range(iters):
        hat = dict(z=z.copy(), v=v.copy(), theta=theta.copy(), beta=beta.copy(), lam=lam.copy())     # w^_m: (22) starts here
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
            zn[k, :nx] = w[:nx] if x_lo is None else np.clip(w[:nx], np.asarray(x_lo, dtype=np.float64) / sx, np.asarray(x_hi, dtype=np.float64) / sx)
            zn[k, nx:] = proj(k, w[nx:])
            vn[k] = 0.5 * (zn[k] + gamma)
            theta[k] = theta[k] + xi[k] - zn[k]
            beta[k] = beta[k] + Bdu - vn[k]
            lam[k] = lam[k] + zn[k] - Axi - vn[k] - eb[k]
        z, v = zn, vn
        r_prim = float(np.max(np.abs(xi - z)))
        if trace is not None:
            trace.append((xi * S, z * S))
        if accel:
            w_m = dict(z=z, v=v, theta=theta, beta=beta, lam=lam)
            dz, dv = z - hat["z"], v - hat["v"]
            c_m = rho * sum(float(np.sum((w_m[k] - hat[k]) ** 2)) for k in ("theta", "beta", "lam")) \
                + rho * float(np.sum(dz ** 2) + np.sum(dv ** 2) + np.sum((dz - dv) ** 2))
            if np.isfinite(c_prev):
                margin = min(margin, abs(c_m - eta * c_prev) / max(c_m, eta * c_prev, 1e-300))   # how close the decision was
            if c_m < eta * c_prev:
                a_next = 0.5 * (1.0 + np.sqrt(1.0 + 4.0 * alpha * alpha))
                mom = (alpha - 1.0) / a_next
                nxt = {k: w_m[k] + mom * (w_m[k] - w_prev[k]) for k in names}
                alpha, c_prev = a_next, c_m
            else:
                restarts += 1
                nxt = {k: w_prev[k].copy() for k in names}
                alpha, c_prev = 1.0, c_prev / eta
            c_hist.append(c_prev)
            w_prev = {k: w_m[k].copy() for k in names}
            if _ < iters - 1:                                   # the returned iterate is w_M itself
                z, v, theta, beta, lam = (nxt[k] for k in names)
    out = dict(xi=xi * S, z=z * S, du=du * su, v=v * S, theta=theta * S, beta=beta * S, lam=lam * S, r_prim=r_prim)
    if accel:
        out.update(restarts=restarts, c=np.array(c_hist), margin=margin)
    return out
