"""Independent numpy/scipy codings used to PIN the oracle (never used by the oracle or the CUDA path).

Each function here is a second, differently-structured statement of something the paper or the
mathematics fixes, so that a mistake in oracle/pinmpc_oracle.c (a dropped term, a wrong sign or
index, a transposed operand) shows up as a disagreement:

  srb_ode / euler_step      continuous single-rigid-body ODE of BASELINE.json config 0 + forward Euler
  kkt_eqstep                dense KKT system of the equality-constrained step (eq. (16), (21a))
  riccati_lqr_textbook      sequential Riccati LQR in the "+p" textbook form with np.linalg.solve
  brute_project_wrench      enumeration of all faces of the foot wrench set
  dense_qp / active_set_qp  condensed QP (16)-(17) with a KKT-certificate active-set solve
"""
from __future__ import annotations

import itertools

import numpy as np

NX = 13


# ---------------------------------------------------------------------------------------------
# dynamics: the continuous ODE as BASELINE.json config 0 words it
# ---------------------------------------------------------------------------------------------
def rotz(psi):
    c, s = np.cos(psi), np.sin(psi)
    return np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])


def srb_ode(x, u, yaw, r, mass, Ib, n_wrench, n_force, ext=None):
    """d/dt of x = [Theta, p, omega, v, g]:  dTheta = R_z(yaw)^T omega, dp = v,
    domega = I_w^{-1} sum(r_i x f_i + m_i), dv = sum f_i / m + g e_z, dg = 0."""
    Rz = rotz(yaw)
    Iw = Rz @ Ib @ Rz.T
    omega, v, g = x[6:9], x[9:12], x[12]
    tau = np.zeros(3); F = np.zeros(3)
    for i in range(n_wrench):
        f = u[3 * i:3 * i + 3]; m = u[3 * n_wrench + 3 * i:3 * n_wrench + 3 * i + 3]
        tau += np.cross(r[i], f) + m; F += f
    for j in range(n_force):
        f = u[6 * n_wrench + 3 * j:6 * n_wrench + 3 * j + 3]
        tau += np.cross(r[n_wrench + j], f); F += f
    if ext is not None:
        F = F + ext[:3]; tau = tau + ext[3:]
    dx = np.zeros(NX)
    dx[0:3] = Rz.T @ omega
    dx[3:6] = v
    dx[6:9] = np.linalg.solve(Iw, tau)
    dx[9:12] = F / mass + np.array([0.0, 0.0, g])
    return dx


# ---------------------------------------------------------------------------------------------
# equality-constrained step, two independent ways
# ---------------------------------------------------------------------------------------------
def kkt_eqstep(A, Bm, c, Qd, Rd, rho, x0, x_ref, u_ref, z, y):
    """min sum 1/2|x_{k+1}-xbar_{k+1}|_Q^2 + 1/2|u_k-ubar_k|_R^2 + rho/2 |u_k - z_k + y_k|^2
    s.t. x_{k+1} = A_k x_k + B_k u_k + c_k, as ONE dense KKT system in v = [u_0,x_1,...,u_{N-1},x_N]."""
    N, nu = Bm.shape[0], Bm.shape[2]
    nv = N * (nu + NX); ne = N * NX
    H = np.zeros((nv, nv)); f = np.zeros(nv); G = np.zeros((ne, nv)); b = np.zeros(ne)
    iu = lambda k: k * (nu + NX)
    ix = lambda k: k * (nu + NX) + nu        # x_{k+1}
    for k in range(N):
        H[iu(k):iu(k) + nu, iu(k):iu(k) + nu] = np.diag(Rd + rho)
        f[iu(k):iu(k) + nu] = Rd * u_ref[k] + rho * (z[k] - y[k])
        H[ix(k):ix(k) + NX, ix(k):ix(k) + NX] = np.diag(Qd)
        f[ix(k):ix(k) + NX] = Qd * x_ref[k]
        G[k * NX:(k + 1) * NX, ix(k):ix(k) + NX] = np.eye(NX)
        G[k * NX:(k + 1) * NX, iu(k):iu(k) + nu] = -Bm[k]
        if k == 0:
            b[:NX] = A[0] @ x0 + c[0]
        else:
            G[k * NX:(k + 1) * NX, ix(k - 1):ix(k - 1) + NX] = -A[k]
            b[k * NX:(k + 1) * NX] = c[k]
    KKT = np.block([[H, G.T], [G, np.zeros((ne, ne))]])
    sol = np.linalg.solve(KKT, np.concatenate([f, b]))
    v = sol[:nv].reshape(N, nu + NX)
    return v[:, nu:], v[:, :nu]            # x_1..x_N, u_0..u_{N-1}


def riccati_lqr_textbook(A, Bm, c, Qd, Rdiag_total, x0, x_ref, lin_u):
    """Sequential Riccati for  min sum 1/2 x_{k+1}^T Q x_{k+1} - (Q xbar_{k+1})^T x_{k+1}
    + 1/2 u_k^T Rt u_k - lin_u_k^T u_k  with V_k(x) = 1/2 x^T P x + p^T x ("+p" convention),
    P_k = Q + A^T P A - A^T P B (Rt + B^T P B)^{-1} B^T P A, np.linalg.solve everywhere."""
    N, nu = Bm.shape[0], Bm.shape[2]
    Q = np.diag(Qd); Rt = np.diag(Rdiag_total)
    P = Q.copy(); p = -(Qd * x_ref[N - 1])
    Ks = [None] * N; ks = [None] * N
    for k in range(N - 1, -1, -1):
        Ak, Bk, ck = A[k], Bm[k], c[k]
        M = Rt + Bk.T @ P @ Bk
        Ks[k] = np.linalg.solve(M, Bk.T @ P @ Ak)
        ks[k] = np.linalg.solve(M, Bk.T @ (P @ ck + p) - lin_u[k])       # u = -K x - k
        Pn = Ak.T @ P @ Ak - Ak.T @ P @ Bk @ Ks[k]
        pn = Ak.T @ (P @ ck + p) - Ks[k].T @ (Bk.T @ (P @ ck + p) - lin_u[k])
        if k >= 1:
            Pn = Pn + Q; pn = pn - Qd * x_ref[k - 1]
        P, p = Pn, pn
    xs = np.zeros((N, NX)); us = np.zeros((N, nu)); xk = np.array(x0, dtype=float)
    for k in range(N):
        us[k] = -Ks[k] @ xk - ks[k]
        xk = A[k] @ xk + Bm[k] @ us[k] + c[k]
        xs[k] = xk
    return xs, us


# ---------------------------------------------------------------------------------------------
# projection: enumerate every face of the foot wrench set
# ---------------------------------------------------------------------------------------------
def brute_project_wrench(f, m, mu, fz_max, ax, ay, b):
    """Euclidean projection of (f,m) onto {|f_x|,|f_y|<=mu t, |m_x|<=ax t, |m_y|<=ay t, |m_z|<=b t,
    0<=t<=fz_max}, t=f_z, by enumerating all 3^5 * 3 sign/active patterns: each pattern fixes a
    face, the least-squares point on that face is closed-form, the projection is the nearest
    feasible candidate."""
    a = np.array([f[0], f[1], m[0], m[1], m[2]], dtype=float)
    w = np.array([mu, mu, ax, ay, b], dtype=float)
    t0 = float(f[2])
    best, best_d = None, np.inf
    for sig in itertools.product((0, 1, -1), repeat=5):
        sig = np.array(sig, dtype=float)
        cl = sig != 0
        for tmode in ("free", "zero", "cap"):
            if tmode == "free":
                t = (t0 + np.sum(sig[cl] * w[cl] * a[cl])) / (1.0 + np.sum(w[cl] ** 2))
            elif tmode == "zero":
                t = 0.0
            else:
                t = fz_max
            v = np.where(cl, sig * w * t, a)
            if t < -1e-13 or t > fz_max + 1e-13 or np.any(np.abs(v) > w * t + 1e-12):
                continue
            d = (t - t0) ** 2 + np.sum((v - a) ** 2)
            if d < best_d:
                best_d, best = d, (v.copy(), t)
    v, t = best
    return np.array([v[0], v[1], t]), np.array([v[2], v[3], v[4]])


def wrench_set_inequalities(mu, fz_max, ax, ay, b):
    """C v <= d for v = (f_x,f_y,f_z,m_x,m_y,m_z): 12 rows."""
    rows, rhs = [], []
    for idx, wgt in ((0, mu), (1, mu), (3, ax), (4, ay), (5, b)):
        for sgn in (1.0, -1.0):
            r = np.zeros(6); r[idx] = sgn; r[2] = -wgt
            rows.append(r); rhs.append(0.0)
    r = np.zeros(6); r[2] = -1.0; rows.append(r); rhs.append(0.0)
    r = np.zeros(6); r[2] = 1.0; rows.append(r); rhs.append(fz_max)
    return np.array(rows), np.array(rhs)


# ---------------------------------------------------------------------------------------------
# the whole QP (16)-(17), condensed, with an exact active-set solve
# ---------------------------------------------------------------------------------------------
def condense(A, Bm, c, x0):
    """x_{1:N} = S U + d for U = (u_0..u_{N-1})."""
    N, nu = Bm.shape[0], Bm.shape[2]
    S = np.zeros((N * NX, N * nu)); d = np.zeros(N * NX)
    xk = np.array(x0, dtype=float)
    for k in range(N):
        xk = A[k] @ xk + c[k]
        d[k * NX:(k + 1) * NX] = xk
        for j in range(k + 1):
            blk = Bm[j]
            for l in range(j + 1, k + 1):
                blk = A[l] @ blk
            S[k * NX:(k + 1) * NX, j * nu:(j + 1) * nu] = blk
    return S, d


def dense_qp(w, env, A, Bm, c):
    """(H, g, C, dvec, Aeq) of  min 1/2 U^T H U + g^T U  s.t. C U <= dvec, U[eq_zero] = 0."""
    N, nu, nw, nf = w.N, w.nu, w.n_wrench, w.n_force
    Qd = w.Qdiag.astype(float); Rd = w.Rdiag.astype(float)
    S, d = condense(A, Bm, c, w.x0[env].astype(float))
    Qb = np.kron(np.eye(N), np.diag(Qd)); Rb = np.kron(np.eye(N), np.diag(Rd))
    xr = w.x_ref[env].astype(float).reshape(-1); ur = w.u_ref[env].astype(float).reshape(-1)
    H = S.T @ Qb @ S + Rb
    g = S.T @ Qb @ (d - xr) - Rb @ ur
    C6, d6 = wrench_set_inequalities(w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef)
    rows, rhs, zero_idx = [], [], []
    for k in range(N):
        for i in range(nw):
            idx = [k * nu + 3 * i + a for a in range(3)] + [k * nu + 3 * nw + 3 * i + a for a in range(3)]
            if w.contact[env, k, i]:
                for r6, h6 in zip(C6, d6):
                    r = np.zeros(N * nu); r[idx] = r6
                    rows.append(r); rhs.append(h6)
            else:
                zero_idx += idx
        for j in range(nf):
            idx = [k * nu + 6 * nw + 3 * j + a for a in range(3)]
            if w.contact[env, k, nw + j]:
                for ii in idx:
                    for sgn in (1.0, -1.0):
                        r = np.zeros(N * nu); r[ii] = sgn
                        rows.append(r); rhs.append(w.hand_fmax)
            else:
                zero_idx += idx
    return H, g, np.array(rows), np.array(rhs), np.array(sorted(zero_idx), dtype=int)


def active_set_qp(H, g, C, dvec, zero_idx, U_init, tol=1e-9, max_iter=500):
    """Primal active-set method for the strictly convex QP; returns (U, multipliers, active set).
    The result is certified by its KKT conditions in the caller, so the route taken is immaterial."""
    n = H.shape[0]
    free = np.setdiff1d(np.arange(n), zero_idx)
    Hf = H[np.ix_(free, free)]; gf = g[free]; Cf = C[:, free]
    u = U_init[free].copy()
    act = []

    def eq_solve(active):
        if len(active) == 0:
            return np.linalg.solve(Hf, -gf), np.zeros(0)
        Ca = Cf[active]
        KKT = np.block([[Hf, Ca.T], [Ca, np.zeros((len(active), len(active)))]])
        sol = np.linalg.lstsq(KKT, np.concatenate([-gf, dvec[active]]), rcond=None)[0]
        return sol[:len(free)], sol[len(free):]

    if np.any(Cf @ u > dvec + 1e-9):
        raise ValueError("active_set_qp needs a feasible start")
    for _ in range(max_iter):
        ustar, lam = eq_solve(act)
        step = ustar - u
        if np.linalg.norm(step) < tol:
            if len(act) == 0 or lam.min() >= -tol:
                break
            act.pop(int(np.argmin(lam)))
            continue
        Cs = Cf @ step
        slack = dvec - Cf @ u
        alpha, block = 1.0, -1
        for i in np.where(Cs > 1e-14)[0]:
            if i in act:
                continue
            a = slack[i] / Cs[i]
            if a < alpha:
                alpha, block = a, i
        u = u + alpha * step
        if block >= 0:
            act.append(int(block))
    U = np.zeros(n); U[free] = u
    lam_full = np.zeros(C.shape[0])
    _, lam = eq_solve(act)
    lam_full[act] = lam
    return U, lam_full, act
