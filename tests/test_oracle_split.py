"""Pins of oracle/split.py (the paper's stage-local ADMM, eq. (18)-(22)).

What the mathematics fixes: the iteration is an ADMM on problem (20), which is the QP (16)-(17) rewritten, so its
limit is that QP's unique optimum (computed here by an independent condensed bounded least-squares solve and by
the dense KKT system); and the joint (z, v) minimisation of (21b) leaves beta + lambda = 0 on every component
and theta = lambda wherever the projection is inactive, after every iteration.
"""
import numpy as np
import pytest
from scipy.optimize import lsq_linear

from oracle import split
from refcheck import kkt_eqstep


def condense(A, Bm, c, x0):
    """x_{1:N} = S U + d for U = (u_0..u_{N-1}), any nx."""
    N, nx, nu = Bm.shape
    S = np.zeros((N * nx, N * nu)); d = np.zeros(N * nx)
    xk = np.array(x0, dtype=float)
    for k in range(N):
        xk = A[k] @ xk + c[k]
        d[k * nx:(k + 1) * nx] = xk
        if k > 0:
            S[k * nx:(k + 1) * nx] = A[k] @ S[(k - 1) * nx:k * nx]
        S[k * nx:(k + 1) * nx, k * nu:(k + 1) * nu] = Bm[k]
    return S, d


def random_ltv(rng, N, nx, nu, e_scale=0.3):
    A = np.eye(nx) + 0.2 * rng.normal(size=(N, nx, nx))
    Bm = 0.5 * rng.normal(size=(N, nx, nu))
    e = e_scale * rng.normal(size=(N, nx))          # time-varying offset: exercises the e_{k+1} reading (D4)
    return A, Bm, e


def box_qp_optimum(A, Bm, e, Qd, Rd, x0, x_ref, u_ref, lo, hi):
    """min sum 1/2|x_{k+1}-xbar|_Q^2 + 1/2|u_k-ubar|_R^2, lo <= u <= hi, by condensing and bounded least squares."""
    N, nx, nu = Bm.shape
    S, d = condense(A, Bm, e, x0)                    # X = S U + d
    Wq = np.kron(np.eye(N), np.diag(np.sqrt(Qd))); Wr = np.kron(np.eye(N), np.diag(np.sqrt(Rd)))
    M = np.vstack([Wq @ S, Wr]); b = np.concatenate([Wq @ (x_ref.reshape(-1) - d), Wr @ u_ref.reshape(-1)])
    res = lsq_linear(M, b, bounds=(np.tile(lo, N), np.tile(hi, N)), method="bvls", tol=1e-14, max_iter=1000)
    U = res.x
    return (S @ U + d).reshape(N, nx), U.reshape(N, nu)


def run(seed, N, nx, nu, iters, lo=None, hi=None, rho=1.0, e_scale=0.3):
    rng = np.random.default_rng(seed)
    A, Bm, e = random_ltv(rng, N, nx, nu, e_scale)
    Qd = rng.uniform(0.5, 2.0, nx); Rd = rng.uniform(0.1, 0.5, nu)
    x0 = rng.normal(size=nx); u_prev = rng.normal(size=nu)
    x_ref = rng.normal(size=(N, nx)); u_ref = 0.2 * rng.normal(size=(N, nu))
    proj = (lambda k, v: v) if lo is None else (lambda k, v: np.clip(v, lo, hi))
    out = split.solve_env(A, Bm, e, Qd, Rd, rho, iters, x0, u_prev, x_ref, u_ref, proj)
    return dict(A=A, Bm=Bm, e=e, Qd=Qd, Rd=Rd, x0=x0, x_ref=x_ref, u_ref=u_ref), out


def test_unconstrained_limit_is_the_kkt_solution():
    N, nx, nu = 5, 3, 2
    p, out = run(1, N, nx, nu, 6000)
    import refcheck
    refcheck.NX, old = nx, refcheck.NX
    try:
        x, u = kkt_eqstep(p["A"], p["Bm"], p["e"], p["Qd"], p["Rd"], 0.0, p["x0"], p["x_ref"], p["u_ref"],
                          np.zeros((N, nu)), np.zeros((N, nu)))
    finally:
        refcheck.NX = old
    assert np.abs(out["xi"][:, :nx] - x).max() < 1e-8
    assert np.abs(out["xi"][:, nx:] - u).max() < 1e-8
    assert out["r_prim"] < 1e-9


@pytest.mark.parametrize("seed", [2, 3])
def test_box_constrained_limit_is_the_qp_optimum(seed):
    N, nx, nu = 6, 3, 2
    lo, hi = np.array([-0.3, -0.1]), np.array([0.2, 0.4])
    p, out = run(seed, N, nx, nu, 20000, lo, hi)
    x, u = box_qp_optimum(p["A"], p["Bm"], p["e"], p["Qd"], p["Rd"], p["x0"], p["x_ref"], p["u_ref"], lo, hi)
    assert np.sum((u <= lo + 1e-9) | (u >= hi - 1e-9)) >= 3          # the bounds are active somewhere
    assert np.abs(out["z"][:, nx:] - u).max() < 1e-6
    assert np.abs(out["z"][:, :nx] - x).max() < 1e-6
    assert np.abs(out["xi"] - out["z"]).max() < 1e-6
    assert np.all(out["z"][:, nx:] >= lo - 1e-15) and np.all(out["z"][:, nx:] <= hi + 1e-15)


def test_constant_offset_limit():
    """Constant offsets e_k = e (the case where the printed e_k and the adopted e_{k+1} inside h_k coincide).  The
    tests above use offsets that change from stage to stage, so they pin the adopted reading: with
    e_k as printed the limit is a different point."""
    N, nx, nu = 5, 3, 2
    rng = np.random.default_rng(7)
    A, Bm, _ = random_ltv(rng, N, nx, nu)
    e = np.tile(0.3 * rng.normal(size=nx), (N, 1))                   # constant offset: readings coincide
    Qd = np.ones(nx); Rd = 0.3 * np.ones(nu)
    x0 = rng.normal(size=nx); x_ref = rng.normal(size=(N, nx)); u_ref = np.zeros((N, nu))
    out = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 6000, x0, np.zeros(nu), x_ref, u_ref, lambda k, v: v)
    x, u = box_qp_optimum(A, Bm, e, Qd, Rd, x0, x_ref, u_ref, np.full(nu, -1e6), np.full(nu, 1e6))
    assert np.abs(out["xi"][:, nx:] - u).max() < 1e-7


@pytest.mark.parametrize("iters", [1, 2, 17])
def test_invariants_of_the_zv_update(iters):
    N, nx, nu = 7, 4, 3
    lo, hi = np.full(nu, -0.05), np.full(nu, 0.05)
    _, out = run(11, N, nx, nu, iters, lo, hi)
    assert np.abs(out["beta"] + out["lam"]).max() < 1e-12            # stationarity in v
    assert np.abs(out["theta"][:, :nx] - out["lam"][:, :nx]).max() < 1e-12   # stationarity in z, free components
    zu = out["z"][:, nx:]
    free = (zu > lo + 1e-12) & (zu < hi - 1e-12)
    d = (out["theta"][:, nx:] - out["lam"][:, nx:])
    assert np.abs(d[free]).max() < 1e-12 if free.any() else True
    assert (~free).any()                                             # and the projection was active somewhere
    # v_k = Bb_k du_k + beta_k^{old} - beta_k^{new}: the (20c) dual update, re-read from the outputs
    assert out["v"].shape == (N, nx + nu)


def test_u_prev_does_not_change_the_limit_but_enters_stage_0():
    N, nx, nu = 4, 3, 2
    rng = np.random.default_rng(5)
    A, Bm, e = random_ltv(rng, N, nx, nu)
    Qd = np.ones(nx); Rd = 0.2 * np.ones(nu); x0 = rng.normal(size=nx)
    x_ref = rng.normal(size=(N, nx)); u_ref = np.zeros((N, nu))
    a = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 5000, x0, np.zeros(nu), x_ref, u_ref, lambda k, v: v)
    b = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 5000, x0, np.ones(nu), x_ref, u_ref, lambda k, v: v)
    assert np.abs(a["xi"] - b["xi"]).max() < 1e-8                    # no cost on du: the optimum ignores u_{-1}
    assert np.abs(a["du"][0] - b["du"][0] - 1.0).max() < 1e-7        # du_0 = u_0 - u_{-1}
    a1 = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 1, x0, np.zeros(nu), x_ref, u_ref, lambda k, v: v)
    b1 = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 1, x0, np.ones(nu), x_ref, u_ref, lambda k, v: v)
    assert np.abs(a1["z"][0] - b1["z"][0]).max() > 1e-3
