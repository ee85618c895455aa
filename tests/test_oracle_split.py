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


# ---------------------------------------------------------------------------------------------------------------
# Variable scaling and accelerated iteration with restart (oracle/split.py header)
# ---------------------------------------------------------------------------------------------------------------
def _box_problem(seed, N=6, nx=3, nu=2):
    rng = np.random.default_rng(seed)
    A, Bm, e = random_ltv(rng, N, nx, nu)
    Qd = rng.uniform(0.5, 2.0, nx); Rd = rng.uniform(0.1, 0.5, nu)
    x0 = rng.normal(size=nx); u_prev = rng.normal(size=nu)
    x_ref = rng.normal(size=(N, nx)); u_ref = 0.2 * rng.normal(size=(N, nu))
    lo, hi = np.array([-0.3, -0.1]), np.array([0.2, 0.4])
    return A, Bm, e, Qd, Rd, x0, u_prev, x_ref, u_ref, lo, hi


def test_uniform_scaling_equals_the_unscaled_iteration_with_rho_over_s2():
    """x = s x~, u = s u~ with one s for everything: A~ = A, B~ = B, e~ = e / s, the cost is multiplied by s^2 and
    the set divided by s.  ADMM with penalty rho on s^2 f(s .) is ADMM with rho / s^2 on f, iterate by iterate: a
    closed-form consequence that fails if any of Q, R, the references, xi_0, the offsets or the set is scaled wrongly."""
    A, Bm, e, Qd, Rd, x0, u_prev, x_ref, u_ref, lo, hi = _box_problem(21)
    proj = lambda k, v: np.clip(v, lo, hi)
    s = 7.0
    for iters in (1, 2, 40):
        a = split.solve_env(A, Bm, e, Qd, Rd, 2.0, iters, x0, u_prev, x_ref, u_ref, proj, scale_x=np.full(3, s), scale_u=s)
        b = split.solve_env(A, Bm, e, Qd, Rd, 2.0 / s ** 2, iters, x0, u_prev, x_ref, u_ref, proj)
        for k in ("xi", "z", "v", "theta", "beta", "lam", "du"):
            assert np.abs(a[k] - b[k]).max() < 1e-11 * (1 + np.abs(b[k]).max()), k
    one = split.solve_env(A, Bm, e, Qd, Rd, 2.0, 9, x0, u_prev, x_ref, u_ref, proj, scale_x=np.ones(3), scale_u=1.0)
    ref = split.solve_env(A, Bm, e, Qd, Rd, 2.0, 9, x0, u_prev, x_ref, u_ref, proj)
    assert np.array_equal(one["z"], ref["z"])


def test_nonuniform_scaling_changes_the_iterates_but_not_the_limit():
    A, Bm, e, Qd, Rd, x0, u_prev, x_ref, u_ref, lo, hi = _box_problem(22)
    proj = lambda k, v: np.clip(v, lo, hi)
    x, u = box_qp_optimum(A, Bm, e, Qd, Rd, x0, x_ref, u_ref, lo, hi)
    sx, su = np.array([0.3, 2.0, 5.0]), 0.4
    few = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 3, x0, u_prev, x_ref, u_ref, proj, scale_x=sx, scale_u=su)
    ref = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 3, x0, u_prev, x_ref, u_ref, proj)
    assert np.abs(few["z"] - ref["z"]).max() > 1e-3
    out = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 30000, x0, u_prev, x_ref, u_ref, proj, scale_x=sx, scale_u=su)
    assert np.abs(out["z"][:, 3:] - u).max() < 1e-6 and np.abs(out["z"][:, :3] - x).max() < 1e-6
    assert np.all(out["z"][:, 3:] >= lo - 1e-12) and np.all(out["z"][:, 3:] <= hi + 1e-12)


def _srb_env(N=10):
    import gen
    import oracle
    w = gen.make_config(0, B=2, N=N)
    A, Bm, c = oracle.assemble(w.nu, w.n_wrench, w.n_force, w.dt, w.yaw, w.foot_r, w.mass, w.inertia, w.ext_wrench)
    c = np.zeros((w.B, w.N, 13)) if c is None else c
    lay = oracle.layout_of(w)
    b = 0
    proj = lambda k, v: oracle.project(lay, w.contact[b, k:k + 1], v[None])[0]
    star = oracle.solve(w, iters=20000, rho=1e-4)                 # the exact-dynamics ADMM at convergence (pinned by
    q = np.asarray(w.Qdiag, dtype=np.float64)                     # tests/test_oracle_converged.py against the dense QP)
    sx = 1.0 / np.sqrt(np.where(q > 0, q, 1.0))
    args = (A[b], Bm[b], c[b], w.Qdiag, w.Rdiag)
    rest = (w.x0[b], w.u_ref[b, 0], w.x_ref[b], w.u_ref[b], proj)
    return w, args, rest, sx, star["x"][b], star["u"][b]


def _err(out, xs, us):
    return max(np.abs(out["z"][:, 13:] - us).max() / (1 + np.abs(us).max()), np.abs(out["z"][:, :13] - xs).max() / (1 + np.abs(xs).max()))


def test_scaling_makes_the_srb_problem_converge_to_the_qp_optimum():
    """SRB config 0 (forces of 400 N with R = 1e-5 next to states of order 1 with Q up to 500): with rho = 1 and no
    scaling the iteration is still 90 % off after 1500 iterations; with Sx = Q^-1/2, su = 100 it reaches the optimum of
    the QP (the exact-dynamics oracle at convergence, itself pinned against the dense QP) — the iterations-to-tolerance pin."""
    w, args, rest, sx, xs, us = _srb_env()
    plain = split.solve_env(*args, 1.0, 1500, *rest)
    assert _err(plain, xs, us) > 0.5
    tr = []
    out = split.solve_env(*args, 1.0, 3000, *rest, scale_x=sx, scale_u=100.0, trace=tr)
    errs = np.array([max(np.abs(z[:, 13:] - us).max() / (1 + np.abs(us).max()), np.abs(z[:, :13] - xs).max() / (1 + np.abs(xs).max())) for _, z in tr])
    assert errs[-1] < 1e-5
    it2, it3 = int(np.argmax(errs < 1e-2)) + 1, int(np.argmax(errs < 1e-3)) + 1
    assert 300 < it2 < 900 and 700 < it3 < 1500, (it2, it3)      # measured: 593 and 1105 (accelerated with restart: 681 and 1225, 471 restarts)
    assert np.abs(out["xi"] - out["z"]).max() / (1 + np.abs(us).max()) < 1e-5


def test_accelerated_iteration_restart_rule_and_limit():
    A, Bm, e, Qd, Rd, x0, u_prev, x_ref, u_ref, lo, hi = _box_problem(23)
    proj = lambda k, v: np.clip(v, lo, hi)
    x, u = box_qp_optimum(A, Bm, e, Qd, Rd, x0, x_ref, u_ref, lo, hi)
    out = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 4000, x0, u_prev, x_ref, u_ref, proj, accel=True)
    c = out["c"]
    assert np.all(c[1:] <= c[:-1] / 0.999 * (1 + 1e-12))          # accepted steps decrease c, a restart divides it by eta
    assert 0 < out["restarts"] < 4000
    assert np.abs(out["z"][:, 3:] - u).max() < 1e-6 and np.abs(out["z"][:, :3] - x).max() < 1e-6
    # the first iteration has a_1 = 1: no momentum yet, identical to the plain iteration; the second differs only if
    # the first was accepted with a_2 > 1, i.e. from the third on
    p1 = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 2, x0, u_prev, x_ref, u_ref, proj)
    a1 = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 2, x0, u_prev, x_ref, u_ref, proj, accel=True)
    assert np.array_equal(p1["z"], a1["z"])
    p3 = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 3, x0, u_prev, x_ref, u_ref, proj)
    a3 = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 3, x0, u_prev, x_ref, u_ref, proj, accel=True)
    assert np.abs(p3["z"] - a3["z"]).max() > 1e-6


def test_accelerated_iteration_on_an_unconstrained_problem_is_faster():
    """Where the theory of the accelerated method applies best (strongly convex, no active set changes) it needs fewer
    iterations than the plain one for the same accuracy."""
    N, nx, nu = 5, 3, 2
    p, _ = run(1, N, nx, nu, 1)
    import refcheck
    refcheck.NX, old = nx, refcheck.NX
    try:
        x, u = kkt_eqstep(p["A"], p["Bm"], p["e"], p["Qd"], p["Rd"], 0.0, p["x0"], p["x_ref"], p["u_ref"], np.zeros((N, nu)), np.zeros((N, nu)))
    finally:
        refcheck.NX = old
    rng = np.random.default_rng(1)
    random_ltv(rng, N, nx, nu); rng.uniform(0.5, 2.0, nx); rng.uniform(0.1, 0.5, nu); rng.normal(size=nx)
    u_prev = rng.normal(size=nu)

    def iters_to(accel):
        tr = []
        split.solve_env(p["A"], p["Bm"], p["e"], p["Qd"], p["Rd"], 1.0, 1500, p["x0"], u_prev, p["x_ref"], p["u_ref"], lambda k, v: v,
                        accel=accel, trace=tr)
        errs = np.array([np.abs(z[:, nx:] - u).max() for _, z in tr])
        return int(np.argmax(errs < 1e-6)) + 1
    n_plain, n_acc = iters_to(False), iters_to(True)
    assert n_acc < n_plain, (n_plain, n_acc)


def test_state_box_limit_is_the_qp_optimum():
    """xi_{k+1} in X_k (a box on the states, eq. (17)) next to the input box: the limit equals the optimum of the
    condensed QP with linear inequality constraints on X = S U + d, solved by SLSQP and polished on its active set."""
    from scipy.optimize import minimize
    N, nx, nu = 5, 3, 2
    A, Bm, e, Qd, Rd, x0, u_prev, x_ref, u_ref, lo, hi = _box_problem(31, N, nx, nu)
    free = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 20000, x0, u_prev, x_ref, u_ref, lambda k, v: np.clip(v, lo, hi))
    xf = free["z"][:, :nx]
    x_lo = np.array([xf[:, 0].min() + 0.3 * np.ptp(xf[:, 0]), -np.inf, -np.inf])           # cuts into the free optimum
    x_hi = np.array([np.inf, xf[:, 1].max() - 0.3 * np.ptp(xf[:, 1]), np.inf])
    out = split.solve_env(A, Bm, e, Qd, Rd, 1.0, 60000, x0, u_prev, x_ref, u_ref, lambda k, v: np.clip(v, lo, hi), x_lo=x_lo, x_hi=x_hi)
    S, d = condense(A, Bm, e, x0)
    Wq = np.kron(np.eye(N), np.diag(Qd)); Wr = np.kron(np.eye(N), np.diag(Rd))
    cost = lambda U: 0.5 * (S @ U + d - x_ref.reshape(-1)) @ Wq @ (S @ U + d - x_ref.reshape(-1)) + 0.5 * (U - u_ref.reshape(-1)) @ Wr @ (U - u_ref.reshape(-1))
    grad = lambda U: S.T @ Wq @ (S @ U + d - x_ref.reshape(-1)) + Wr @ (U - u_ref.reshape(-1))
    cons = []
    Xlo, Xhi = np.tile(x_lo, N), np.tile(x_hi, N)
    for i in range(N * nx):
        if np.isfinite(Xlo[i]):
            cons.append(dict(type="ineq", fun=lambda U, i=i: S[i] @ U + d[i] - Xlo[i], jac=lambda U, i=i: S[i]))
        if np.isfinite(Xhi[i]):
            cons.append(dict(type="ineq", fun=lambda U, i=i: Xhi[i] - S[i] @ U - d[i], jac=lambda U, i=i: -S[i]))
    res = minimize(cost, np.zeros(N * nu), jac=grad, bounds=list(zip(np.tile(lo, N), np.tile(hi, N))), constraints=cons, method="SLSQP",
                   options=dict(ftol=1e-15, maxiter=2000))
    U = res.x; X = (S @ U + d).reshape(N, nx)
    assert res.success
    assert np.sum(np.abs(X[:, 0] - x_lo[0]) < 1e-7) + np.sum(np.abs(X[:, 1] - x_hi[1]) < 1e-7) >= 2   # the state box is active
    assert np.abs(out["z"][:, nx:] - U.reshape(N, nu)).max() < 2e-5
    assert np.abs(out["z"][:, :nx] - X).max() < 2e-5
    assert np.all(out["z"][:, 0] >= x_lo[0] - 1e-12) and np.all(out["z"][:, 1] <= x_hi[1] + 1e-12)
    assert cost(out["z"][:, nx:].reshape(-1)) <= cost(U) + 1e-7
