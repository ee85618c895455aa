"""Pins for oracle O2 + O3 steps 1-3 (the equality-constrained step).  SURVEY.md T1, T6.

north_star: "With no inequality constraints, its equality step must equal a sequential Riccati LQR
solve to 1e-9" — checked against (a) one dense KKT solve and (b) an independent textbook Riccati.
"""
import numpy as np
import pytest

import gen
import oracle
from refcheck import NX, kkt_eqstep, riccati_lqr_textbook


def _env(w, b):
    A, Bm, c = oracle.assemble(w.nu, w.n_wrench, w.n_force, w.dt, w.yaw[b:b + 1], w.foot_r[b:b + 1],
                               w.mass[b:b + 1], w.inertia[b:b + 1],
                               None if w.ext_wrench is None else w.ext_wrench[b:b + 1])
    return A[0], Bm[0], c[0]


def _rel(a, b):
    return np.max(np.abs(a - b)) / (1.0 + np.max(np.abs(b)))


@pytest.mark.parametrize("cfg,N", [(0, 3), (0, 10), (2, 50), (3, 12)])
def test_eqstep_equals_dense_kkt_and_textbook_riccati(cfg, N):
    w = gen.make_config(cfg, B=4, N=N)
    rng = np.random.default_rng(cfg * 100 + N)
    Qd = w.Qdiag.astype(float); Rd = w.Rdiag.astype(float)
    for b in range(w.B):
        A, Bm, c = _env(w, b)
        z = rng.normal(size=(N, w.nu)) * 100; y = rng.normal(size=(N, w.nu)) * 30
        fac = oracle.factor_env(A, Bm, c, Qd, Rd, w.rho)
        x, u = oracle.eqstep_env(A, Bm, c, fac, Qd, Rd, w.rho, w.x0[b], w.x_ref[b], w.u_ref[b], z, y)
        xk, uk = kkt_eqstep(A, Bm, c, Qd, Rd, w.rho, w.x0[b].astype(float), w.x_ref[b].astype(float),
                            w.u_ref[b].astype(float), z, y)
        lin = Rd * w.u_ref[b].astype(float) + w.rho * (z - y)
        xr, ur = riccati_lqr_textbook(A, Bm, c, Qd, Rd + w.rho, w.x0[b].astype(float),
                                      w.x_ref[b].astype(float), lin)
        assert _rel(u, uk) < 1e-9 and _rel(x, xk) < 1e-9
        assert _rel(u, ur) < 1e-9 and _rel(x, xr) < 1e-9
        # dynamics hold exactly along the returned trajectory (north_star: 1e-8)
        xprev = w.x0[b].astype(float)
        for k in range(N):
            assert np.max(np.abs(x[k] - (A[k] @ xprev + Bm[k] @ u[k] + c[k]))) < 1e-10
            xprev = x[k]


def test_eqstep_with_time_varying_affine_term():
    """Random c_k != 0 (generic LTV through the same code): pins s_k = P_{k+1} c_k and g = p - s."""
    rng = np.random.default_rng(11)
    w = gen.make_config(0, B=1, N=6)
    A, Bm, _ = _env(w, 0)
    c = rng.normal(size=(6, NX)) * 0.1
    A = A + rng.normal(size=A.shape) * 0.01          # and a generic dense A_k
    Qd = w.Qdiag.astype(float); Rd = w.Rdiag.astype(float)
    z = rng.normal(size=(6, 12)) * 50; y = rng.normal(size=(6, 12)) * 5
    fac = oracle.factor_env(A, Bm, c, Qd, Rd, 0.37)
    x, u = oracle.eqstep_env(A, Bm, c, fac, Qd, Rd, 0.37, w.x0[0], w.x_ref[0], w.u_ref[0], z, y)
    xk, uk = kkt_eqstep(A, Bm, c, Qd, Rd, 0.37, w.x0[0].astype(float), w.x_ref[0].astype(float),
                        w.u_ref[0].astype(float), z, y)
    assert _rel(u, uk) < 1e-9 and _rel(x, xk) < 1e-9


def test_unconstrained_admm_fixed_point_is_plain_lqr_with_R():
    """T6: with every U_k = R^nu (all contacts 'in contact', no limits) the ADMM fixed point has
    z = u, y = 0 and equals the LQR solution with weight R (not R + rho)."""
    w = gen.make_config(0, B=2, N=8)
    w.contact[:] = 1
    for name in ("mu", "fz_max", "mx_coef", "my_coef", "mz_coef"):
        setattr(w, name, 1e3)                          # |f_x| <= 1e3 f_z etc.: never binds here
    w.fz_max = 1e9
    # only f_z >= 0 cannot be lifted through the layout: a heavy R and a both-feet weight-sharing
    # reference keep the LQR solution's f_z strictly positive, so that constraint never binds
    w.Rdiag[:] = 1.0
    w.u_ref[:] = 0.0
    w.u_ref[:, :, 2] = w.u_ref[:, :, 5] = (w.mass * 9.81 / 2)[:, None]
    res = oracle.solve(w, iters=4000, rho=1.0, eps_abs=1e-12, eps_rel=0.0)
    Qd = w.Qdiag.astype(float); Rd = w.Rdiag.astype(float)
    for b in range(w.B):
        A, Bm, c = _env(w, b)
        lin = Rd * w.u_ref[b].astype(float)
        xr, ur = riccati_lqr_textbook(A, Bm, c, Qd, Rd, w.x0[b].astype(float), w.x_ref[b].astype(float), lin)
        if np.any(ur[:, [2, 5]] < 0):                  # f_z >= 0 is the one constraint that cannot be lifted
            continue
        assert _rel(res["u"][b], ur) < 1e-8 and _rel(res["x"][b], xr) < 1e-8
        assert np.max(np.abs(res["y"][b])) < 1e-6 * (1 + np.max(np.abs(ur)))
        assert np.max(np.abs(res["z"][b] - res["u"][b])) < 1e-9 * (1 + np.max(np.abs(ur)))
        break
    else:
        pytest.fail("no env with an interior LQR solution in the sample")


def test_factor_P0_is_symmetric_psd_and_K_matches_definition():
    w = gen.make_config(1, B=1, N=20)
    A, Bm, c = _env(w, 0)
    Qd = w.Qdiag.astype(float); Rd = w.Rdiag.astype(float)
    fac = oracle.factor_env(A, Bm, c, Qd, Rd, w.rho)
    P0 = fac["P0"]
    assert np.max(np.abs(P0 - P0.T)) < 1e-9 * np.max(np.abs(P0))
    assert np.linalg.eigvalsh(P0).min() > -1e-8 * np.max(np.abs(P0))
    # last stage: P_N = Q  =>  M = Rt + B^T Q B, K = M^-1 B^T Q A, Phi = A - B K
    k = 19
    M = np.diag(Rd + w.rho) + Bm[k].T @ np.diag(Qd) @ Bm[k]
    np.testing.assert_allclose(fac["L"][k] @ fac["L"][k].T, M, rtol=1e-12, atol=1e-12)
    Kdef = np.linalg.solve(M, Bm[k].T @ np.diag(Qd) @ A[k])
    np.testing.assert_allclose(fac["K"][k], Kdef, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(fac["Phi"][k], A[k] - Bm[k] @ Kdef, rtol=1e-10, atol=1e-12)
