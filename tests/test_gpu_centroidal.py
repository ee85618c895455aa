"""GPU parity of the paper's own 9-state centroidal model (eq. (1)-(4)) through the C ABI:
pinmpc_assemble_centroidal against oracle/centroidal.py, and the stage-local ADMM on it (pinmpc_split_solve_ex with
nx = 9, variable scaling and the state box X_k of eq. (17)) against oracle/split.py.  Tolerances as for the main path."""
import numpy as np
import pytest

import gen
import oracle
from oracle import centroidal as cd, split

pytestmark = pytest.mark.gpu


def _t(a, dt=np.float32):
    import torch
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).cuda()


@pytest.mark.parametrize("cfg,B,N", [(0, 16, 10), (3, 9, 17), (2, 64, 50)])
def test_assembly_matches_oracle(cfg, B, N):
    from paper_2606_05687_b200 import binding
    w = gen.make_config(cfg, B=B, N=N)
    A, Bm, e = binding.assemble_centroidal(w.n_wrench, w.n_force, w.dt, _t(w.mass), _t(w.foot_r))
    Ao, Bo, eo = cd.assemble(w.n_wrench, w.n_force, w.dt, w.mass, w.foot_r)
    assert A.shape == Ao.shape and Bm.shape == Bo.shape and e.shape == eo.shape
    for g, o in ((A, Ao), (Bm, Bo), (e, eo)):
        g = g.cpu().numpy()
        assert np.abs(g - o).max() <= 2e-7 * (1 + np.abs(o).max())
        assert np.array_equal(g == 0, o == 0)                         # structural zeros are exact zeros


def _run(cfg, B, N, iters, box, accel=False):
    from paper_2606_05687_b200 import binding, make_layout
    w = gen.make_config(cfg, B=B, N=N)
    v = gen.centroidal_view(w)
    A, Bm, e = binding.assemble_centroidal(w.n_wrench, w.n_force, w.dt, _t(w.mass), _t(w.foot_r))
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    sx = 1.0 / np.sqrt(v["Qdiag"].astype(np.float64))
    u_prev = w.u_ref[:, 0].astype(np.float32)
    kw = dict(x_lo=v["x_lo"], x_hi=v["x_hi"]) if box else {}
    out = binding.split_solve(A, Bm, e, _t(v["x0"]), _t(u_prev), _t(v["x_ref"]), _t(w.u_ref), _t(w.contact, np.uint8), lay, v["Qdiag"], w.Rdiag,
                              1.0, iters, scale_x=sx.astype(np.float32), scale_u=100.0, accel=accel, **kw)
    xi, z, r = (t.cpu().numpy() for t in out[:3])
    An, Bn, en = (t.cpu().numpy().astype(np.float64) for t in (A, Bm, e))      # both sides consume the same float32 dynamics
    lay_o = oracle.layout_of(w)
    ref = []
    for b in range(B):
        proj = lambda k, vv, b=b: oracle.project(lay_o, w.contact[b, k:k + 1], vv[None])[0]
        ref.append(split.solve_env(An[b], Bn[b], en[b], v["Qdiag"], w.Rdiag, 1.0, iters, v["x0"][b], u_prev[b], v["x_ref"][b], w.u_ref[b], proj,
                                   scale_x=sx.astype(np.float32).astype(np.float64), scale_u=100.0, accel=accel,
                                   x_lo=v["x_lo"] if box else None, x_hi=v["x_hi"] if box else None))
    return w, v, xi, z, r, ref


def _check(xi, z, ref, skip=()):
    worst = 0.0
    for b, o in enumerate(ref):
        if b in skip:
            continue
        # per-block tolerances: positions (order 1), momenta (order 50), inputs (order 400)
        for name, g in (("xi", xi[b]), ("z", z[b])):
            for sl, tol in ((slice(0, 3), 1e-4), (slice(3, 9), 1e-4), (slice(9, None), 1e-3)):
                t = tol * (1 + np.abs(o[name][:, sl]).max())
                d = np.abs(g[:, sl] - o[name][:, sl]).max()
                worst = max(worst, d / t)
                assert d <= t, f"env {b} {name}[{sl}]: {d / t:.2f} tol"
    return worst


@pytest.mark.parametrize("cfg,B,N,iters,box", [(0, 16, 10, 80, False), (0, 16, 10, 80, True), (3, 8, 15, 60, True), (2, 6, 50, 40, True)])
def test_stage_local_admm_on_the_centroidal_model(cfg, B, N, iters, box):
    w, v, xi, z, r, ref = _run(cfg, B, N, iters, box)
    assert xi.shape == (B, N, 9 + w.nu)
    worst = _check(xi, z, ref)
    print(f"centroidal cfg {cfg} B={B} N={N} box={box}: worst error / tol {worst:.3f}")
    if box:
        assert np.all(z[:, :, 2] <= v["x_hi"][2] * (1 + 1e-6)) and np.all(np.abs(z[:, :, 3]) <= 20.0 * (1 + 1e-6))
        free = _run(cfg, B, N, iters, False)[3]
        assert np.abs(free[:, :, :9] - z[:, :, :9]).max() > 1e-3      # the box changed the iterates: it binds somewhere


def test_state_box_binds_at_convergence_and_accelerated_variant_runs():
    w, v, xi, z, r, ref = _run(0, 8, 10, 1500, True)
    assert np.median(r) < 1e-3                                        # xi = z (an env whose box cannot be met keeps a residual)
    for b, o in enumerate(ref):
        assert abs(r[b] - o["r_prim"]) <= 1e-3 * o["r_prim"] + 1e-4
    at_hi = np.isclose(z[:, :, 2], v["x_hi"][2], rtol=1e-6).sum() + np.isclose(np.abs(z[:, :, 3]), 20.0, rtol=1e-6).sum()
    assert at_hi > 0
    _check(xi, z, ref)
    w, v, xi, z, r, ref = _run(0, 8, 10, 40, True, accel=True)
    robust = [b for b, o in enumerate(ref) if o["margin"] > 1e-4]
    assert len(robust) >= 4
    _check(xi, z, ref, skip=[b for b in range(8) if b not in robust])
