"""GPU parity: the CUDA path (through the C ABI) vs the fp64 oracle on the same seeded inputs.

north_star tolerances, per env, after the same fixed iteration count:
    max|du| <= 1e-3 (1 + |u_ref|_inf),  max|dx| <= 1e-4 (1 + |x_ref|_inf),  residuals to 1e-3 relative
with "ref" read as the oracle's solution AND as the tracking reference, enforcing the tighter of
the two (reading D14); residual floor per reading D15 (5e-5 (1 + |u|_inf)).
"""
import numpy as np
import pytest

import gen
import oracle

pytestmark = pytest.mark.gpu

METHODS = ["srb", "dense"]


def _method(name):
    from paper_2606_05687_b200 import METHOD_DENSE, METHOD_SRB
    return {"srb": METHOD_SRB, "dense": METHOD_DENSE}[name]


def run_gpu(w, method="srb", iters=None, rho=None, tol=None, dynamics=None):
    import torch
    from paper_2606_05687_b200 import Solver, make_layout
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho if rho is None else rho,
               iters=w.iters if iters is None else iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt,
               method=_method(method), dense_workspace=(method == "dense" or dynamics is not None))
    s.set_workload(w)
    if dynamics is not None:
        s.set_dynamics(*dynamics)
    if tol is not None:
        s.set_tolerance(*tol)
    s.solve()
    out = s.get(aux=True)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["launches"] = s.launch_count()
    s.close()
    return res


# Absolute floor of the residual comparison per unit of (1 + |u|_inf) (reading D15): r_prim = max|u - z| is a
# difference of O(|u|) float32 numbers, so its absolute error is a few ulp of |u| whatever its own size.
RES_FLOOR = 5e-5
WORST_RES = {"r_prim": -1.0, "r_dual": -1.0}


def check_parity(w, got, ref, envs=None):
    """got: GPU outputs for all envs of w (or for `envs`); ref: oracle outputs for `envs`."""
    sel = slice(None) if envs is None else envs
    u = got["u"][sel].astype(np.float64); x = got["x"][sel].astype(np.float64)
    ax = tuple(range(1, u.ndim))
    du = np.abs(u - ref["u"]).max(axis=ax); dx = np.abs(x - ref["x"]).max(axis=ax)
    un = np.abs(ref["u"]).max(axis=ax)
    if w.u_ref is not None:                         # (u_ref = NULL: there is no tracking reference to take the norm of)
        un = np.minimum(un, np.abs(w.u_ref[sel]).max(axis=ax))
    xn = np.minimum(np.abs(ref["x"]).max(axis=ax), np.abs(w.x_ref[sel]).max(axis=ax))
    tol_u = 1e-3 * (1 + un); tol_x = 1e-4 * (1 + xn)
    worst_u = np.max(du / tol_u); worst_x = np.max(dx / tol_x)
    assert worst_u <= 1.0, f"max|du| / tol = {worst_u:.3f} (env {np.argmax(du / tol_u)})"
    assert worst_x <= 1.0, f"max|dx| / tol = {worst_x:.3f} (env {np.argmax(dx / tol_x)})"
    # residuals: 1e-3 relative (north_star) plus an absolute floor (reading D15).  r_prim = max|u - z|
    # is a difference of O(|u|) fp32 numbers, so it inherits the ABSOLUTE error of u and z, which
    # north_star itself allows to be 1e-3 (1 + |u|); the floor is 1/20 of that allowance.
    floor = RES_FLOOR * (1 + np.abs(ref["u"]).max(axis=ax))
    for name in ("r_prim", "r_dual"):
        r = got[name][sel].astype(np.float64)
        err = np.abs(r - ref[name])
        # measured excess over the relative bar, in units of (1 + |u|_inf): what the floor has to cover
        WORST_RES[name] = max(WORST_RES[name], float(np.max((err - 1e-3 * ref[name]) / (1 + np.abs(ref["u"]).max(axis=ax)))))
        assert np.all(err <= 1e-3 * ref[name] + floor), (name, float(np.max(err / (1e-3 * ref[name] + floor))))
    assert np.array_equal(got["iters_done"][sel], ref["iters_done"])
    # z and y are not part of north_star's bar.  Both live in the units of u (y accumulates u - z every
    # iteration, so it inherits u's absolute rounding error), hence both get u's allowance.
    dz = np.abs(got["z"][sel] - ref["z"]).max(axis=ax); dy = np.abs(got["y"][sel] - ref["y"]).max(axis=ax)
    assert np.all(dz <= 2 * tol_u), f"max|dz| / tol = {np.max(dz / tol_u):.3f}"
    assert np.all(dy <= tol_u), f"max|dy| / tol = {np.max(dy / tol_u):.3f}"
    return worst_u, worst_x


def sample_envs(B, n, seed=0):
    if B <= n:
        return np.arange(B)
    rng = np.random.default_rng(seed)
    idx = np.unique(np.concatenate([[0, 1, B - 2, B - 1], rng.choice(B, n - 4, replace=False)]))
    return np.sort(idx)


# ---------------------------------------------------------------------------------------------
def test_assembly_matches_oracle():
    """S1: pinmpc_get_dynamics vs oracle O1 (element by element; fp32 rounding only)."""
    import torch
    from paper_2606_05687_b200 import Solver
    for cfg, B, N in ((0, 64, 10), (3, 37, 7)):
        w = gen.make_config(cfg, B=B, N=N)
        s = Solver(w.nu, w.N, w.B, dt=w.dt, Qdiag=w.Qdiag, Rdiag=w.Rdiag)
        s.set_workload(w)
        A, Bm, c = [t.cpu().numpy().astype(np.float64) for t in s.get_dynamics()]
        torch.cuda.synchronize()
        Ao, Bo, co = oracle.assemble(w.nu, w.n_wrench, w.n_force, w.dt, w.yaw, w.foot_r, w.mass, w.inertia, w.ext_wrench)
        assert np.max(np.abs(A - Ao)) <= 2e-7 * np.max(np.abs(Ao))
        assert np.max(np.abs(Bm - Bo)) <= 4e-6 * np.max(np.abs(Bo))
        assert np.max(np.abs(c - co)) <= 4e-6 * max(np.max(np.abs(co)), 1e-12)
        assert np.array_equal(A == 0, Ao == 0) and np.array_equal(Bm == 0, Bo == 0)      # sparsity pattern
        s.close()


@pytest.mark.parametrize("method", METHODS)
def test_config0_all_envs(method):
    w = gen.make_config(0)
    got = run_gpu(w, method)
    ref = oracle.solve(w)
    wu, wx = check_parity(w, got, ref)
    print(f"c0 {method}: worst du/tol {wu:.3f} dx/tol {wx:.3f} launches {got['launches']}")
    # properties that hold exactly on the GPU side as well
    assert np.all(got["x"][:, :, 12] == np.float32(-9.81))
    sw = w.contact == 0
    assert np.all(got["z"][:, :, 0:3][sw[:, :, 0]] == 0) and np.all(got["z"][:, :, 9:12][sw[:, :, 1]] == 0)


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_full_size_configs_sampled_envs(cfg, method):
    """BASELINE.json configs 1-3 at full size in the launch configuration bench.py times; the oracle
    recomputes a sample of envs one by one (envs are independent QPs)."""
    w = gen.make_config(cfg)
    got = run_gpu(w, method)
    envs = sample_envs(w.B, 192, seed=cfg)
    ref = oracle.solve(gen.subset(w, envs))
    wu, wx = check_parity(w, got, ref, envs)
    print(f"c{cfg} {method}: worst du/tol {wu:.3f} dx/tol {wx:.3f}")
    # at-any-size properties on ALL envs: finite, gravity state untouched, swing z exactly zero
    assert np.isfinite(got["u"]).all() and np.isfinite(got["x"]).all()
    assert np.all(got["x"][:, :, 12] == np.float32(-9.81))
    assert np.all(got["iters_done"] == w.iters)
    assert np.all(got["z"][:, :, 0:3][w.contact[:, :, 0] == 0] == 0)


@pytest.mark.parametrize("B,N", [(1024, 10), (4096, 25), (1024, 100), (16384, 50), (65536, 100)])
def test_sweep_points_sampled_envs(B, N):
    w = gen.make_config(4, B=B, N=N)
    got = run_gpu(w, "srb")
    envs = sample_envs(B, 96, seed=N)
    ref = oracle.solve(gen.subset(w, envs))
    check_parity(w, got, ref, envs)
    assert np.isfinite(got["u"]).all()


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("B,N,nu", [(1, 1, 12), (3, 2, 12), (37, 7, 12), (5, 33, 18), (130, 13, 18), (2, 128, 12)])
def test_ragged_and_degenerate_shapes(B, N, nu, method):
    w = gen.make_config(3 if nu == 18 else 1, B=B, N=N, iters=30)
    got = run_gpu(w, method)
    check_parity(w, got, oracle.solve(w))


def test_all_swing_and_all_stance_stages():
    w = gen.make_config(0, B=8, N=6)
    w.contact[0:4] = 0            # flight: every contact off => z == 0, u is driven to 0
    w.contact[4:8] = 1            # double support
    for m in METHODS:
        got = run_gpu(w, m)
        check_parity(w, got, oracle.solve(w))
        assert np.all(got["z"][0:4] == 0)


def test_generic_ltv_through_set_dynamics():
    """pinmpc_set_dynamics: arbitrary dense A_k, B_k, c_k (dense variant)."""
    rng = np.random.default_rng(0)
    w = gen.make_config(0, B=16, N=9)
    A, Bm, c = oracle.assemble(w.nu, w.n_wrench, w.n_force, w.dt, w.yaw, w.foot_r, w.mass, w.inertia)
    A = (A + rng.normal(size=A.shape) * 1e-3).astype(np.float32)
    Bm = (Bm + rng.normal(size=Bm.shape) * 1e-4).astype(np.float32)
    c = (rng.normal(size=c.shape) * 1e-3).astype(np.float32)
    got = run_gpu(w, "dense", dynamics=(A, Bm, c))
    ref = oracle.solve(w, A=A, Bm=Bm, c=c)
    check_parity(w, got, ref)


@pytest.mark.parametrize("method", METHODS)
def test_well_scaled_rho_and_early_exit(method):
    """rho = 1e-2 with tolerances: the stop decision is an integer taken from fp32 vs fp64 residuals,
    so compare each env against the oracle run for exactly the iteration count the GPU took."""
    w = gen.make_config(0, B=16, N=10)
    got = run_gpu(w, method, iters=3000, rho=1e-2, tol=(1e-2, 1e-3, 10))
    ref_tol = oracle.solve(w, iters=3000, rho=1e-2, eps_abs=1e-2, eps_rel=1e-3, check_every=10)
    it = got["iters_done"]
    assert np.all(it % 10 == 0) and np.all(it < 3000) and np.all(it >= 10)
    assert np.all(np.abs(it - ref_tol["iters_done"]) <= 10)          # at most one check interval apart
    for b in range(w.B):
        ref = oracle.solve(gen.subset(w, [b]), iters=int(it[b]), rho=1e-2)
        sub = {k: (v[b:b + 1] if isinstance(v, np.ndarray) else v) for k, v in got.items()}
        check_parity(gen.subset(w, [b]), sub, ref)


def test_error_codes_on_device():
    import torch
    from paper_2606_05687_b200 import PinmpcError, Solver, binding
    w = gen.make_config(0, B=4, N=5)
    s = Solver(w.nu, w.N, w.B, dt=w.dt)
    with pytest.raises(PinmpcError) as e:
        s.solve()
    assert e.value.status == binding.ESTATE
    s.set_workload(w)
    with pytest.raises(PinmpcError) as e:
        s.get()
    assert e.value.status == binding.ESTATE
    with pytest.raises(PinmpcError) as e:          # small workspace has no room for dense dynamics
        s.set_dynamics(torch.zeros(4, 5, 13, 13), torch.zeros(4, 5, 13, 12))
    assert e.value.status == binding.EALLOC
    s.solve(); s.get()
    torch.cuda.synchronize()
    s.close()


@pytest.mark.parametrize("B,N,nu", [(37, 13, 12), (21, 50, 12), (19, 9, 18)])
def test_results_do_not_depend_on_envs_per_cta(B, N, nu):
    """pinmpc_set_tuning: every CTA shape (1..16 envs, ragged last CTA, odd N => ragged second stage
    of the stage threads) gives the oracle's answer."""
    import torch
    from paper_2606_05687_b200 import METHOD_SRB, Solver, make_layout
    w = gen.make_config(3 if nu == 18 else 2, B=B, N=N, iters=25)
    ref = oracle.solve(w)
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    for G in (1, 2, 5, 6, 7, 11, 16):
        s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho, iters=w.iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt, method=METHOD_SRB)
        s.set_workload(w)
        s.set_tuning(G)
        s.solve()
        out = s.get(aux=True)
        torch.cuda.synchronize()
        check_parity(w, {k: v.cpu().numpy() for k, v in out.items()}, ref)
        s.close()


def test_kernel_timing_hook():
    """pinmpc_set_profiling / pinmpc_get_kernel_ms: three positive durations that add up to about the solve."""
    import torch
    from paper_2606_05687_b200 import PinmpcError, Solver, binding
    w = gen.make_config(1, B=256, N=20)
    s = Solver(w.nu, w.N, w.B, dt=w.dt, iters=w.iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag)
    s.set_workload(w)
    s.solve()
    with pytest.raises(PinmpcError) as e:
        s.kernel_ms()
    assert e.value.status == binding.ESTATE
    s.set_profiling(True)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream = torch.cuda.current_stream()
    a.record(stream); s.solve(); b.record(stream)
    ms = s.kernel_ms()
    torch.cuda.synchronize()
    assert len(ms) == 3 and all(m > 0 for m in ms)
    assert sum(ms) <= a.elapsed_time(b) * 1.05 + 0.05
    assert ms[2] > ms[0]
    s.close()


def test_maximum_horizon_and_single_env():
    """N = PINMPC_N_MAX (256) with B = 1 and B = 3: one env per CTA, arena of 82 KB per env."""
    for B in (1, 3):
        w = gen.make_config(1, B=B, N=256, iters=20)
        got = run_gpu(w, "srb")
        check_parity(w, got, oracle.solve(w))


@pytest.mark.parametrize("method", METHODS)
def test_warm_start(method):
    """pinmpc_set_warm_start.  (a) The ADMM state is (z, y): 30 cold iterations, then 20
    from their z, y = 50 cold iterations of the oracle.  (b) Receding horizon: a new problem started from the
    previous z, y shifted by one stage vs the oracle started from the same values."""
    import torch
    from paper_2606_05687_b200 import Solver, make_layout
    w = gen.make_config(1, B=48, N=21, iters=50)
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)

    def solve(work, iters, z0=None, y0=None):
        s = Solver(work.nu, work.N, work.B, layout=lay, rho=work.rho, iters=iters, Qdiag=work.Qdiag, Rdiag=work.Rdiag,
                   dt=work.dt, method=_method(method), dense_workspace=(method == "dense"))
        s.set_workload(work)
        s.set_warm_start(z0, y0)
        s.solve()
        out = s.get(aux=True)
        torch.cuda.synchronize()
        res = {k: v.cpu().numpy() for k, v in out.items()}
        s.close()
        return res

    first = solve(w, 30)
    second = solve(w, 20, first["z"], first["y"])
    ref = oracle.solve(w, iters=50)
    second["iters_done"] = second["iters_done"] + 30
    check_parity(w, second, ref)
    # (b) the next MPC problem (another seed of the same generator), started from the shifted previous solution
    w2 = gen.make_config(2, B=48, N=21, iters=15)
    z0 = np.concatenate([first["z"][:, 1:], first["z"][:, -1:]], axis=1)
    y0 = np.concatenate([first["y"][:, 1:], first["y"][:, -1:]], axis=1)
    got = solve(w2, 15, np.ascontiguousarray(z0), np.ascontiguousarray(y0))
    check_parity(w2, got, oracle.solve(w2, iters=15, z0=z0, y0=y0))
    # and back to a cold start on the same handle semantics: None, None
    cold = solve(w2, 15, None, None)
    check_parity(w2, cold, oracle.solve(w2, iters=15))


def test_warm_start_argument_check():
    import torch
    from paper_2606_05687_b200 import PinmpcError, Solver, binding
    w = gen.make_config(0, B=4, N=5)
    s = Solver(w.nu, w.N, w.B, dt=w.dt)
    with pytest.raises(PinmpcError) as e:
        binding.pinmpc_set_warm_start(s.h, torch.zeros(4, 5, 12, device="cuda"), None)
    assert e.value.status == binding.EINVAL
    s.close()


def _stage_window(w, a, N, x0):
    from dataclasses import replace
    kw = {}
    for f in ("x_ref", "u_ref", "contact", "foot_r", "yaw", "ext_wrench"):
        v = getattr(w, f)
        kw[f] = None if v is None else np.ascontiguousarray(v[:, a:a + N])
    return replace(w, N=N, x0=np.ascontiguousarray(x0, dtype=np.float32), name=f"{w.name}_win{a}", **kw)


def test_receding_horizon_shift():
    """pinmpc_shift_aux: z0[b,k] = z[b,min(k+shift,N-1)] bit for bit (a copy), and what it is for: the next MPC
    problem (window moved by one stage, x0 = the predicted x_1) started from the shifted z, y meets the same
    tolerance in fewer iterations than from a cold start."""
    import torch
    from paper_2606_05687_b200 import PinmpcError, Solver, binding, make_layout
    N = 20
    long = gen.make_config(1, B=96, N=N + 1, iters=3000)
    lay = make_layout(long.n_wrench, long.n_force, long.mu, long.fz_max, long.mx_coef, long.my_coef, long.mz_coef, long.hand_fmax)
    w0 = _stage_window(long, 0, N, long.x0)
    s = Solver(w0.nu, N, w0.B, layout=lay, rho=1e-2, iters=3000, Qdiag=w0.Qdiag, Rdiag=w0.Rdiag, dt=w0.dt)   # well-scaled rho
    zbuf = torch.empty((w0.B, N, w0.nu), device="cuda"); ybuf = torch.empty_like(zbuf)
    with pytest.raises(PinmpcError) as e:                     # nothing solved yet
        binding.pinmpc_shift_aux(s.h, 1, zbuf, ybuf, None)
    assert e.value.status == binding.ESTATE
    s.set_tolerance(1e-2, 1e-3, 5)
    s.set_workload(w0)
    s.solve()
    first = {k: v.cpu().numpy() for k, v in s.get(aux=True).items()}
    for bad in (-1, N + 1):
        with pytest.raises(PinmpcError) as e:
            binding.pinmpc_shift_aux(s.h, bad, zbuf, ybuf, None)
        assert e.value.status == binding.EINVAL
    for shift in (0, 1, 3, N):
        binding.pinmpc_shift_aux(s.h, shift, zbuf, ybuf, None)
        idx = np.minimum(np.arange(N) + shift, N - 1)
        assert np.array_equal(zbuf.cpu().numpy(), first["z"][:, idx])
        assert np.array_equal(ybuf.cpu().numpy(), first["y"][:, idx])
    # the next MPC update
    w1 = _stage_window(long, 1, N, first["x"][:, 0])
    s.shift_warm_start(1)                                     # before set_problem: it reads the last solve's z, y
    s.set_workload(w1)
    s.solve()
    warm = {k: v.cpu().numpy() for k, v in s.get().items()}
    s.set_warm_start(None, None)
    s.solve()
    cold = {k: v.cpu().numpy() for k, v in s.get().items()}
    s.close()
    assert cold["iters_done"].max() < 3000                    # both converged to the tolerance
    assert warm["iters_done"].mean() < 0.8 * cold["iters_done"].mean(), (warm["iters_done"].mean(), cold["iters_done"].mean())
    # (u itself is not compared: with R = 1e-5 the optimum is nearly flat in u, so two runs stopped at the same
    # tolerance differ by far more than the tolerance)
    for run in (warm, cold):
        assert np.all(run["r_prim"] <= 1e-2 + 1e-3 * np.abs(run["u"]).max(axis=(1, 2)) * 1.01)
