"""GPU parity at full size, every env ("Parity uses every env for c0-c3 and >= 1024 envs per c4 point"),
and on inputs that reach every branch of the product kernels: random contact flags per (env, stage, contact) so that
flight, single- and double-support stages sit in one warp, full SPD inertia, non-uniform weights, u_ref = NULL,
hands without an external wrench, horizons up to PINMPC_N_MAX, every horizon-chunk setting.  The workloads are
copies of the seeded gen/ configs mutated here; the generator itself is unchanged.
"""
from dataclasses import replace

import numpy as np
import pytest

import gen
import oracle
from test_gpu_parity import check_parity, sample_envs

pytestmark = pytest.mark.gpu


def run(w, method="srb", chunks=None, envs_per_cta=None, iters=None):
    import torch
    from paper_2606_05687_b200 import METHOD_DENSE, METHOD_SRB, Solver, make_layout
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho, iters=w.iters if iters is None else iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag,
               dt=w.dt, method=METHOD_DENSE if method == "dense" else METHOD_SRB, dense_workspace=(method == "dense"))
    s.set_workload(w)
    if chunks is not None:
        s.set_horizon_chunks(chunks)
    if envs_per_cta is not None:
        s.set_tuning(envs_per_cta)
    s.solve()
    out = s.get(aux=True)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res["shape"] = s.launch_shape() if method != "dense" else None
    s.close()
    return res


# the three solver variants a full-size comparison covers: chunked TMEM kernel (default), sequential-pass kernel, dense
VARIANTS = [("srb", None), ("srb", 1), ("dense", None)]


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_full_size_configs_every_env(cfg):
    w = gen.make_config(cfg)
    ref = oracle.solve(w)
    for method, chunks in VARIANTS:
        got = run(w, method, chunks)
        wu, wx = check_parity(w, got, ref)
        print(f"c{cfg} {method} chunks={chunks} shape={got['shape']}: worst du/tol {wu:.3f} dx/tol {wx:.3f}")
        assert np.all(got["x"][:, :, 12] == np.float32(-9.81))
        assert np.all(got["iters_done"] == w.iters)
        assert np.all(got["z"][:, :, 0:3][w.contact[:, :, 0] == 0] == 0)
        if method == "srb":
            assert (got["shape"][1] == 1) == (chunks == 1)


@pytest.mark.parametrize("B", gen.SWEEP_B)
@pytest.mark.parametrize("N", gen.SWEEP_N)
def test_every_sweep_point_1024_envs(B, N):
    """BASELINE.json config 4: all 16 (B, N) points, 1024 envs of each against the oracle (all of them at B = 1024)."""
    w = gen.make_config(4, B=B, N=N)
    got = run(w)
    envs = sample_envs(B, 1024, seed=B + N)
    ref = oracle.solve(gen.subset(w, envs))
    wu, wx = check_parity(w, got, ref, envs)
    print(f"c4 B={B} N={N} shape={got['shape']}: worst du/tol {wu:.3f} dx/tol {wx:.3f}")
    assert np.isfinite(got["u"]).all() and np.isfinite(got["x"]).all()
    assert np.all(got["iters_done"] == w.iters)


def _random_rotations(rng, n):
    q, r = np.linalg.qr(rng.normal(size=(n, 3, 3)))
    q = q * np.sign(np.diagonal(r, axis1=1, axis2=2))[:, None, :]
    q[np.linalg.det(q) < 0, :, 0] *= -1
    return q


def mutate(w, seed, contacts=True, spd_inertia=True, weights=True, u_ref_none=False, ext_none=False):
    """A copy of workload w with random contact flags, full SPD inertia and non-uniform weights."""
    rng = np.random.default_rng(seed)
    kw = {}
    if contacts:
        kw["contact"] = (rng.random(w.contact.shape) < 0.5).astype(np.uint8)     # flight, single and double support mixed
    if spd_inertia:
        R = _random_rotations(rng, w.B)
        d = rng.uniform(0.5, 3.0, (w.B, 3))
        kw["inertia"] = np.einsum("bij,bj,bkj->bik", R, d, R).astype(np.float32)   # R diag(d) R^T
    if weights:
        kw["Rdiag"] = np.exp(rng.uniform(np.log(1e-6), np.log(1e-3), w.nu)).astype(np.float32)
        kw["Qdiag"] = (w.Qdiag * rng.uniform(0.5, 2.0, 13)).astype(np.float32)
    if u_ref_none:
        kw["u_ref"] = None
    if ext_none:
        kw["ext_wrench"] = None
    return replace(w, name=w.name + "_mut", **kw)


@pytest.mark.parametrize("cfg,B,N,opts", [
    (2, 4096, 50, {}),                                       # headline shape
    (1, 4096, 25, {}),                                       # odd number of stages per worker / stage thread
    (3, 2048, 30, {}),                                       # hands with random contact flags, external wrench
    (3, 1500, 21, {"ext_none": True}),                       # nu = 18 without ext_wrench
    (2, 1000, 50, {"u_ref_none": True}),                     # u_ref = NULL
    (2, 777, 37, {"contacts": False}),                       # generator's gait, SPD inertia and weights only
])
def test_random_contacts_spd_inertia_weights(cfg, B, N, opts):
    w = mutate(gen.make_config(cfg, B=B, N=N), seed=1000 * cfg + N, **opts)
    if opts.get("contacts", True):
        nf = w.contact[..., :2].sum(-1)
        assert (nf == 0).any() and (nf == 1).any() and (nf == 2).any()
    ref = oracle.solve(w)
    for method, chunks in VARIANTS:
        got = run(w, method, chunks)
        wu, wx = check_parity(w, got, ref)
        print(f"{w.name} {method} chunks={chunks}: worst du/tol {wu:.3f} dx/tol {wx:.3f}")
        off = w.contact == 0
        assert np.all(got["z"][:, :, 0:3][off[:, :, 0]] == 0) and np.all(got["z"][:, :, 6:9][off[:, :, 0]] == 0)
        assert np.all(got["z"][:, :, 3:6][off[:, :, 1]] == 0) and np.all(got["z"][:, :, 9:12][off[:, :, 1]] == 0)
        if w.nu == 18:
            assert np.all(got["z"][:, :, 12:15][off[:, :, 2]] == 0) and np.all(got["z"][:, :, 15:18][off[:, :, 3]] == 0)


@pytest.mark.parametrize("cfg,B,N", [(0, 64, 10), (3, 129, 7), (2, 300, 50)])
def test_product_assembly_records(cfg, B, N):
    """S1 on the PRODUCT kernel (k_assemble_srb): its records expanded back to A_k, B_k, c_k against oracle O1, and its
    S_k, T_k^-1 against their definitions evaluated in float64 from the oracle's B_k (SPD inertia, random weights)."""
    import torch
    from paper_2606_05687_b200 import Solver, make_layout
    w = mutate(gen.make_config(cfg, B=B, N=N), seed=7 + cfg, contacts=False)
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho, dt=w.dt, Qdiag=w.Qdiag, Rdiag=w.Rdiag)
    s.set_workload(w)
    A, Bm, c, S, Ti = [t.cpu().numpy().astype(np.float64) for t in s.get_srb_assembly()]
    torch.cuda.synchronize()
    s.close()
    Ao, Bo, co = oracle.assemble(w.nu, w.n_wrench, w.n_force, w.dt, w.yaw, w.foot_r, w.mass, w.inertia, w.ext_wrench)
    assert np.max(np.abs(A - Ao)) <= 2e-7 * np.max(np.abs(Ao))
    assert np.max(np.abs(Bm - Bo)) <= 2e-5 * np.max(np.abs(Bo))          # I_w is inverted in float32 on the way back
    assert np.max(np.abs(c - co)) <= 2e-5 * max(np.max(np.abs(co)), 1e-12)
    assert np.array_equal(A == 0, Ao == 0) and np.array_equal(Bm == 0, Bo == 0)
    # S = (Bh Rt^-1 Bh^T)^-1 with Bh = rows 6..11 of B, Rt = R + rho I
    Rt_inv = 1.0 / (w.Rdiag.astype(np.float64) + w.rho)
    Bh = Bo[:, :, 6:12, :]
    Sd = np.linalg.inv(np.einsum("bkij,j,bklj->bkil", Bh, Rt_inv, Bh))
    iu = np.triu_indices(6)
    assert np.max(np.abs(S - Sd[:, :, iu[0], iu[1]]) / np.max(np.abs(Sd), axis=(2, 3))[:, :, None]) <= 5e-5
    # T = Schur complement of the force block of Lam = Gh Rt^-1 Gh^T, Gh = D^-1 Bh, D = blkdiag(dt I_w^-1, dt/m I)
    Dinv = np.zeros((w.B, w.N, 6, 6))
    Dinv[:, :, :3, :3] = np.linalg.inv(Bo[:, :, 6:9, 6:9])                  # (dt I_w^-1)^-1: the moment block of foot 0
    for a in range(3):
        Dinv[:, :, 3 + a, 3 + a] = (w.mass.astype(np.float64) / w.dt)[:, None]
    Gh = Dinv @ Bh
    Lam = np.einsum("bkij,j,bklj->bkil", Gh, Rt_inv, Gh)
    T = Lam[:, :, :3, :3] - Lam[:, :, :3, 3:] @ np.linalg.inv(Lam[:, :, 3:, 3:]) @ Lam[:, :, 3:, :3]
    Tid = np.linalg.inv(T)
    i3 = np.triu_indices(3)
    assert np.max(np.abs(Ti - Tid[:, :, i3[0], i3[1]]) / np.max(np.abs(Tid), axis=(2, 3))[:, :, None]) <= 5e-5


@pytest.mark.parametrize("B,N", [(3, 400), (1, 512), (5, 300)])
def test_long_horizons(B, N):
    """PAPER.md:L314 "even to N = 400": the structured solver up to PINMPC_N_MAX = 512, both iteration kernels."""
    w = gen.make_config(1, B=B, N=N, iters=20)
    ref = oracle.solve(w)
    for chunks in (None, 1):
        got = run(w, "srb", chunks)
        wu, wx = check_parity(w, got, ref)
        print(f"N={N} B={B} chunks={chunks} shape={got['shape']}: worst du/tol {wu:.3f} dx/tol {wx:.3f}")


def test_horizon_chunk_settings():
    """pinmpc_set_horizon_chunks: every admissible chunk count gives the oracle's answer; inadmissible ones are refused."""
    from paper_2606_05687_b200 import PinmpcError, Solver, binding
    for cfg, B, N in ((2, 40, 50), (3, 23, 30), (1, 9, 6), (1, 5, 1), (1, 4, 13)):
        w = gen.make_config(cfg, B=B, N=N, iters=25)
        ref = oracle.solve(w)
        L = 6 if w.nu == 12 else 4
        lo = -(-N // L)
        hi = min(N, max(-(-N // (L - 1)), lo))
        for chunks in sorted({0, 1, lo, hi, (lo + hi) // 2}):
            for G in (None, 1, 3):
                got = run(w, "srb", chunks, G)
                check_parity(w, got, ref)
                if chunks > 1:
                    assert got["shape"][1] == chunks
                if chunks == 1:
                    assert got["shape"][1] == 1
    w = gen.make_config(2, B=4, N=50)
    s = Solver(w.nu, w.N, w.B, dt=w.dt)
    for bad in (2, 8, 11, 51):                       # ceil(50 / chunks) > 6, more chunk operators than the workspace holds, > N
        with pytest.raises(PinmpcError) as e:
            s.set_horizon_chunks(bad)
        assert e.value.status in (binding.EUNSUPPORTED, binding.EINVAL)
    with pytest.raises(PinmpcError):
        s.launch_shape()                             # nothing solved yet
    s.close()
