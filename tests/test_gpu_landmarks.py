"""GPU parity of the predictive landmarks / prediction-confidence reward (eq. (10)-(14)) against
oracle/landmarks.py through the C ABI.  Inputs are seeded and synthetic: the "realised CoM" is a random walk,
the predictions are random perturbations of it (the paper's simulator is not available).

Bar: the number of landmarks used is exact (integer work); the reward is fp32 exp of an fp32 sum of at most
eight terms of magnitude <= ~10: |r_gpu - r_orc| <= 2e-6 + 4e-6 * (-log r_orc) * r_orc, i.e. a few ulps of the
exponent; written below as atol 2e-6 + rtol-on-exponent 4e-6.
"""
import ctypes

import numpy as np
import pytest

import gen
from oracle.landmarks import LandmarkOracle

pytestmark = pytest.mark.gpu

PAPER_ALPHA = [0.5, 0.25, 0.15, 0.07, 0.03]


def check_reward(r_gpu, used_gpu, r_ref, used_ref):
    assert np.array_equal(used_gpu, used_ref)
    expo = -np.log(np.maximum(r_ref, 1e-300))
    tol = 2e-6 + 4e-6 * expo * r_ref
    err = np.abs(r_gpu.astype(np.float64) - r_ref)
    assert np.all(err <= tol), f"max err/tol {np.max(err / tol):.2f}"


def rollout(B, N, s, alpha, Qc, sigma, T, solve_every, seed, resets=True):
    import torch
    from paper_2606_05687_b200 import Landmarks, make_landmark_cfg
    rng = np.random.default_rng(seed)
    cfg = make_landmark_cfg(s, alpha, Qc, sigma)
    lm = Landmarks(B, N, cfg)
    orc = LandmarkOracle(B, N, np.asarray(s, dtype=np.float32), alpha, Qc, sigma)
    t = rng.integers(0, 3 * N, size=B).astype(np.int32)          # every env has its own clock
    c = rng.normal(size=(B, 3)).astype(np.float32)
    checked = 0
    for step in range(T):
        td = torch.from_numpy(t).cuda()
        r, used = lm.reward(torch.from_numpy(c).cuda(), td)
        r_ref, used_ref = orc.reward(c, t)
        check_reward(r.cpu().numpy(), used.cpu().numpy(), r_ref, used_ref)
        checked += int(used_ref.sum())
        if step % solve_every == 0:
            # predicted trajectory: the true walk direction plus noise growing with the look-ahead
            x = rng.normal(size=(B, N, 13)).astype(np.float32)
            x[:, :, 3:6] = c[:, None, :] + (0.02 * sigma * 10) * np.sqrt(np.arange(1, N + 1))[None, :, None] * rng.normal(size=(B, N, 3))
            x = x.astype(np.float32)
            lm.push(torch.from_numpy(x).cuda(), td)
            orc.push(x, t)
        if resets and step % 7 == 3:
            mask = rng.random(B) < 0.2
            lm.reset(torch.from_numpy(mask.astype(np.uint8)).cuda())
            orc.reset(mask)
            t = np.where(mask, 0, t).astype(np.int32)             # time restarts with the episode
        c = (c + 0.01 * rng.normal(size=(B, 3))).astype(np.float32)
        t = t + 1
    return checked


@pytest.mark.parametrize("B,N,solve_every", [(300, 7, 1), (129, 10, 3), (64, 1, 1), (1, 50, 5)])
def test_rollout_matches_oracle(B, N, solve_every):
    used = rollout(B, N, np.linspace(0, 1, 5), PAPER_ALPHA, [1.0, 1.0, 4.0], 0.05, 3 * N + 12, solve_every, seed=11 + N)
    assert used > 0


def test_rollout_full_size_config2():
    # B = 4096, N = 50 (config 2), the paper's schedule, re-solve every 5 steps; no resets so
    # that every landmark, including n = N, is eventually compared
    used = rollout(4096, 50, np.linspace(0, 1, 5), PAPER_ALPHA, [1.0, 1.0, 1.0], 0.05, 62, 5, seed=2, resets=False)
    assert used > 4096 * 5


def test_eight_landmarks_and_uneven_s():
    rollout(200, 30, [0.0, 0.05, 0.1, 0.2, 0.35, 0.5, 0.8, 1.0], [0.3, 0.2, 0.15, 0.12, 0.1, 0.07, 0.04, 0.02], [2.0, 0.5, 1.0], 0.1,
            100, 2, seed=5)


def test_push_from_solver_workspace():
    """pinmpc_landmark_push_solver reads x_1..x_N of the last solve in place: same rewards as pushing pinmpc_get's copy."""
    import torch
    from paper_2606_05687_b200 import Landmarks, Solver, make_landmark_cfg, make_layout
    w = gen.make_config(0)
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho, iters=w.iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt)
    s.set_workload(w)
    s.solve()
    cfg = make_landmark_cfg(np.linspace(0, 1, 5), PAPER_ALPHA, [1.0, 1.0, 1.0], 0.5)
    lm = Landmarks(w.B, w.N, cfg)
    t0 = torch.zeros(w.B, dtype=torch.int32, device="cuda")
    lm.push_solver(s, t0)
    x = s.get()["x"].cpu().numpy()
    orc = LandmarkOracle(w.B, w.N, np.linspace(0, 1, 5).astype(np.float32), PAPER_ALPHA, [1.0, 1.0, 1.0], 0.5)
    orc.push(x, np.zeros(w.B, dtype=np.int32))
    c = (x[:, 0, 3:6] + 0.1).astype(np.float32)
    for n in sorted(set(orc.n)):
        t = np.full(w.B, n, dtype=np.int32)
        r, used = lm.reward(torch.from_numpy(c).cuda(), torch.from_numpy(t).cuda())
        r_ref, used_ref = orc.reward(c, t)
        assert used_ref.min() >= 1
        check_reward(r.cpu().numpy(), used.cpu().numpy(), r_ref, used_ref)
    s.close()


def test_argument_checks():
    import torch
    from paper_2606_05687_b200 import binding as b
    lib = b.load()
    good = b.make_landmark_cfg([0, 1], [0.7, 0.3])
    assert lib.pinmpc_landmark_ring_bytes(4, 10, ctypes.byref(good)) == 4 * 2 * 11 * 16
    bad = b.make_landmark_cfg([0, 1], [0.7, 0.3]); bad.n_landmarks = 9
    assert lib.pinmpc_landmark_ring_bytes(4, 10, ctypes.byref(bad)) == 0
    bad2 = b.make_landmark_cfg([0, 1], [0.7, 0.3], sigma_c=0.0)
    bad3 = b.make_landmark_cfg([0, 1.5], [0.7, 0.3])
    ring = torch.zeros(4 * 2 * 11 * 16, dtype=torch.uint8, device="cuda")
    x = torch.zeros((4, 10, 13), device="cuda"); t = torch.zeros(4, dtype=torch.int32, device="cuda")
    c = torch.zeros((4, 3), device="cuda"); r = torch.zeros(4, device="cuda")
    P = lambda v: None if v is None else ctypes.c_void_p(v.data_ptr())
    for cfg in (bad, bad2, bad3):
        assert lib.pinmpc_landmark_push(P(ring), 4, 10, ctypes.byref(cfg), P(x), P(t), None) == b.EINVAL
        assert lib.pinmpc_landmark_reward(P(ring), 4, 10, ctypes.byref(cfg), P(c), P(t), P(r), None, None) == b.EINVAL
        assert lib.pinmpc_landmark_reset(P(ring), 4, 10, ctypes.byref(cfg), None, None) == b.EINVAL
    assert lib.pinmpc_landmark_push(P(ring), 4, 10, ctypes.byref(good), None, P(t), None) == b.EINVAL
    assert lib.pinmpc_landmark_reward(P(ring), 4, 10, ctypes.byref(good), P(c), None, P(r), None, None) == b.EINVAL
    assert lib.pinmpc_landmark_reward(None, 4, 10, ctypes.byref(good), P(c), P(t), P(r), None, None) == b.EINVAL
    # B = 0 is a no-op
    assert lib.pinmpc_landmark_push(None, 0, 10, ctypes.byref(good), None, None, None) == b.OK
    assert lib.pinmpc_landmark_reward(None, 0, 10, ctypes.byref(good), None, None, None, None, None) == b.OK
    # a fresh ring has no landmarks: r = 1, used = 0 (n_used may be NULL)
    assert lib.pinmpc_landmark_reset(P(ring), 4, 10, ctypes.byref(good), None, None) == b.OK
    assert lib.pinmpc_landmark_reward(P(ring), 4, 10, ctypes.byref(good), P(c), P(t), P(r), None, None) == b.OK
    torch.cuda.synchronize()
    assert torch.all(r == 1.0)
