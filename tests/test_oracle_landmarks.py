"""Pins of oracle/landmarks.py against what the paper fixes (eq. (10)-(14), Remark 1)."""
import math
import os

import numpy as np
import pytest

from oracle.landmarks import LandmarkOracle, landmark_steps

GOLD = os.path.join(os.path.dirname(__file__), "golden", "landmark_schedule.txt")


def paper_alpha():
    for line in open(GOLD):
        if line.startswith("alpha"):
            return [float(v) for v in line.split()[1:]]
    raise AssertionError("no alpha line")


def test_paper_schedule_is_horizon_monotone():
    a = paper_alpha()
    assert len(a) == 5 and all(a[i] > a[i + 1] > 0 for i in range(4))       # eq. (14)
    assert abs(sum(a) - 1.0) < 1e-12


@pytest.mark.parametrize("N", [1, 2, 5, 10, 30, 50, 256])
def test_eq10_endpoints_and_range(N):
    # "delta_0 corresponds to the next MPC step and delta_{NL-1} = H corresponds to the end of the horizon"
    s = np.linspace(0.0, 1.0, 5).astype(np.float32)
    n = landmark_steps(s, N)
    assert n[0] == 1 and n[-1] == N
    assert all(1 <= v <= N for v in n) and all(n[i] <= n[i + 1] for i in range(4))


def test_eq10_hand_values():
    # N = 50: s (N-1) = 0, 12.25, 24.5, 36.75, 49  ->  n = 1, 13, 25, 37, 50
    assert landmark_steps([0.0, 0.25, 0.5, 0.75, 1.0], 50) == [1, 13, 25, 37, 50]
    # N = 10: 0, 2.25, 4.5, 6.75, 9 -> 1, 3, 5, 7, 10
    assert landmark_steps([0.0, 0.25, 0.5, 0.75, 1.0], 10) == [1, 3, 5, 7, 10]


def make_x(B, N, c_of_time, d_of_lookahead, t):
    """Solver output of a solve at time t whose CoM prediction for time t+n is c_true(t+n) + d(n)."""
    x = np.zeros((B, N, 13))
    for n in range(1, N + 1):
        x[:, n - 1, 3:6] = c_of_time(t + n) + d_of_lookahead(n)
    x[:, :, 0:3] = 7.0          # other entries must not matter
    x[:, :, 6:] = -3.0
    return x


def c_true(t):
    return np.array([0.3 * t, -0.1 * t, 0.9 + 0.01 * t])


def test_hand_worked_reward_all_landmarks():
    # N = 5, s = (0, .5, 1) -> n = (1, 3, 5).  Every solve over-predicts x by 0.01 n (lookahead n), so at any
    # time t >= 5 the errors are e_l = (-0.01 n_l, 0, 0).  With Qc = (4,1,1), sigma = 0.1, alpha = (.5,.3,.2):
    #   sum = [0.5*4*0.01^2 + 0.3*4*0.03^2 + 0.2*4*0.05^2] / 0.01 = [0.0002 + 0.00108 + 0.002] / 0.01 = 0.328
    B, N = 2, 5
    o = LandmarkOracle(B, N, [0.0, 0.5, 1.0], [0.5, 0.3, 0.2], [4.0, 1.0, 1.0], 0.1)
    d = lambda n: np.array([0.01 * n, 0.0, 0.0])
    for t in range(9):
        tt = np.full(B, t)
        r, used = o.reward(np.tile(c_true(t), (B, 1)), tt)
        if t >= 5:
            assert used.tolist() == [3, 3]
            assert abs(r[0] - math.exp(-0.328)) < 1e-7 and r[1] == r[0]   # parameters are float32 values
        o.push(make_x(B, N, c_true, d, t), tt)


def test_partial_availability_at_episode_start():
    # t = 0: nothing stored -> sum over an empty set, r = 1.  t = 1: only the n = 1 landmark of the solve at 0;
    # t = 3: n = 1 (solve at 2) and n = 3 (solve at 0).  Same errors as above: -log r = 0.02, then 0.02 + 0.108.
    B, N = 1, 5
    o = LandmarkOracle(B, N, [0.0, 0.5, 1.0], [0.5, 0.3, 0.2], [4.0, 1.0, 1.0], 0.1)
    d = lambda n: np.array([0.01 * n, 0.0, 0.0])
    expect = {0: (0, 0.0), 1: (1, 0.02), 2: (1, 0.02), 3: (2, 0.128), 4: (2, 0.128), 5: (3, 0.328)}
    for t in range(6):
        r, used = o.reward(c_true(t)[None], [t])
        assert used[0] == expect[t][0]
        assert abs(-math.log(r[0]) - expect[t][1]) < 1e-7
        o.push(make_x(B, N, c_true, d, t), [t])


def test_remark1_next_step_supervision():
    # alpha = (1, 0, ..., 0): the reward is strict next-step tracking, exp(-|c_t - c_hat^{t-1}(dt)|^2 / sigma^2),
    # whatever the far landmarks say.
    B, N = 1, 10
    o = LandmarkOracle(B, N, np.linspace(0, 1, 5), [1.0, 0, 0, 0, 0], [1.0, 1.0, 1.0], 0.2)
    rng = np.random.default_rng(3)
    prev_next = None
    for t in range(12):
        c = rng.normal(size=3)
        r, _ = o.reward(c[None], [t])
        if prev_next is not None:
            assert abs(r[0] - math.exp(-np.sum((c - prev_next) ** 2) / 0.04)) < 1e-12
        x = rng.normal(size=(B, N, 13))
        prev_next = x[0, 0, 3:6].copy()         # x_1 of this solve = prediction for t + 1
        o.push(x, [t])


def test_remark1_uniform_weights_average():
    # alpha_l = 1/NL: -log r = mean over the landmarks of |e_l|^2 / sigma^2
    B, N, NL = 1, 9, 3
    o = LandmarkOracle(B, N, [0.0, 0.5, 1.0], [1 / 3] * 3, [1.0, 1.0, 1.0], 1.0)
    rng = np.random.default_rng(5)
    xs = []
    for t in range(10):
        x = rng.normal(size=(B, N, 13))
        xs.append(x)
        o.push(x, [t])
    t = 10
    c = rng.normal(size=3)
    r, used = o.reward(c[None], [t])
    errs = [np.sum((c - xs[t - n][0, n - 1, 3:6]) ** 2) for n in (1, 5, 9)]
    assert used[0] == 3
    assert abs(-math.log(r[0]) - np.mean(errs)) < 1e-6      # 1/3 is rounded to float32 in the oracle


def test_bounds_monotonicity_and_reset():
    B, N = 3, 6
    a = paper_alpha()
    o = LandmarkOracle(B, N, np.linspace(0, 1, 5), a, [1.0, 1.0, 1.0], 0.05)
    x = np.zeros((B, N, 13))
    for t in range(7):
        o.push(x, np.full(B, t))
    t = np.full(B, 7)
    r0, used = o.reward(np.zeros((B, 3)), t)
    assert used.tolist() == [5] * B and np.all(r0 == 1.0)              # zero error: r = 1 (upper bound)
    r1, _ = o.reward(np.full((B, 3), 0.01), t)
    r2, _ = o.reward(np.full((B, 3), 0.02), t)
    assert np.all((0 < r2) & (r2 < r1) & (r1 < 1.0))                   # r in (0, 1], decreasing in the error
    # the same error hurts more on the nearest landmark than on the farthest (prediction confidence)
    near = LandmarkOracle(1, N, np.linspace(0, 1, 5), a, [1.0] * 3, 0.05)
    far = LandmarkOracle(1, N, np.linspace(0, 1, 5), a, [1.0] * 3, 0.05)
    xn = np.zeros((1, N, 13)); xn[0, 0, 3] = 0.03                       # error in x_1 only
    xf = np.zeros((1, N, 13)); xf[0, N - 1, 3] = 0.03                   # error in x_N only
    near.push(xn, [0]); far.push(xf, [0])
    rn, _ = near.reward(np.zeros((1, 3)), [1])
    rf, _ = far.reward(np.zeros((1, 3)), [N])
    assert rn[0] < rf[0] < 1.0
    assert abs(math.log(rn[0]) / math.log(rf[0]) - a[0] / a[-1]) < 1e-5
    # reset of env 1 only
    o.reset([False, True, False])
    r, used = o.reward(np.full((B, 3), 0.01), t)
    assert used.tolist() == [5, 0, 5] and r[1] == 1.0 and r[0] == r1[0]
