"""Pins for oracle O1 (dynamics assembly).  SURVEY.md 8(c)-O1 / T5; BASELINE.json config 0."""
import os

import numpy as np
import pytest

import gen
import oracle
from refcheck import NX, rotz, srb_ode

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _one_stage(yaw, r, mass, Ib, dt, nu=12, ext=None):
    nw, nf = 2, (2 if nu == 18 else 0)
    r = np.asarray(r, float).reshape(1, 1, nw + nf, 3)
    A, Bm, c = oracle.assemble(nu, nw, nf, dt, np.array([[yaw]]), r, np.array([mass]),
                               np.asarray(Ib, float).reshape(1, 3, 3),
                               None if ext is None else np.asarray(ext, float).reshape(1, 1, 6))
    return A[0, 0], Bm[0, 0], c[0, 0]


def test_golden_hand_derived_stage():
    """Every value in tests/golden/assembly_yaw90.txt was derived by hand (see its header)."""
    r = [[0.1, 0.2, -0.9], [0.0, 0.0, -0.9]]
    A, Bm, _ = _one_stage(np.pi / 2, r, 50.0, np.diag([1.0, 2.0, 4.0]), 0.04)
    n = 0
    for line in open(os.path.join(GOLD, "assembly_yaw90.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, i, j, v = line.split()
        M = A if name == "A" else Bm
        assert abs(M[int(i), int(j)] - float(v)) < 1e-15, line
        n += 1
    assert n == 34


def test_yaw_zero_structure():
    """yaw = 0 => R_z = I: A[0:3,6:9] = dt I, I_w^-1 = I_b^-1; sparsity pattern of A and B."""
    Ib = np.diag([0.7, 1.3, 2.9]); dt = 0.03
    r = np.array([[0.05, 0.1, -0.9], [-0.02, -0.12, -0.88]])
    A, Bm, c = _one_stage(0.0, r, 42.0, Ib, dt)
    Aexp = np.eye(NX); Aexp[0:3, 6:9] = dt * np.eye(3); Aexp[3:6, 9:12] = dt * np.eye(3); Aexp[11, 12] = dt
    np.testing.assert_allclose(A, Aexp, atol=1e-16)
    assert np.all(Bm[0:6] == 0) and np.all(Bm[12] == 0) and np.all(c == 0)
    np.testing.assert_allclose(Bm[6:9, 6:9], dt * np.linalg.inv(Ib), atol=1e-16)
    np.testing.assert_allclose(Bm[6:9, 9:12], dt * np.linalg.inv(Ib), atol=1e-16)
    np.testing.assert_allclose(Bm[9:12, 0:3], dt / 42.0 * np.eye(3), atol=1e-18)
    assert np.all(Bm[9:12, 6:12] == 0)


@pytest.mark.parametrize("nu", [12, 18])
def test_one_step_equals_forward_euler_of_the_ode(nu):
    """x + dt f(x,u) with f the continuous ODE of BASELINE.json config 0, coded with np.cross and
    np.linalg.solve, must equal A x + B u + c for random x,u (pins every block, sign and index)."""
    rng = np.random.default_rng(7)
    nw, nf = 2, (2 if nu == 18 else 0)
    for _ in range(20):
        yaw = rng.uniform(-np.pi, np.pi); dt = rng.uniform(0.01, 0.05); mass = rng.uniform(30, 70)
        G = rng.normal(size=(3, 3)); Ib = G @ G.T + 0.5 * np.eye(3)            # full SPD inertia
        r = rng.uniform(-1, 1, (nw + nf, 3)); ext = rng.normal(size=6) * 10
        x = rng.normal(size=NX); u = rng.normal(size=nu) * 50
        A, Bm, c = _one_stage(yaw, r, mass, Ib, dt, nu=nu, ext=ext)
        euler = x + dt * srb_ode(x, u, yaw, r, mass, Ib, nw, nf, ext=ext)
        np.testing.assert_allclose(A @ x + Bm @ u + c, euler, rtol=0, atol=1e-11)


def test_cross_product_block_and_gravity_state():
    rng = np.random.default_rng(3)
    Ib = np.diag([1.0, 2.0, 3.0]); yaw = 0.8; dt = 0.04; m = 55.0
    r = rng.uniform(-1, 1, (2, 3))
    A, Bm, _ = _one_stage(yaw, r, m, Ib, dt)
    Iwi = rotz(yaw) @ np.linalg.inv(Ib) @ rotz(yaw).T
    f = rng.normal(size=3)
    for i in range(2):
        np.testing.assert_allclose(Bm[6:9, 3 * i:3 * i + 3] @ f, dt * Iwi @ np.cross(r[i], f), atol=1e-14)
    # the constant-gravity state: x[12] stays put, and only v_z sees it
    x = rng.normal(size=NX); x[12] = -9.81
    assert (A @ x)[12] == -9.81
    np.testing.assert_allclose(A[:, 12], np.eye(NX)[12] + dt * np.eye(NX)[11], atol=0)


def test_batched_matches_per_stage_and_generator_shapes():
    w = gen.make_config(0)
    A, Bm, c = oracle.assemble(w.nu, w.n_wrench, w.n_force, w.dt, w.yaw, w.foot_r, w.mass, w.inertia)
    assert A.shape == (64, 10, 13, 13) and Bm.shape == (64, 10, 13, 12) and c.shape == (64, 10, 13)
    b, k = 17, 6
    A1, B1, c1 = _one_stage(float(w.yaw[b, k]), w.foot_r[b, k].astype(float), float(w.mass[b]),
                            w.inertia[b].astype(float), w.dt)
    assert np.array_equal(A[b, k], A1) and np.array_equal(Bm[b, k], B1) and np.array_equal(c[b, k], c1)
    # swing contacts still get their B columns (SURVEY 8(c)-O1 last bullet)
    sw = np.argwhere(w.contact[..., 0] == 0)[0]
    assert np.any(Bm[sw[0], sw[1], 6:9, 0:3] != 0)
