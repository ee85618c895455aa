"""Pins of oracle/centroidal.py (the paper's 9-state centroidal model, eq. (1)-(4)).

What physics and the already pinned 13-state assembly fix: free fall in closed form, a force through the CoM and a pure
couple, and — after the change of variables l_G = m v, k_G = I_w omega — the translational and angular rows of the
single-rigid-body model of oracle.assemble (C, pinned in tests/test_oracle_assembly.py)."""
import numpy as np

import gen
import oracle
from oracle import centroidal as cd


def rollout(A, Bm, e, x0, u):
    x = [np.asarray(x0, dtype=float)]
    for k in range(A.shape[0]):
        x.append(A[k] @ x[-1] + Bm[k] @ u[k] + e[k])
    return np.array(x)


def test_free_fall_closed_form():
    m, dt, N = 41.5, 0.03, 25
    A, Bm, e = cd.assemble(2, 0, dt, [m], np.zeros((1, N, 2, 3)))
    c0, v0 = np.array([0.1, -0.2, 0.9]), np.array([0.4, 0.1, 1.5])
    x = rollout(A[0], Bm[0], e[0], np.concatenate([c0, m * v0, [0.3, 0.2, 0.1]]), np.zeros((N, 12)))
    n = np.arange(N + 1)[:, None]
    g = np.array([0.0, 0.0, -9.81])
    assert np.allclose(x[:, 3:6], m * (v0 + n * dt * g), atol=1e-10)                       # l = m v, dv/dt = g
    # explicit Euler position: c_n = c_0 + n dt v_0 + dt^2 g n (n - 1) / 2
    assert np.allclose(x[:, 0:3], c0 + n * dt * v0 + dt * dt * g * n * (n - 1) / 2, atol=1e-10)
    assert np.allclose(x[:, 6:9], [0.3, 0.2, 0.1])                                         # no wrench: k_G is conserved


def test_force_through_the_com_and_pure_couple():
    m, dt = 50.0, 0.04
    r = np.array([[0.2, -0.1, -0.9], [-0.2, 0.1, 0.9]])                                   # two opposite levers
    A, Bm, e = cd.assemble(2, 0, dt, [m], r[None, None])
    x0 = np.zeros(9)
    u = np.zeros(12); u[0:3] = 7.0 * r[0]                                                  # force along its own lever
    x1 = A[0, 0] @ x0 + Bm[0, 0] @ u + e[0, 0]
    assert np.allclose(x1[6:9], 0.0, atol=1e-12)                                           # no moment about the CoM
    assert np.allclose(x1[3:6], dt * (7.0 * r[0] + [0, 0, -m * 9.81]))
    f = np.array([3.0, -5.0, 11.0])
    u = np.zeros(12); u[0:3] = f; u[3:6] = -f                                              # couple at +r, -r... levers r0 and r1 = -r0
    x1 = A[0, 0] @ x0 + Bm[0, 0] @ u + e[0, 0]
    assert np.allclose(x1[3:6] - e[0, 0, 3:6], 0.0, atol=1e-12)                            # net force zero
    tau = f[[1, 2, 0]] * 0 + np.array([r[0][1] * f[2] - r[0][2] * f[1], r[0][2] * f[0] - r[0][0] * f[2], r[0][0] * f[1] - r[0][1] * f[0]])
    assert np.allclose(x1[6:9], 2 * dt * tau, atol=1e-12)                                  # 2 dt r x f
    u = np.zeros(12); u[6:9] = [1.0, 2.0, 3.0]                                             # a contact moment goes straight into k_G
    x1 = A[0, 0] @ x0 + Bm[0, 0] @ u + e[0, 0]
    assert np.allclose(x1[6:9], dt * np.array([1.0, 2.0, 3.0])) and np.allclose(x1[0:3], 0.0)


def test_agrees_with_the_single_rigid_body_assembly():
    """13-state SRB: x = [Theta, p, omega, v, g].  With l = m v and k = I_w omega its p-, v- and omega-rows are eq. (2)-(4)."""
    for cfg in (0, 3):
        w = gen.make_config(cfg, B=3, N=7)
        A13, B13, c13 = oracle.assemble(w.nu, w.n_wrench, w.n_force, w.dt, w.yaw, w.foot_r, w.mass, w.inertia, None)
        A, Bm, e = cd.assemble(w.n_wrench, w.n_force, w.dt, w.mass, w.foot_r)
        for b in range(w.B):
            m = float(w.mass[b])
            for k in range(w.N):
                # position rows: p+ = p + dt v  <->  c+ = c + dt/m l
                assert np.allclose(A13[b, k, 3:6, 9:12] / m, A[b, k, 0:3, 3:6], atol=1e-12)
                # velocity rows times m: m v+ = m v + dt sum f (+ dt m g through the gravity state)
                assert np.allclose(m * B13[b, k, 9:12], Bm[b, k, 3:6], atol=1e-9)
                assert np.allclose(m * A13[b, k, 9:12, 12] * -9.81, e[b, k, 3:6], atol=1e-9)
                # angular rows times I_w: I_w omega+ = I_w omega + dt sum (r x f + tau); I_w = R_z I_b R_z^T
                cs, sn = np.cos(w.yaw[b, k]), np.sin(w.yaw[b, k])
                Rz = np.array([[cs, -sn, 0], [sn, cs, 0], [0, 0, 1.0]])
                Iw = Rz @ np.asarray(w.inertia[b], dtype=float) @ Rz.T
                assert np.allclose(Iw @ B13[b, k, 6:9], Bm[b, k, 6:9], atol=1e-9)
        A9, B9, e9 = cd.pad13(A, Bm, e)
        assert A9.shape == A13.shape and np.all(A9[..., 9:, :9] == 0) and np.all(B9[..., 9:, :] == 0)
