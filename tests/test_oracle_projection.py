"""Pins for oracle O4 (exact Euclidean projection onto U_k).  SURVEY.md T4, T8, T9."""
import os

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import oracle
from refcheck import brute_project_wrench, wrench_set_inequalities

GOLD = os.path.join(os.path.dirname(__file__), "golden")
LAY = oracle.Layout(2, 0, 0.5, 600.0, 0.02, 0.02, 0.01, 150.0)
LAY_H = oracle.Layout(2, 2, 0.5, 600.0, 0.02, 0.02, 0.01, 150.0)


def proj_foot(f, m, lay=LAY):
    v = np.zeros((1, 12)); v[0, 0:3] = f; v[0, 6:9] = m
    z = oracle.project(lay, np.array([[1, 0]], np.uint8), v)
    assert np.all(z[0, 3:6] == 0) and np.all(z[0, 9:12] == 0)      # the swing foot is zeroed
    return z[0, 0:3], z[0, 6:9]


def test_golden_hand_derived_cases():
    n = 0
    for line in open(os.path.join(GOLD, "projection_cases.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [float(t) for t in line.split("#")[0].split()]
        fo, mo = proj_foot(v[0:3], v[3:6])
        np.testing.assert_allclose(np.concatenate([fo, mo]), v[6:12], rtol=0, atol=1e-12, err_msg=line)
        n += 1
    assert n == 11


def _random_points(rng, n):
    """Mix of scales so that every face (apex, cap, 1..5 clipped coordinates) is hit."""
    pts = []
    for _ in range(n):
        kind = rng.integers(0, 4)
        fz = [rng.normal() * 300, rng.uniform(-50, 700), rng.uniform(500, 900), rng.normal() * 5][kind]
        f = np.array([rng.normal() * [200, 50, 400, 3][kind], rng.normal() * [200, 50, 400, 3][kind], fz])
        m = rng.normal(size=3) * [10, 2, 20, 0.1][kind]
        pts.append((f, m))
    return pts


def test_matches_brute_force_face_enumeration():
    rng = np.random.default_rng(5)
    faces = set()
    for f, m in _random_points(rng, 400):
        fo, mo = proj_foot(f, m)
        fb, mb = brute_project_wrench(f, m, 0.5, 600.0, 0.02, 0.02, 0.01)
        np.testing.assert_allclose(np.concatenate([fo, mo]), np.concatenate([fb, mb]), rtol=0, atol=1e-9)
        y = np.array([fo[0], fo[1], mo[0], mo[1], mo[2]]); wv = np.array([.5, .5, .02, .02, .01]) * fo[2]
        faces.add((int(np.sum(np.abs(np.abs(y) - wv) < 1e-12)), fo[2] == 0.0, fo[2] == 600.0))
    assert len(faces) >= 8           # the sample really exercised many different faces


def test_other_layout_constants_against_brute_force():
    rng = np.random.default_rng(9)
    lay = oracle.Layout(2, 0, 0.8, 250.0, 0.05, 0.11, 0.3, 150.0)
    for f, m in _random_points(rng, 150):
        fo, mo = proj_foot(f, m, lay)
        fb, mb = brute_project_wrench(f, m, 0.8, 250.0, 0.05, 0.11, 0.3)
        np.testing.assert_allclose(np.concatenate([fo, mo]), np.concatenate([fb, mb]), rtol=0, atol=1e-9)


def test_against_scipy_slsqp():
    from scipy.optimize import minimize
    rng = np.random.default_rng(1)
    C, d = wrench_set_inequalities(0.5, 600.0, 0.02, 0.02, 0.01)
    for f, m in _random_points(rng, 25):
        a = np.concatenate([f, m])
        res = minimize(lambda v: 0.5 * np.sum((v - a) ** 2), np.array([0, 0, 1.0, 0, 0, 0]), jac=lambda v: v - a,
                       constraints=[{"type": "ineq", "fun": lambda v: d - C @ v, "jac": lambda v: -C}],
                       method="SLSQP", options={"ftol": 1e-14, "maxiter": 300})
        fo, mo = proj_foot(f, m)
        assert np.max(np.abs(np.concatenate([fo, mo]) - res.x)) < 1e-5 * (1 + np.max(np.abs(a)))


finite = st.floats(-2000, 2000, allow_nan=False, allow_infinity=False)


@settings(max_examples=300, deadline=None)
@given(st.tuples(finite, finite, finite, finite, finite, finite), st.tuples(finite, finite, finite, finite, finite, finite))
def test_property_feasible_idempotent_nonexpansive(a, b):
    a = np.array(a); b = np.array(b)
    C, d = wrench_set_inequalities(0.5, 600.0, 0.02, 0.02, 0.01)
    pa = np.concatenate(proj_foot(a[:3], a[3:])); pb = np.concatenate(proj_foot(b[:3], b[3:]))
    assert np.all(C @ pa <= d + 1e-9)                                        # feasible
    paa = np.concatenate(proj_foot(pa[:3], pa[3:]))
    assert np.max(np.abs(paa - pa)) <= 1e-10 * (1 + np.max(np.abs(pa)))      # idempotent
    assert np.linalg.norm(pa - pb) <= np.linalg.norm(a - b) * (1 + 1e-12) + 1e-12   # non-expansive
    # variational inequality: <a - P(a), v - P(a)> <= 0 for every v in the set (here v = P(b))
    assert np.dot(a - pa, pb - pa) <= 1e-7 * (1 + np.linalg.norm(a) * np.linalg.norm(b))


def test_moreau_decomposition_for_the_uncapped_cone():
    """f_max = inf makes W a closed convex cone: a = P_W(a) + P_{W polar}(a) with <.,.> = 0."""
    rng = np.random.default_rng(2)
    lay = oracle.Layout(2, 0, 0.5, 1e300, 0.02, 0.02, 0.01, 150.0)
    for f, m in _random_points(rng, 200):
        a = np.concatenate([f, m])
        p = np.concatenate(proj_foot(f, m, lay))
        q = a - p                                            # must lie in the polar cone
        assert abs(np.dot(p, q)) < 1e-8 * (1 + np.dot(a, a))
        # polar cone test: <q, v> <= 0 for the extreme rays v of W (t=1, y_i = +-w_i)
        for sg in np.ndindex(2, 2, 2, 2, 2):
            s = 2 * np.array(sg) - 1.0
            ray = np.array([s[0] * .5, s[1] * .5, 1.0, s[2] * .02, s[3] * .02, s[4] * .01])
            assert np.dot(q, ray) < 1e-8 * (1 + np.linalg.norm(a))


def test_swing_zero_and_hand_box():
    rng = np.random.default_rng(4)
    v = rng.normal(size=(50, 18)) * 200
    contact = rng.integers(0, 2, (50, 4)).astype(np.uint8)
    z = oracle.project(LAY_H, contact, v)
    for i in range(50):
        for foot in range(2):
            blk = np.concatenate([z[i, 3 * foot:3 * foot + 3], z[i, 6 + 3 * foot:9 + 3 * foot]])
            if not contact[i, foot]:
                assert np.all(blk == 0.0)                      # T8: swing => exactly zero
            else:
                fb, mb = brute_project_wrench(v[i, 3 * foot:3 * foot + 3], v[i, 6 + 3 * foot:9 + 3 * foot],
                                              0.5, 600.0, 0.02, 0.02, 0.01)
                np.testing.assert_allclose(blk, np.concatenate([fb, mb]), atol=1e-9)
        for h in range(2):
            blk = z[i, 12 + 3 * h:15 + 3 * h]
            exp = np.clip(v[i, 12 + 3 * h:15 + 3 * h], -150, 150) if contact[i, 2 + h] else np.zeros(3)
            assert np.array_equal(blk, exp)
