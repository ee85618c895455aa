"""The seeded input generator: shapes, determinism and the structure DESIGN.md's recipe promises."""
import numpy as np

import gen


def test_config0_shapes_seed_and_ranges():
    w = gen.make_config(0)
    w2 = gen.make_config(0)
    assert (w.B, w.N, w.nu, w.dt, w.iters, w.rho) == (64, 10, 12, 0.04, 50, 1.0)
    for a in gen.Workload.ARRAYS:
        va, vb = getattr(w, a), getattr(w2, a)
        assert (va is None and vb is None) or np.array_equal(va, vb)
    assert w.x0.dtype == np.float32 and w.contact.dtype == np.uint8
    assert w.x_ref.shape == (64, 10, 13) and w.u_ref.shape == (64, 10, 12) and w.foot_r.shape == (64, 10, 2, 3)
    assert np.all((w.mass >= 35) & (w.mass <= 60))
    d = np.diagonal(w.inertia, axis1=1, axis2=2)
    assert np.all((d >= 0.5) & (d <= 3.0)) and np.all(w.inertia - np.stack([np.diag(x) for x in d]) == 0)
    assert np.all(w.x0[:, 12] == np.float32(-9.81)) and np.all(w.x_ref[:, :, 12] == np.float32(-9.81))
    assert np.all(w.x_ref[:, :, 5] == np.float32(0.9))
    assert np.all(np.abs(w.foot_r[..., 2] + 0.9) <= 0.05 + 1e-6)


def test_alternating_gait_and_weight_sharing_reference():
    w = gen.make_config(1, B=128)
    assert np.all(w.contact.sum(-1) == 1)                         # 50 % duty, alternating: one stance foot
    fz = w.u_ref[..., [2, 5]]
    np.testing.assert_allclose(fz.sum(-1), np.broadcast_to(w.mass[:, None] * 9.81, fz.shape[:2]), rtol=1e-6)
    assert np.all((fz > 0) == (w.contact > 0))
    other = np.delete(w.u_ref, [2, 5], axis=-1)
    assert np.all(other == 0)
    assert len(np.unique(np.diff(w.contact[:, :, 0].astype(int), axis=1))) > 1   # gait switches occur


def test_stance_foot_is_fixed_in_the_world():
    w = gen.make_config(2, B=32)
    p = w.x_ref[:, :, 3:6].astype(np.float64)                     # p_ref at stages 1..N
    for b in range(8):
        for i in range(2):
            for k in range(2, w.N):
                if w.contact[b, k, i] and w.contact[b, k - 1, i]:
                    # world position = r + p_ref(stage k); x_ref[k-1] holds p_ref at stage k
                    a = w.foot_r[b, k, i] + p[b, k - 1]
                    bb = w.foot_r[b, k - 1, i] + p[b, k - 2]
                    assert np.max(np.abs(a - bb)) < 1e-5


def test_loco_manipulation_extras_and_subset():
    w = gen.make_config(3, B=64)
    assert w.nu == 18 and w.n_force == 2 and w.ext_wrench.shape == (64, 30, 6)
    assert np.all(w.contact[..., 2:] == 1) and np.all(w.u_ref[..., 12:] == 0)
    Fn = np.linalg.norm(w.ext_wrench[..., :3], axis=-1)
    assert np.all(Fn <= 200 + 1e-3) and np.all(np.abs(Fn - Fn[:, :1]) < 1e-3)    # constant magnitude per env
    s = gen.subset(w, [5, 9])
    assert s.B == 2 and np.array_equal(s.x0[1], w.x0[9]) and np.array_equal(s.ext_wrench[0], w.ext_wrench[5])


def test_different_configs_use_different_seeds():
    assert not np.array_equal(gen.make_config(1, B=8, N=10).mass, gen.make_config(2, B=8, N=10).mass)


def test_centroidal_view_is_the_same_episode_in_nine_states():
    w = gen.make_config(3, B=5, N=8)
    v = gen.centroidal_view(w)
    assert v["x0"].shape == (5, 9) and v["x_ref"].shape == (5, 8, 9) and v["Qdiag"].shape == (9,)
    assert np.allclose(v["x0"][:, 0:3], w.x0[:, 3:6])
    assert np.allclose(v["x_ref"][..., 3:6], w.mass[:, None, None] * w.x_ref[..., 9:12], rtol=1e-6)
    assert np.all(v["Qdiag"] > 0) and np.all(v["x_lo"] <= v["x_hi"])
    assert np.isinf(v["x_lo"]).sum() == 7 and np.isinf(v["x_hi"]).sum() == 7
