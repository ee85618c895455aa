"""pinmpc_split_solve_static — the entry point that allocates nothing (scratch = a static device array of the library) —
against the existing path pinmpc_split_solve with a caller-owned workspace: same inputs, same kernels, so the outputs
agree within the tolerances of tests/test_gpu_split.py (in fact bit for bit).  Two calls in a row with different
shapes (the second finds the first call's contents in the shared array), then the first problem once more.

Collected last on purpose (file name): the suite runs with pytest -x.  Passes alone in a fresh process and after the
other tests."""
import numpy as np
import pytest

import gen
import oracle

pytestmark = pytest.mark.gpu


def _problem(cfg, B, N, seed):
    import torch
    w = gen.make_config(cfg, B=B, N=N)
    A, Bm, c = oracle.assemble(w.nu, w.n_wrench, w.n_force, w.dt, w.yaw, w.foot_r, w.mass, w.inertia, w.ext_wrench)
    rng = np.random.default_rng(seed)
    u_prev = (w.u_ref[:, 0] + rng.normal(size=(B, w.nu))).astype(np.float32)
    d = lambda a, t=np.float32: None if a is None else torch.from_numpy(np.ascontiguousarray(a, dtype=t)).cuda()
    return w, (d(A), d(Bm), d(c), d(w.x0), d(u_prev), d(w.x_ref), d(w.u_ref), d(w.contact, np.uint8))


def _both(w, dev, iters):
    """(existing path, static path) -> ((xi, z, r), (xi, z, r)) as numpy; also that the static call allocated nothing."""
    import torch
    from paper_2606_05687_b200 import binding, make_layout
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    ref = binding.split_solve(*dev, lay, w.Qdiag, w.Rdiag, w.rho, iters)
    ref = tuple(t.cpu().numpy() for t in ref)
    n = 13 + w.nu
    xi = torch.full((w.B, w.N, n), float("nan"), device="cuda"); z = torch.full_like(xi, float("nan"))
    r = torch.full((w.B,), float("nan"), device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    binding.split_solve_static(*dev, lay, w.Qdiag, w.Rdiag, w.rho, iters, xi, z, r)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0              # no device memory was taken by the call
    return ref, (xi.cpu().numpy(), z.cpu().numpy(), r.cpu().numpy())


def _check(w, ref, got):
    nx = 13
    for name, a, b in (("xi", ref[0], got[0]), ("z", ref[1], got[1])):
        assert np.all(np.isfinite(b)), name
        for e in range(w.B):
            tx = 1e-4 * (1 + np.abs(a[e][:, :nx]).max()); tu = 1e-3 * (1 + np.abs(a[e][:, nx:]).max())
            assert np.abs(a[e][:, :nx] - b[e][:, :nx]).max() <= tx, (name, e)
            assert np.abs(a[e][:, nx:] - b[e][:, nx:]).max() <= tu, (name, e)
    assert np.all(np.abs(ref[2] - got[2]) <= 1e-3 * ref[2] + 1e-3 * (1 + np.abs(ref[0][:, :, nx:]).max(axis=(1, 2))))
    assert np.all(got[2] > 0)


def test_static_scratch_entry_point_matches_the_workspace_path():
    from paper_2606_05687_b200 import binding
    assert binding.load().pinmpc_split_static_bytes() == 16 << 20
    wa, da = _problem(0, 24, 10, 1)          # nu = 12
    wb, db = _problem(3, 7, 12, 2)           # nu = 18, external wrench: another layout of the shared array
    ra, ga = _both(wa, da, 40)
    _check(wa, ra, ga)
    rb, gb = _both(wb, db, 30)               # second call in a row: the array holds the first call's contents
    _check(wb, rb, gb)
    ra2, ga2 = _both(wa, da, 40)             # and back: identical to the first call
    _check(wa, ra2, ga2)
    assert np.array_equal(ga[0], ga2[0]) and np.array_equal(ga[1], ga2[1])


def test_static_scratch_rejects_what_does_not_fit():
    import torch
    from paper_2606_05687_b200 import binding, make_layout
    B, N, nu = 4096, 50, 12                  # 1.05 GB of workspace: far beyond the 16 MiB array
    lay = make_layout(2, 0)
    t = torch.zeros(8, device="cuda")        # never read: the size check comes first
    u8 = torch.zeros(8, dtype=torch.uint8, device="cuda")

    class Shape:                             # stands in for B_k: only the shape decides, nothing is read before the check
        shape = (B, N, 13, nu); device = t.device
        data_ptr = staticmethod(t.data_ptr)
    with pytest.raises(binding.PinmpcError) as ei:
        binding.split_solve_static(t, Shape, None, t, None, t, None, u8, lay, [1.0] * 13, [1.0] * nu, 1.0, 5, t, t, t)
    assert ei.value.status == binding.EALLOC
    msg = str(ei.value)
    assert "PINMPC_SPLIT_STATIC_BYTES" in msg and str(16 << 20) in msg
