"""Thin ctypes binding of libpinmpc.so (include/pinmpc.h): argument marshalling only.

Every step of the path (assembly, factorisation, ADMM iterations, projection, residuals) runs in
the CUDA kernels behind the C ABI.  PyTorch is used here for device memory and streams only.
There is no CPU fallback: if the shared library is missing or cannot be loaded this module raises.
The function names mirror the C entry points one to one; `Solver` is a convenience holder that
keeps the borrowed tensors alive.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_char_p, c_float, c_int, c_size_t, c_void_p

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libpinmpc.so")
NX = 13

OK, EINVAL, EALLOC, ECUDA, ESTATE, EUNSUPPORTED = range(6)
METHOD_AUTO, METHOD_DENSE, METHOD_SRB = 0, 1, 2
_STATUS = {0: "PINMPC_OK", 1: "PINMPC_EINVAL", 2: "PINMPC_EALLOC", 3: "PINMPC_ECUDA", 4: "PINMPC_ESTATE",
           5: "PINMPC_EUNSUPPORTED"}

EXPORTS = ("pinmpc_workspace_bytes", "pinmpc_workspace_bytes_method", "pinmpc_create", "pinmpc_set_weights",
           "pinmpc_set_tolerance", "pinmpc_set_method", "pinmpc_set_tuning", "pinmpc_set_horizon_chunks", "pinmpc_get_launch_shape", "pinmpc_set_problem", "pinmpc_set_dynamics", "pinmpc_solve",
           "pinmpc_get", "pinmpc_get_aux", "pinmpc_get_dynamics", "pinmpc_get_srb_assembly", "pinmpc_last_launch_count", "pinmpc_last_error",
           "pinmpc_destroy", "pinmpc_set_profiling", "pinmpc_get_kernel_ms",
           "pinmpc_set_warm_start", "pinmpc_shift_aux", "pinmpc_landmark_ring_bytes", "pinmpc_landmark_reset", "pinmpc_landmark_push",
           "pinmpc_landmark_push_solver", "pinmpc_landmark_reward", "pinmpc_split_workspace_bytes", "pinmpc_split_solve",
           "pinmpc_split_workspace_bytes_ex", "pinmpc_split_solve_ex", "pinmpc_assemble_centroidal",
           "pinmpc_split_static_bytes", "pinmpc_split_solve_static")
MAX_LANDMARKS = 8


class PinmpcError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class Layout(ctypes.Structure):
    _fields_ = [("n_wrench", c_int), ("n_force", c_int), ("mu", c_float), ("fz_max", c_float),
                ("mx_coef", c_float), ("my_coef", c_float), ("mz_coef", c_float), ("hand_fmax", c_float)]


class Problem(ctypes.Structure):
    _fields_ = [(n, c_void_p) for n in ("x0", "x_ref", "u_ref", "contact", "foot_r", "yaw", "mass", "inertia",
                                        "ext_wrench")]


class SplitProblem(ctypes.Structure):
    _fields_ = [(n, c_void_p) for n in ("A", "Bm", "c", "x0", "u_prev", "x_ref", "u_ref", "contact")]


class SplitOptions(ctypes.Structure):
    _fields_ = [("h_scale_x", POINTER(c_float)), ("scale_u", c_float), ("accel", c_int), ("eta", c_float), ("d_restarts", c_void_p),
                ("nx", c_int), ("h_x_lo", POINTER(c_float)), ("h_x_hi", POINTER(c_float))]


class LandmarkCfg(ctypes.Structure):
    _fields_ = [("n_landmarks", c_int), ("s", c_float * MAX_LANDMARKS), ("alpha", c_float * MAX_LANDMARKS),
                ("Qc", c_float * 3), ("sigma_c", c_float)]


_lib = None


def load():
    """Load libpinmpc.so (built in-tree by paper_2606_05687_b200.build / __graft_entry__.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_05687_b200.build` (needs nvcc). "
                          "There is no CPU fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    lib.pinmpc_workspace_bytes.restype = c_size_t
    lib.pinmpc_workspace_bytes.argtypes = [c_int, c_int, c_int, c_int, POINTER(Layout)]
    lib.pinmpc_workspace_bytes_method.restype = c_size_t
    lib.pinmpc_workspace_bytes_method.argtypes = [c_int, c_int, c_int, c_int, POINTER(Layout), c_int]
    lib.pinmpc_create.restype = c_int
    lib.pinmpc_create.argtypes = [POINTER(c_void_p), c_int, c_int, c_int, c_int, POINTER(Layout), c_float, c_int,
                                  c_void_p, c_size_t]
    lib.pinmpc_set_weights.restype = c_int
    lib.pinmpc_set_weights.argtypes = [c_void_p, POINTER(c_float), POINTER(c_float), c_float]
    lib.pinmpc_set_tolerance.restype = c_int
    lib.pinmpc_set_tolerance.argtypes = [c_void_p, c_float, c_float, c_int]
    lib.pinmpc_set_method.restype = c_int
    lib.pinmpc_set_method.argtypes = [c_void_p, c_int]
    lib.pinmpc_set_tuning.restype = c_int
    lib.pinmpc_set_tuning.argtypes = [c_void_p, c_int]
    lib.pinmpc_set_horizon_chunks.restype = c_int
    lib.pinmpc_set_horizon_chunks.argtypes = [c_void_p, c_int]
    lib.pinmpc_get_launch_shape.restype = c_int
    lib.pinmpc_get_launch_shape.argtypes = [c_void_p, POINTER(c_int), POINTER(c_int)]
    lib.pinmpc_set_problem.restype = c_int
    lib.pinmpc_set_problem.argtypes = [c_void_p, POINTER(Problem)]
    lib.pinmpc_set_dynamics.restype = c_int
    lib.pinmpc_set_dynamics.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pinmpc_solve.restype = c_int
    lib.pinmpc_solve.argtypes = [c_void_p, c_void_p]
    lib.pinmpc_get.restype = c_int
    lib.pinmpc_get.argtypes = [c_void_p] + [c_void_p] * 6
    lib.pinmpc_get_aux.restype = c_int
    lib.pinmpc_get_aux.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pinmpc_get_dynamics.restype = c_int
    lib.pinmpc_get_dynamics.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pinmpc_get_srb_assembly.restype = c_int
    lib.pinmpc_get_srb_assembly.argtypes = [c_void_p] + [c_void_p] * 6
    lib.pinmpc_last_launch_count.restype = c_int
    lib.pinmpc_last_launch_count.argtypes = [c_void_p]
    lib.pinmpc_last_error.restype = c_char_p
    lib.pinmpc_last_error.argtypes = [c_void_p]
    lib.pinmpc_set_warm_start.restype = c_int
    lib.pinmpc_set_warm_start.argtypes = [c_void_p, c_void_p, c_void_p]
    lib.pinmpc_set_profiling.restype = c_int
    lib.pinmpc_set_profiling.argtypes = [c_void_p, c_int]
    lib.pinmpc_get_kernel_ms.restype = c_int
    lib.pinmpc_get_kernel_ms.argtypes = [c_void_p, POINTER(c_float)]
    lib.pinmpc_shift_aux.restype = c_int
    lib.pinmpc_shift_aux.argtypes = [c_void_p, c_int, c_void_p, c_void_p, c_void_p]
    lib.pinmpc_landmark_ring_bytes.restype = c_size_t
    lib.pinmpc_landmark_ring_bytes.argtypes = [c_int, c_int, POINTER(LandmarkCfg)]
    lib.pinmpc_landmark_reset.restype = c_int
    lib.pinmpc_landmark_reset.argtypes = [c_void_p, c_int, c_int, POINTER(LandmarkCfg), c_void_p, c_void_p]
    lib.pinmpc_landmark_push.restype = c_int
    lib.pinmpc_landmark_push.argtypes = [c_void_p, c_int, c_int, POINTER(LandmarkCfg), c_void_p, c_void_p, c_void_p]
    lib.pinmpc_landmark_push_solver.restype = c_int
    lib.pinmpc_landmark_push_solver.argtypes = [c_void_p, c_void_p, POINTER(LandmarkCfg), c_void_p, c_void_p]
    lib.pinmpc_landmark_reward.restype = c_int
    lib.pinmpc_landmark_reward.argtypes = [c_void_p, c_int, c_int, POINTER(LandmarkCfg)] + [c_void_p] * 5
    lib.pinmpc_split_workspace_bytes.restype = c_size_t
    lib.pinmpc_split_workspace_bytes.argtypes = [c_int, c_int, c_int]
    lib.pinmpc_split_solve.restype = c_int
    lib.pinmpc_split_solve.argtypes = [c_int, c_int, c_int, POINTER(Layout), POINTER(c_float), POINTER(c_float), c_float, c_int,
                                       POINTER(SplitProblem), c_void_p, c_size_t, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pinmpc_split_workspace_bytes_ex.restype = c_size_t
    lib.pinmpc_split_workspace_bytes_ex.argtypes = [c_int, c_int, c_int, POINTER(SplitOptions)]
    lib.pinmpc_split_solve_ex.restype = c_int
    lib.pinmpc_split_solve_ex.argtypes = [c_int, c_int, c_int, POINTER(Layout), POINTER(c_float), POINTER(c_float), c_float, c_int,
                                          POINTER(SplitProblem), POINTER(SplitOptions), c_void_p, c_size_t, c_void_p, c_void_p, c_void_p,
                                          c_void_p]
    lib.pinmpc_split_static_bytes.restype = c_size_t
    lib.pinmpc_split_static_bytes.argtypes = []
    lib.pinmpc_split_solve_static.restype = c_int
    lib.pinmpc_split_solve_static.argtypes = [c_int, c_int, c_int, POINTER(Layout), POINTER(c_float), POINTER(c_float), c_float, c_int,
                                              POINTER(SplitProblem), POINTER(SplitOptions), c_void_p, c_void_p, c_void_p, c_void_p]
    lib.pinmpc_assemble_centroidal.restype = c_int
    lib.pinmpc_assemble_centroidal.argtypes = [c_int, c_int, c_int, c_int, c_float] + [c_void_p] * 6
    lib.pinmpc_destroy.restype = None
    lib.pinmpc_destroy.argtypes = [c_void_p]
    _lib = lib
    return lib


def _check(status, h=None):
    if status != OK:
        raise PinmpcError(status, load().pinmpc_last_error(h).decode())


def _ptr(t):
    return None if t is None else c_void_p(t.data_ptr())


def make_layout(n_wrench=2, n_force=0, mu=0.5, fz_max=600.0, mx_coef=0.02, my_coef=0.02, mz_coef=0.01,
                hand_fmax=150.0) -> Layout:
    return Layout(n_wrench, n_force, mu, fz_max, mx_coef, my_coef, mz_coef, hand_fmax)


# ---- one-to-one wrappers -------------------------------------------------------------------------
def pinmpc_workspace_bytes(nx, nu, N, B, layout, method=None) -> int:
    lib = load()
    if method is None:
        return int(lib.pinmpc_workspace_bytes(nx, nu, N, B, ctypes.byref(layout)))
    return int(lib.pinmpc_workspace_bytes_method(nx, nu, N, B, ctypes.byref(layout), method))


def pinmpc_create(nx, nu, N, B, layout, rho, iters, workspace_ptr, workspace_bytes):
    h = c_void_p()
    st = load().pinmpc_create(ctypes.byref(h), nx, nu, N, B, ctypes.byref(layout), rho, iters,
                              c_void_p(workspace_ptr), workspace_bytes)
    _check(st, None)
    return h


def pinmpc_set_weights(h, Qdiag, Rdiag, dt):
    q = (c_float * len(Qdiag))(*[float(v) for v in Qdiag])
    r = (c_float * len(Rdiag))(*[float(v) for v in Rdiag])
    _check(load().pinmpc_set_weights(h, q, r, float(dt)), h)


def pinmpc_set_tolerance(h, eps_abs, eps_rel, check_every):
    _check(load().pinmpc_set_tolerance(h, float(eps_abs), float(eps_rel), int(check_every)), h)


def pinmpc_set_method(h, method):
    _check(load().pinmpc_set_method(h, int(method)), h)


def pinmpc_set_tuning(h, envs_per_cta):
    _check(load().pinmpc_set_tuning(h, int(envs_per_cta)), h)


def pinmpc_set_horizon_chunks(h, chunks):
    _check(load().pinmpc_set_horizon_chunks(h, int(chunks)), h)


def pinmpc_get_launch_shape(h):
    g, c = c_int(0), c_int(0)
    _check(load().pinmpc_get_launch_shape(h, ctypes.byref(g), ctypes.byref(c)), h)
    return int(g.value), int(c.value)


def pinmpc_set_problem(h, x0, x_ref, u_ref, contact, foot_r, yaw, mass, inertia, ext_wrench=None):
    p = Problem(*[(None if t is None else t.data_ptr()) for t in
                  (x0, x_ref, u_ref, contact, foot_r, yaw, mass, inertia, ext_wrench)])
    _check(load().pinmpc_set_problem(h, ctypes.byref(p)), h)


def pinmpc_set_dynamics(h, A, Bm, c=None):
    _check(load().pinmpc_set_dynamics(h, _ptr(A), _ptr(Bm), _ptr(c)), h)


def pinmpc_solve(h, stream=0):
    _check(load().pinmpc_solve(h, c_void_p(stream)), h)


def pinmpc_get(h, x=None, u=None, r_prim=None, r_dual=None, iters_done=None, stream=0):
    _check(load().pinmpc_get(h, _ptr(x), _ptr(u), _ptr(r_prim), _ptr(r_dual), _ptr(iters_done), c_void_p(stream)), h)


def pinmpc_get_aux(h, z=None, y=None, stream=0):
    _check(load().pinmpc_get_aux(h, _ptr(z), _ptr(y), c_void_p(stream)), h)


def pinmpc_get_dynamics(h, A=None, Bm=None, c=None, stream=0):
    _check(load().pinmpc_get_dynamics(h, _ptr(A), _ptr(Bm), _ptr(c), c_void_p(stream)), h)


def pinmpc_last_launch_count(h) -> int:
    return int(load().pinmpc_last_launch_count(h))


def pinmpc_set_warm_start(h, z0=None, y0=None):
    _check(load().pinmpc_set_warm_start(h, _ptr(z0), _ptr(y0)), h)


def pinmpc_shift_aux(h, shift, z0, y0, stream=None):
    _check(load().pinmpc_shift_aux(h, int(shift), _ptr(z0), _ptr(y0), stream), h)


def pinmpc_set_profiling(h, on):
    _check(load().pinmpc_set_profiling(h, int(bool(on))), h)


def pinmpc_get_kernel_ms(h):
    ms = (c_float * 3)()
    _check(load().pinmpc_get_kernel_ms(h, ms), h)
    return [float(v) for v in ms]


def pinmpc_get_srb_assembly(h, A, Bm, c, S, Tinv, stream=0):
    _check(load().pinmpc_get_srb_assembly(h, _ptr(A), _ptr(Bm), _ptr(c), _ptr(S), _ptr(Tinv), c_void_p(stream)), h)


def pinmpc_destroy(h):
    load().pinmpc_destroy(h)


# ---- convenience holder ---------------------------------------------------------------------------
class Solver:
    """Owns the workspace (a torch uint8 tensor) and keeps borrowed problem tensors alive."""

    def __init__(self, nu, N, B, layout=None, rho=1.0, iters=100, Qdiag=None, Rdiag=None, dt=0.03,
                 method=METHOD_AUTO, device="cuda:0", dense_workspace=None):
        import torch
        load()
        self.torch = torch
        self.device = torch.device(device)
        self.nu, self.N, self.B = int(nu), int(N), int(B)
        self.layout = layout or make_layout(2, 2 if nu == 18 else 0)
        if dense_workspace is None:
            dense_workspace = method == METHOD_DENSE
        wm = METHOD_DENSE if dense_workspace else METHOD_SRB
        self.workspace_bytes = pinmpc_workspace_bytes(NX, nu, N, B, self.layout, wm)
        if self.workspace_bytes == 0:
            raise PinmpcError(EUNSUPPORTED, "unsupported sizes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=self.device)
            self.h = pinmpc_create(NX, nu, N, B, self.layout, float(rho), int(iters), self.workspace.data_ptr(),
                                   self.workspace_bytes)
        if Qdiag is not None or Rdiag is not None or dt is not None:
            Qd = [500, 500, 100, 50, 50, 200, 1, 1, 1, 20, 20, 10, 0] if Qdiag is None else list(Qdiag)
            Rd = [1e-5] * nu if Rdiag is None else list(Rdiag)
            pinmpc_set_weights(self.h, Qd, Rd, dt)
        if method != METHOD_AUTO:
            pinmpc_set_method(self.h, method)
        self._keep = {}

    def _dev(self, a, dtype):
        torch = self.torch
        if a is None:
            return None
        if not isinstance(a, torch.Tensor):
            a = torch.from_numpy(a)
        return a.to(device=self.device, dtype=dtype).contiguous()

    def set_problem(self, x0, x_ref, u_ref, contact, foot_r, yaw, mass, inertia, ext_wrench=None):
        t = self.torch
        f = t.float32
        k = dict(x0=self._dev(x0, f), x_ref=self._dev(x_ref, f), u_ref=self._dev(u_ref, f),
                 contact=self._dev(contact, t.uint8), foot_r=self._dev(foot_r, f), yaw=self._dev(yaw, f),
                 mass=self._dev(mass, f), inertia=self._dev(inertia, f), ext_wrench=self._dev(ext_wrench, f))
        B, N, nu = self.B, self.N, self.nu
        nc = self.layout.n_wrench + self.layout.n_force
        shapes = dict(x0=(B, NX), x_ref=(B, N, NX), u_ref=(B, N, nu), contact=(B, N, nc), foot_r=(B, N, nc, 3),
                      yaw=(B, N), mass=(B,), inertia=(B, 3, 3), ext_wrench=(B, N, 6))
        for name, v in k.items():
            if v is not None and tuple(v.shape) != shapes[name]:
                raise ValueError(f"{name}: shape {tuple(v.shape)} != {shapes[name]}")
        self._keep.update(k)
        pinmpc_set_problem(self.h, **k)

    def set_workload(self, w):
        self.set_problem(w.x0, w.x_ref, w.u_ref, w.contact, w.foot_r, w.yaw, w.mass, w.inertia, w.ext_wrench)

    def set_dynamics(self, A, Bm, c=None):
        f = self.torch.float32
        k = dict(A=self._dev(A, f), Bm=self._dev(Bm, f), c=self._dev(c, f))
        self._keep.update(k)
        pinmpc_set_dynamics(self.h, k["A"], k["Bm"], k["c"])

    def set_tolerance(self, eps_abs, eps_rel, check_every=1):
        pinmpc_set_tolerance(self.h, eps_abs, eps_rel, check_every)

    def set_method(self, method):
        pinmpc_set_method(self.h, method)

    def set_tuning(self, envs_per_cta):
        pinmpc_set_tuning(self.h, envs_per_cta)

    def set_horizon_chunks(self, chunks):
        pinmpc_set_horizon_chunks(self.h, chunks)

    def launch_shape(self):
        return pinmpc_get_launch_shape(self.h)

    def set_warm_start(self, z0=None, y0=None):
        """Start the next solves from z0, y0 [B,N,nu] (None, None: cold start)."""
        f = self.torch.float32
        z0, y0 = self._dev(z0, f), self._dev(y0, f)
        for v in (z0, y0):
            if v is not None and tuple(v.shape) != (self.B, self.N, self.nu):
                raise ValueError(f"warm start: shape {tuple(v.shape)} != {(self.B, self.N, self.nu)}")
        self._keep.update(warm_z=z0, warm_y=y0)
        pinmpc_set_warm_start(self.h, z0, y0)

    def shift_warm_start(self, shift=1, stream=None):
        """Receding-horizon update: shift z, y of the last solve by `shift` stages on the device and use them as
        the start of the next solves.  Call it before handing over the next problem (set_problem forgets the solve)."""
        t = self.torch
        z0 = t.empty((self.B, self.N, self.nu), dtype=t.float32, device=self.device)
        y0 = t.empty_like(z0)
        pinmpc_shift_aux(self.h, shift, z0, y0, self._stream(stream))
        self._keep.update(warm_z=z0, warm_y=y0)
        pinmpc_set_warm_start(self.h, z0, y0)
        return z0, y0

    def set_profiling(self, on=True):
        pinmpc_set_profiling(self.h, on)

    def kernel_ms(self):
        """[assembly, factorisation, iteration] milliseconds of the last profiled solve (synchronises)."""
        return pinmpc_get_kernel_ms(self.h)

    def _stream(self, stream):
        if stream is None:
            stream = self.torch.cuda.current_stream(self.device)
        return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)

    def solve(self, stream=None):
        pinmpc_solve(self.h, self._stream(stream))

    def launch_count(self):
        return pinmpc_last_launch_count(self.h)

    def get(self, stream=None, aux=False):
        t = self.torch
        B, N, nu = self.B, self.N, self.nu
        o = dict(x=t.empty((B, N, NX), dtype=t.float32, device=self.device),
                 u=t.empty((B, N, nu), dtype=t.float32, device=self.device),
                 r_prim=t.empty(B, dtype=t.float32, device=self.device),
                 r_dual=t.empty(B, dtype=t.float32, device=self.device),
                 iters_done=t.empty(B, dtype=t.int32, device=self.device))
        s = self._stream(stream)
        pinmpc_get(self.h, o["x"], o["u"], o["r_prim"], o["r_dual"], o["iters_done"], s)
        if aux:
            o["z"] = t.empty((B, N, nu), dtype=t.float32, device=self.device)
            o["y"] = t.empty((B, N, nu), dtype=t.float32, device=self.device)
            pinmpc_get_aux(self.h, o["z"], o["y"], s)
        return o

    def get_dynamics(self, stream=None):
        t = self.torch
        B, N, nu = self.B, self.N, self.nu
        A = t.empty((B, N, NX, NX), dtype=t.float32, device=self.device)
        Bm = t.empty((B, N, NX, nu), dtype=t.float32, device=self.device)
        c = t.empty((B, N, NX), dtype=t.float32, device=self.device)
        pinmpc_get_dynamics(self.h, A, Bm, c, self._stream(stream))
        return A, Bm, c

    def get_srb_assembly(self, stream=None):
        """A, Bm, c expanded from the structured solver's own assembly records, plus its S [B,N,21] and Tinv [B,N,6]."""
        t = self.torch
        B, N, nu = self.B, self.N, self.nu
        mk = lambda *shape: t.empty(shape, dtype=t.float32, device=self.device)
        A, Bm, c, S, Ti = mk(B, N, NX, NX), mk(B, N, NX, nu), mk(B, N, NX), mk(B, N, 21), mk(B, N, 6)
        pinmpc_get_srb_assembly(self.h, A, Bm, c, S, Ti, self._stream(stream))
        return A, Bm, c, S, Ti

    def close(self):
        if getattr(self, "h", None) is not None:
            pinmpc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- predictive landmarks + prediction-confidence reward (include/pinmpc.h, eq. (10)-(14)) ----------
def make_landmark_cfg(s, alpha, Qc=(1.0, 1.0, 1.0), sigma_c=0.05) -> LandmarkCfg:
    if len(s) != len(alpha) or not 1 <= len(s) <= MAX_LANDMARKS:
        raise PinmpcError(EINVAL, "1..8 landmarks, len(s) == len(alpha)")
    c = LandmarkCfg()
    c.n_landmarks = len(s)
    for i, (a, b) in enumerate(zip(s, alpha)):
        c.s[i], c.alpha[i] = float(a), float(b)
    for j in range(3):
        c.Qc[j] = float(Qc[j])
    c.sigma_c = float(sigma_c)
    return c


class Landmarks:
    """Owns the device ring buffer; every method is one C-ABI call (argument marshalling only)."""

    def __init__(self, B, N, cfg: LandmarkCfg, device="cuda:0"):
        import torch
        self.torch, self.device = torch, torch.device(device)
        self.B, self.N, self.cfg = int(B), int(N), cfg
        nbytes = load().pinmpc_landmark_ring_bytes(self.B, self.N, ctypes.byref(cfg))
        if nbytes == 0 and self.B > 0:
            raise PinmpcError(EINVAL, "invalid landmark configuration")
        self.ring = torch.empty(max(nbytes, 16), dtype=torch.uint8, device=self.device)
        self.reset()

    def _s(self, stream):
        return c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream.cuda_stream)

    def reset(self, mask=None, stream=None):
        _check(load().pinmpc_landmark_reset(_ptr(self.ring), self.B, self.N, ctypes.byref(self.cfg), _ptr(mask), self._s(stream)))

    def push(self, x, t, stream=None):
        _check(load().pinmpc_landmark_push(_ptr(self.ring), self.B, self.N, ctypes.byref(self.cfg), _ptr(x), _ptr(t), self._s(stream)))

    def push_solver(self, solver, t, stream=None):
        _check(load().pinmpc_landmark_push_solver(solver.h, _ptr(self.ring), ctypes.byref(self.cfg), _ptr(t), self._s(stream)), solver.h)

    def reward(self, c_real, t, stream=None):
        tt = self.torch
        r = tt.empty(self.B, dtype=tt.float32, device=self.device)
        used = tt.empty(self.B, dtype=tt.int32, device=self.device)
        _check(load().pinmpc_landmark_reward(_ptr(self.ring), self.B, self.N, ctypes.byref(self.cfg), _ptr(c_real), _ptr(t),
                                             _ptr(r), _ptr(used), self._s(stream)))
        return r, used


# ---- the paper's own stage-local ADMM (include/pinmpc.h, eq. (18)-(22)) ---------------------------------
class SplitSolver:
    """Owns the workspace and the output tensors of pinmpc_split_solve_ex; solve() is one asynchronous C-ABI call.
    scale_x (13 positive numbers) / scale_u: variable scaling; accel: Nesterov acceleration with restart (include/pinmpc.h)."""

    def __init__(self, nu, N, B, layout, Qdiag, Rdiag, rho, iters, device="cuda:0", scale_x=None, scale_u=1.0, accel=False, eta=0.999,
                 nx=NX, x_lo=None, x_hi=None):
        import torch
        self.torch, self.device = torch, torch.device(device)
        self.nu, self.N, self.B, self.layout, self.rho, self.iters = int(nu), int(N), int(B), layout, float(rho), int(iters)
        self.nx = int(nx)
        self.restarts = torch.zeros(self.B, dtype=torch.int32, device=self.device) if accel else None
        arr = lambda a: None if a is None else (c_float * self.nx)(*[float(v) for v in a])
        null = ctypes.cast(None, POINTER(c_float))
        self._sx, self._lo, self._hi = arr(scale_x), arr(x_lo), arr(x_hi)
        self.opts = SplitOptions(self._sx if self._sx is not None else null, float(scale_u), int(bool(accel)),
                                 float(eta), None if self.restarts is None else self.restarts.data_ptr(), self.nx,
                                 self._lo if self._lo is not None else null, self._hi if self._hi is not None else null)
        self.workspace_bytes = load().pinmpc_split_workspace_bytes_ex(self.nu, self.N, self.B, ctypes.byref(self.opts))
        if self.workspace_bytes == 0:
            raise PinmpcError(EUNSUPPORTED, "unsupported sizes")
        self.ws = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=self.device)
        self.xi = torch.empty((self.B, self.N, self.nx + self.nu), dtype=torch.float32, device=self.device)
        self.z = torch.empty_like(self.xi)
        self.r_prim = torch.empty(self.B, dtype=torch.float32, device=self.device)
        self.Qd = (c_float * NX)(*([float(v) for v in Qdiag] + [0.0] * (NX - len(Qdiag)))); self.Rd = (c_float * self.nu)(*[float(v) for v in Rdiag])

    def launch_count(self):
        """Kernel launches of one solve (factorisation + iterations + outputs)."""
        scaled = self._sx is not None or self.opts.scale_u not in (0.0, 1.0)
        per_it = 4 if self.opts.accel else 2
        return 1 + per_it * self.iters - (2 if self.opts.accel else 0) + 1 + (3 if scaled else 0) + (1 if self.opts.accel else 0)

    def solve(self, A, Bm, c, x0, u_prev, x_ref, u_ref, contact, stream=None):
        prob = SplitProblem(*[None if t is None else t.data_ptr() for t in (A, Bm, c, x0, u_prev, x_ref, u_ref, contact)])
        st = c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream.cuda_stream)
        _check(load().pinmpc_split_solve_ex(self.nu, self.N, self.B, ctypes.byref(self.layout), self.Qd, self.Rd, self.rho, self.iters,
                                            ctypes.byref(prob), ctypes.byref(self.opts), _ptr(self.ws), self.workspace_bytes, _ptr(self.xi),
                                            _ptr(self.z), _ptr(self.r_prim), st))
        return self.xi, self.z, self.r_prim


def split_solve_static(A, Bm, c, x0, u_prev, x_ref, u_ref, contact, layout, Qdiag, Rdiag, rho, iters, xi, z, r_prim, stream=None):
    """pinmpc_split_solve_static on torch CUDA tensors: no workspace, nothing allocated by the call (the scratch is a static
    device array of the library, pinmpc_split_static_bytes() bytes).  xi, z [B,N,nx+nu] and r_prim [B] are caller-owned
    outputs.  Raises PinmpcError (EALLOC with the sizes in the message) when the problem does not fit.  Asynchronous."""
    import torch
    B, N, nx, nu = Bm.shape
    Qd = (c_float * NX)(*([float(v) for v in Qdiag] + [0.0] * (NX - len(Qdiag)))); Rd = (c_float * nu)(*[float(v) for v in Rdiag])
    prob = SplitProblem(*[None if t is None else t.data_ptr() for t in (A, Bm, c, x0, u_prev, x_ref, u_ref, contact)])
    null = ctypes.cast(None, POINTER(c_float))
    opts = SplitOptions(null, 1.0, 0, 0.0, None, int(nx), null, null)
    st = c_void_p(torch.cuda.current_stream(Bm.device).cuda_stream if stream is None else stream.cuda_stream)
    rc = load().pinmpc_split_solve_static(nu, N, B, ctypes.byref(layout), Qd, Rd, float(rho), int(iters), ctypes.byref(prob), ctypes.byref(opts),
                                          _ptr(xi), _ptr(z), _ptr(r_prim), st)
    if rc != OK:
        raise PinmpcError(rc, load().pinmpc_last_error(None).decode())


def assemble_centroidal(n_wrench, n_force, dt, mass, foot_r, stream=None):
    """pinmpc_assemble_centroidal on torch CUDA tensors: mass [B], foot_r [B,N,nc,3] -> A [B,N,9,9], Bm [B,N,9,nu], e [B,N,9]."""
    import torch
    B, N = foot_r.shape[:2]
    nu = 6 * n_wrench + 3 * n_force
    A = torch.empty((B, N, 9, 9), dtype=torch.float32, device=foot_r.device)
    Bm = torch.empty((B, N, 9, nu), dtype=torch.float32, device=foot_r.device)
    e = torch.empty((B, N, 9), dtype=torch.float32, device=foot_r.device)
    st = c_void_p(torch.cuda.current_stream(foot_r.device).cuda_stream if stream is None else stream.cuda_stream)
    rc = load().pinmpc_assemble_centroidal(B, N, n_wrench, n_force, float(dt), _ptr(mass), _ptr(foot_r), _ptr(A), _ptr(Bm), _ptr(e), st)
    if rc != OK:
        raise PinmpcError(rc, "pinmpc_assemble_centroidal")
    return A, Bm, e


def split_solve(A, Bm, c, x0, u_prev, x_ref, u_ref, contact, layout, Qdiag, Rdiag, rho, iters, stream=None, scale_x=None, scale_u=1.0,
                accel=False, eta=0.999, return_restarts=False, x_lo=None, x_hi=None):
    """One pinmpc_split_solve_ex call on torch CUDA tensors (float32, contiguous; c, u_prev, u_ref may be None).
    Returns (xi [B,N,13+nu], z [B,N,13+nu], r_prim [B]) (+ restarts [B] int32 when asked for); synchronises the stream."""
    import torch
    B, N, nx, nu = Bm.shape
    s = SplitSolver(nu, N, B, layout, Qdiag, Rdiag, rho, iters, device=Bm.device, scale_x=scale_x, scale_u=scale_u, accel=accel, eta=eta,
                    nx=nx, x_lo=x_lo, x_hi=x_hi)
    out = s.solve(A, Bm, c, x0, u_prev, x_ref, u_ref, contact, stream)
    torch.cuda.current_stream(Bm.device).synchronize()
    return out + (s.restarts,) if return_restarts else out
