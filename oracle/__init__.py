"""float64 CPU oracle — TEST INFRASTRUCTURE ONLY (see pinmpc_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2606_05687_b200 and never imports it.

The arithmetic lives in pinmpc_oracle.c (plain C, fp64).  This file compiles it with gcc
(`build()`), loads it with ctypes and marshals numpy arrays; inputs given as float32 are
up-cast to float64, nothing else is done to them.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_int, c_ubyte, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pinmpc_oracle.c")
_LIB = os.path.join(_HERE, "libpinmpc_oracle.so")
NX = 13


class Layout(ctypes.Structure):
    _fields_ = [("n_wrench", c_int), ("n_force", c_int), ("mu", c_double), ("fz_max", c_double),
                ("mx_coef", c_double), ("my_coef", c_double), ("mz_coef", c_double), ("hand_fmax", c_double)]


def build(force: bool = False) -> str:
    """Compile the oracle (gcc -O2 -fopenmp, no BLAS, no intrinsics)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c99", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_solve.restype = c_int
        _lib.orc_factor_env.restype = c_int
        _lib.orc_max_threads.restype = c_int
    return _lib


def _d(a, shape=None):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _p(a):
    return None if a is None else a.ctypes.data_as(c_void_p)


def layout_of(w) -> Layout:
    """Layout from any object with the constraint-layout attributes (e.g. gen.Workload)."""
    return Layout(int(w.n_wrench), int(w.n_force), float(w.mu), float(w.fz_max), float(w.mx_coef),
                  float(w.my_coef), float(w.mz_coef), float(w.hand_fmax))


def max_threads() -> int:
    return int(lib().orc_max_threads())


def assemble(nu, n_wrench, n_force, dt, yaw, foot_r, mass, inertia, ext_wrench=None):
    """O1: returns A[B,N,13,13], Bm[B,N,13,nu], c[B,N,13] (float64)."""
    yaw = _d(yaw)
    B, N = yaw.shape
    nc = n_wrench + n_force
    foot_r = _d(foot_r, (B, N, nc, 3)); mass = _d(mass, (B,)); inertia = _d(inertia, (B, 3, 3))
    ext = _d(ext_wrench, (B, N, 6)) if ext_wrench is not None else None
    A = np.empty((B, N, NX, NX)); Bm = np.empty((B, N, NX, nu)); c = np.empty((B, N, NX))
    lib().orc_assemble(c_int(B), c_int(N), c_int(nu), c_int(n_wrench), c_int(n_force), c_double(dt),
                       _p(yaw), _p(foot_r), _p(mass), _p(inertia), _p(ext), _p(A), _p(Bm), _p(c))
    return A, Bm, c


def factor_env(A, Bm, c, Qd, Rd, rho):
    """O2 for one env: returns dict(K[N,nu,13], L[N,nu,nu], Phi[N,13,13], s[N,13], P0[13,13])."""
    A = _d(A); Bm = _d(Bm); c = _d(c); Qd = _d(Qd, (NX,))
    N, nu = A.shape[0], Bm.shape[2]
    Rd = _d(Rd, (nu,))
    K = np.empty((N, nu, NX)); L = np.empty((N, nu, nu)); Phi = np.empty((N, NX, NX)); s = np.empty((N, NX))
    P0 = np.empty((NX, NX))
    rc = lib().orc_factor_env(c_int(N), c_int(nu), _p(A), _p(Bm), _p(c), _p(Qd), _p(Rd), c_double(rho),
                              _p(K), _p(L), _p(Phi), _p(s), _p(P0))
    if rc:
        raise FloatingPointError("M_k not positive definite")
    return dict(K=K, L=L, Phi=Phi, s=s, P0=P0)


def eqstep_env(A, Bm, c, fac, Qd, Rd, rho, x0, x_ref, u_ref, z, y):
    """O3 steps 1-3 for one env and given z,y: returns x[N,13] (x_1..x_N), u[N,nu]."""
    A = _d(A); Bm = _d(Bm); c = _d(c)
    N, nu = A.shape[0], Bm.shape[2]
    x = np.empty((N, NX)); u = np.empty((N, nu)); kap = np.empty((N, nu))
    u_ref = _d(u_ref, (N, nu)) if u_ref is not None else None
    args = [_d(fac["K"]), _d(fac["L"]), _d(fac["Phi"]), _d(fac["s"]), _d(Qd, (NX,)), _d(Rd, (nu,))]
    x0 = _d(x0, (NX,)); x_ref = _d(x_ref, (N, NX)); z = _d(z, (N, nu)); y = _d(y, (N, nu))
    lib().orc_eqstep_env(c_int(N), c_int(nu), _p(A), _p(Bm), _p(c), _p(args[0]), _p(args[1]), _p(args[2]),
                         _p(args[3]), _p(args[4]), _p(args[5]), c_double(rho), _p(x0), _p(x_ref), _p(u_ref),
                         _p(z), _p(y), _p(x), _p(u), _p(kap))
    return x, u


def project(layout: Layout, contact, v):
    """O4: z = Proj_{U_k}(v) row by row.  contact[M,nc] uint8, v[M,nu] -> z[M,nu]."""
    v = _d(v)
    M, nu = v.shape
    contact = np.ascontiguousarray(contact, dtype=np.uint8)
    nc = layout.n_wrench + layout.n_force
    assert contact.shape == (M, nc)
    z = np.empty_like(v)
    f = lib().orc_project_stage
    for i in range(M):
        f(ctypes.byref(layout), c_int(nu), contact[i].ctypes.data_as(c_void_p), v[i].ctypes.data_as(c_void_p),
          z[i].ctypes.data_as(c_void_p))
    return z


def solve(w, A=None, Bm=None, c=None, iters=None, rho=None, eps_abs=0.0, eps_rel=0.0, check_every=1,
          z0=None, y0=None, nthreads=0):
    """Full batched solve of a gen.Workload-like object `w` (O1..O4).

    With A/Bm/c given the assembly is bypassed (generic LTV).  Returns a dict with x[B,N,13],
    u[B,N,nu], z, y, r_prim[B], r_dual[B], iters_done[B].
    """
    B, N, nu = int(w.B), int(w.N), int(w.nu)
    nc = int(w.n_wrench + w.n_force)
    lay = layout_of(w)
    iters = int(w.iters if iters is None else iters)
    rho = float(w.rho if rho is None else rho)
    Qd = _d(w.Qdiag, (NX,)); Rd = _d(w.Rdiag, (nu,))
    x0 = _d(w.x0, (B, NX)); x_ref = _d(w.x_ref, (B, N, NX))
    u_ref = _d(w.u_ref, (B, N, nu)) if w.u_ref is not None else None
    contact = np.ascontiguousarray(w.contact, dtype=np.uint8)
    assert contact.shape == (B, N, nc)
    if A is not None:
        A = _d(A, (B, N, NX, NX)); Bm = _d(Bm, (B, N, NX, nu)); c = _d(c, (B, N, NX))
        yaw = foot_r = mass = inertia = ext = None
    else:
        yaw = _d(w.yaw, (B, N)); foot_r = _d(w.foot_r, (B, N, nc, 3)); mass = _d(w.mass, (B,))
        inertia = _d(w.inertia, (B, 3, 3))
        ext = _d(w.ext_wrench, (B, N, 6)) if w.ext_wrench is not None else None
    x = np.empty((B, N, NX)); u = np.empty((B, N, nu))
    z = np.zeros((B, N, nu)) if z0 is None else np.array(z0, dtype=np.float64, order="C")
    y = np.zeros((B, N, nu)) if y0 is None else np.array(y0, dtype=np.float64, order="C")
    rp = np.empty(B); rd = np.empty(B); it = np.empty(B, dtype=np.int32)
    fails = lib().orc_solve(
        c_int(B), c_int(N), c_int(nu), ctypes.byref(lay), c_double(float(w.dt)), c_double(rho), c_int(iters),
        c_double(eps_abs), c_double(eps_rel), c_int(check_every), _p(Qd), _p(Rd), _p(x0), _p(x_ref), _p(u_ref),
        contact.ctypes.data_as(c_void_p), _p(A), _p(Bm), _p(c), _p(yaw), _p(foot_r), _p(mass), _p(inertia),
        _p(ext), _p(x), _p(u), _p(z), _p(y), _p(rp), _p(rd), it.ctypes.data_as(c_void_p), c_int(nthreads))
    if fails:
        raise FloatingPointError(f"{fails} envs: M_k not positive definite")
    return dict(x=x, u=u, z=z, y=y, r_prim=rp, r_dual=rd, iters_done=it)
