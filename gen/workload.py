"""Seeded synthetic MPC batches shaped like the paper's RL workload.

The paper's inputs (simulator states, Raibert footholds, gait clock)
are not available, so every input is synthetic.  The recipe is BASELINE.json `configs` with the
gaps filled as listed in DESIGN.md ("Input recipe").  This module only *makes inputs*: rotations
here place feet and references in the world; nothing of the solver (assembly, Riccati, ADMM,
projection) lives here.

All random draws are float64 arrays of leading dimension B from numpy `Generator(PCG64(seed))`,
in a fixed order; results are cast to float32 once.  Both the oracle and the CUDA path consume
those float32 values (the oracle up-casts them to float64).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

SEED_BASE = 26060568700
NX = 13
GRAVITY = 9.81

# cost weights and constraint constants of BASELINE.json config 0
Q_DIAG = np.array([500, 500, 100, 50, 50, 200, 1, 1, 1, 20, 20, 10, 0], dtype=np.float64)
R_SCALE = 1e-5

# BASELINE.json configs 0..3 (+ the sweep generator = config 1's recipe with seed index 4)
CONFIGS = {
    0: dict(name="c0_tiny_walk", B=64, N=10, dt=0.04, iters=50, nu=12, fixed_period=0.4),
    1: dict(name="c1_rl_scale", B=4096, N=20, dt=0.03, iters=100, nu=12, fixed_period=None),
    2: dict(name="c2_long_horizon", B=4096, N=50, dt=0.03, iters=100, nu=12, fixed_period=None),
    3: dict(name="c3_loco_manip", B=16384, N=30, dt=0.03, iters=100, nu=18, fixed_period=None),
    4: dict(name="c4_sweep", B=4096, N=50, dt=0.03, iters=100, nu=12, fixed_period=None),
}
SWEEP_B = (1024, 4096, 16384, 65536)
SWEEP_N = (10, 25, 50, 100)


@dataclass
class Workload:
    name: str
    B: int
    N: int
    nu: int
    n_wrench: int
    n_force: int
    dt: float
    rho: float
    iters: int
    seed: int
    # constraint layout (BASELINE.json config 0 / config 3)
    mu: float = 0.5
    fz_max: float = 600.0
    mx_coef: float = 0.02
    my_coef: float = 0.02
    mz_coef: float = 0.01
    hand_fmax: float = 150.0
    # weights
    Qdiag: np.ndarray = field(default=None, repr=False)   # [13] f32
    Rdiag: np.ndarray = field(default=None, repr=False)   # [nu] f32
    # per-env problem data, float32 unless noted
    x0: np.ndarray = field(default=None, repr=False)          # [B,13]
    x_ref: np.ndarray = field(default=None, repr=False)       # [B,N,13]   reference for x_1..x_N
    u_ref: np.ndarray = field(default=None, repr=False)       # [B,N,nu]
    contact: np.ndarray = field(default=None, repr=False)     # [B,N,nc] uint8
    foot_r: np.ndarray = field(default=None, repr=False)      # [B,N,nc,3]
    yaw: np.ndarray = field(default=None, repr=False)         # [B,N]
    mass: np.ndarray = field(default=None, repr=False)        # [B]
    inertia: np.ndarray = field(default=None, repr=False)     # [B,3,3]
    ext_wrench: Optional[np.ndarray] = field(default=None, repr=False)  # [B,N,6] or None

    @property
    def nc(self) -> int:
        return self.n_wrench + self.n_force

    ARRAYS = ("x0", "x_ref", "u_ref", "contact", "foot_r", "yaw", "mass", "inertia", "ext_wrench")


def _rotz_apply(psi: np.ndarray, v: np.ndarray) -> np.ndarray:
    """R_z(psi) v for psi[...], v[...,3]."""
    c, s = np.cos(psi), np.sin(psi)
    out = np.empty(np.broadcast_shapes(psi.shape + (3,), v.shape), dtype=np.float64)
    out[..., 0] = c * v[..., 0] - s * v[..., 1]
    out[..., 1] = s * v[..., 0] + c * v[..., 1]
    out[..., 2] = v[..., 2]
    return out


def make_workload(name: str, B: int, N: int, dt: float, iters: int, nu: int = 12,
                  fixed_period: Optional[float] = None, seed: int = SEED_BASE,
                  rho: float = 1.0) -> Workload:
    if nu not in (12, 18):
        raise ValueError("nu must be 12 (feet) or 18 (feet + two hands)")
    hands = nu == 18
    nw, nf = 2, (2 if hands else 0)
    nc = nw + nf
    rng = np.random.Generator(np.random.PCG64(seed))

    # ---- draws, fixed order --------------------------------------
    mass = rng.uniform(35.0, 60.0, B)                         # 1
    Ib_diag = rng.uniform(0.5, 3.0, (B, 3))                   # 2
    yaw0 = rng.uniform(-np.pi, np.pi, B)                      # 3
    yaw_rate = rng.uniform(-0.5, 0.5, B)                      # 4
    v_cmd = rng.uniform(-1.0, 1.0, (B, 2))                    # 5
    if fixed_period is None:
        period = rng.uniform(0.3, 0.5, B)                     # 6
    else:
        period = np.full(B, float(fixed_period))
    phase0 = rng.uniform(0.0, 1.0, B)                         # 7
    foot_off = np.empty((B, 2, 3))                            # 8  body-frame offsets, i = L, R
    foot_off[..., 0] = rng.uniform(-0.10, 0.10, (B, 2))       #    fore-aft
    foot_off[..., 1] = rng.uniform(-0.15, 0.15, (B, 2))       #    lateral
    foot_off[..., 2] = rng.uniform(-0.95, -0.85, (B, 2))      #    vertical
    x0_noise = rng.normal(0.0, 0.02, (B, 12))                 # 9
    if hands:
        payload = rng.uniform(0.0, 10.0, B)                   # 10
        cart_force = rng.uniform(0.0, 200.0, B)               # 11
        reach = rng.uniform(0.3, 0.5, (B, 2))                 # 12
        mass = mass + payload

    # ---- derived references ------------------------------------------------------------------
    k = np.arange(N + 1, dtype=np.float64)
    psi = yaw0[:, None] + yaw_rate[:, None] * k[None, :] * dt            # [B,N+1]
    vb = np.zeros((B, 1, 3)); vb[:, 0, :2] = v_cmd
    v_ref = _rotz_apply(psi, vb)                                         # [B,N+1,3]
    p_ref = np.empty((B, N + 1, 3))
    p_ref[:, 0] = (0.0, 0.0, 0.9)
    for j in range(N):
        p_ref[:, j + 1] = p_ref[:, j] + dt * v_ref[:, j]
    xbar = np.zeros((B, N + 1, NX))
    xbar[..., 2] = psi
    xbar[..., 3:6] = p_ref
    xbar[..., 8] = yaw_rate[:, None]
    xbar[..., 9:12] = v_ref
    xbar[..., 12] = -GRAVITY
    x0 = xbar[:, 0].copy()
    x0[:, :12] += x0_noise

    # ---- contact schedule: alternating gait, 50 % duty ----------------------------------------
    phi = np.mod(phase0[:, None] + k[None, :N] * dt / period[:, None], 1.0)   # [B,N]
    contact = np.zeros((B, N, nc), dtype=np.uint8)
    contact[..., 0] = phi < 0.5
    contact[..., 1] = phi >= 0.5
    if hands:
        contact[..., 2:] = 1

    # ---- contact positions relative to the CoM, world-aligned axes ----------------------------
    foot_r = np.empty((B, N, nc, 3))
    for i in range(2):
        world = np.zeros((B, 3))                 # stance-foot world position since touchdown
        for j in range(N):
            swing_r = _rotz_apply(psi[:, j], foot_off[:, i])             # under the hip
            st = contact[:, j, i].astype(bool)
            td = st & (~contact[:, j - 1, i].astype(bool) if j > 0 else np.ones(B, bool))
            world[td] = swing_r[td] + p_ref[td, j]
            foot_r[:, j, i] = np.where(st[:, None], world - p_ref[:, j], swing_r)
    if hands:
        for h in range(2):
            hb = np.stack([reach[:, h], np.full(B, 0.2 if h == 0 else -0.2), np.full(B, 0.1)], -1)
            foot_r[:, :, 2 + h] = _rotz_apply(psi[:, :N], hb[:, None, :])

    # ---- input reference: stance feet share the weight ----------------------------------------
    u_ref = np.zeros((B, N, nu))
    n_stance = contact[..., :2].sum(-1).astype(np.float64)
    share = mass[:, None] * GRAVITY / np.maximum(n_stance, 1.0)
    for i in range(2):
        u_ref[..., 3 * i + 2] = np.where(contact[..., i] > 0, share, 0.0)

    ext = None
    if hands:
        ex = np.zeros((B, 1, 3)); ex[..., 0] = 1.0
        F_ext = -cart_force[:, None, None] * _rotz_apply(psi[:, :N], ex)          # [B,N,3]
        rb = np.stack([reach.mean(-1), np.zeros(B), np.full(B, 0.1)], -1)
        r_app = _rotz_apply(psi[:, :N], rb[:, None, :])
        ext = np.concatenate([F_ext, np.cross(r_app, F_ext)], -1)                 # (F, tau)

    inertia = np.zeros((B, 3, 3))
    for a in range(3):
        inertia[:, a, a] = Ib_diag[:, a]

    f32 = np.float32
    return Workload(
        name=name, B=B, N=N, nu=nu, n_wrench=nw, n_force=nf, dt=float(dt), rho=float(rho),
        iters=int(iters), seed=int(seed),
        Qdiag=Q_DIAG.astype(f32), Rdiag=np.full(nu, R_SCALE, dtype=f32),
        x0=x0.astype(f32), x_ref=np.ascontiguousarray(xbar[:, 1:]).astype(f32),
        u_ref=u_ref.astype(f32), contact=contact, foot_r=foot_r.astype(f32),
        yaw=np.ascontiguousarray(psi[:, :N]).astype(f32), mass=mass.astype(f32),
        inertia=inertia.astype(f32), ext_wrench=None if ext is None else ext.astype(f32))


def make_config(idx: int, B: Optional[int] = None, N: Optional[int] = None,
                iters: Optional[int] = None) -> Workload:
    """BASELINE.json config `idx` (0..4); B/N/iters override the shape (sweep points, tests)."""
    c = dict(CONFIGS[idx])
    if B is not None:
        c["B"] = int(B)
    if N is not None:
        c["N"] = int(N)
    if iters is not None:
        c["iters"] = int(iters)
    if B is not None or N is not None:
        c["name"] = f"{c['name']}_B{c['B']}_N{c['N']}"
    return make_workload(seed=SEED_BASE + idx, **c)


def subset(w: Workload, env_idx) -> Workload:
    """The same problems restricted to the listed envs (envs are independent QPs)."""
    env_idx = np.asarray(env_idx, dtype=np.int64)
    kw = {}
    for a in Workload.ARRAYS:
        v = getattr(w, a)
        kw[a] = None if v is None else np.ascontiguousarray(v[env_idx])
    return replace(w, B=int(env_idx.size), name=f"{w.name}_sub{env_idx.size}", **kw)


def centroidal_view(w: Workload) -> dict:
    """Inputs of the paper's 9-state centroidal model (eq. (1): xi = [c ; l_G ; k_G]) for the same synthetic
    episode: CoM position from the position entries of the 13-state arrays, momenta as mass x velocity entries and
    body-inertia diagonal x angular-velocity entries (inputs only; the dynamics come from the assembly).  Adds fixed
    weights of the momenta's units and a state box X_k (eq. (17)): a CoM height ceiling and a bound on the fore-aft
    linear momentum, chosen so that both bind on part of the envs."""
    m = w.mass.astype(np.float64)
    Ib = np.diagonal(w.inertia.astype(np.float64), axis1=1, axis2=2)
    x0 = np.concatenate([w.x0[:, 3:6], m[:, None] * w.x0[:, 9:12], Ib * w.x0[:, 6:9]], axis=-1)
    x_ref = np.concatenate([w.x_ref[..., 3:6], m[:, None, None] * w.x_ref[..., 9:12], Ib[:, None, :] * w.x_ref[..., 6:9]], axis=-1)
    Qd = np.array([50.0, 50.0, 200.0, 1e-2, 1e-2, 5e-3, 0.4, 0.4, 0.4])
    x_lo = np.array([-np.inf, -np.inf, 0.80, -20.0, -np.inf, -np.inf, -np.inf, -np.inf, -np.inf])
    x_hi = np.array([np.inf, np.inf, 0.905, 20.0, np.inf, np.inf, np.inf, np.inf, np.inf])
    return dict(x0=x0.astype(np.float32), x_ref=x_ref.astype(np.float32), Qdiag=Qd.astype(np.float32),
                x_lo=x_lo.astype(np.float32), x_hi=x_hi.astype(np.float32))
