"""float64 oracle of the predictive landmarks and the prediction-confidence reward — TEST INFRASTRUCTURE ONLY.

PAPER.md:L98-130, eq. (10)-(14) and Remark 1.  Only tests/ may import this; it shares
no code with paper_2606_05687_b200 and never imports it.  Pinned by tests/test_oracle_landmarks.py.

The paper's definitions, restated:

  eq. (10)  n_l = 1 + floor(s_l (N - 1)),  delta_l = n_l dt,  s_0 = 0, s_{NL-1} = 1
  eq. (11)  an MPC solve at time t stores { (t + delta_l, c_hat^t(delta_l)) },  l = 0..NL-1
  eq. (12)  e_l(t) = c_t - c_hat^{t - delta_l}(delta_l); landmarks that do not exist are omitted
  eq. (13)  r_t = exp( - sum_l alpha_l |e_l(t)|^2_{Qc} / sigma_c^2 )

Readings: time is an integer count of MPC steps dt per env (it restarts with the episode);
c_hat^t(n dt) is the (p_x, p_y, p_z) part of the predicted state x_n of the solve made at time t
(x_n = row n-1 of the solver's output x_1..x_N, entries 3:6); |e|^2_{Qc} = sum_j Qc_j e_j^2 with a
diagonal Q_c; the product s_l (N - 1) is taken in float64 on the float32 value of s_l.

Storage is a plain dictionary keyed by (env, landmark, target time): nothing is ever overwritten or
evicted, so the oracle has no ring-buffer logic to get wrong.
"""
from __future__ import annotations

import math

import numpy as np


def landmark_steps(s, N: int):
    """eq. (10): n_l = 1 + floor(s_l (N - 1)) for every s_l (float32 values, float64 product)."""
    return [1 + int(math.floor(float(np.float32(sl)) * (N - 1))) for sl in s]


class LandmarkOracle:
    def __init__(self, B: int, N: int, s, alpha, Qc, sigma_c: float):
        assert len(s) == len(alpha) and len(Qc) == 3
        self.B, self.N = B, N
        self.n = landmark_steps(s, N)
        self.alpha = [float(np.float32(a)) for a in alpha]
        self.Qc = [float(np.float32(q)) for q in Qc]
        self.sigma_c = float(np.float32(sigma_c))
        self.store = {}

    def reset(self, mask=None):
        """Start of an episode: the landmarks of the masked envs (all if None) no longer exist."""
        for key in list(self.store):
            if mask is None or mask[key[0]]:
                del self.store[key]

    def push(self, x, t):
        """eq. (11).  x [B,N,13] = x_1..x_N of the solve made at time t[b] of env b."""
        x = np.asarray(x, dtype=np.float64)
        for b in range(self.B):
            for l, n in enumerate(self.n):
                self.store[(b, l, int(t[b]) + n)] = x[b, n - 1, 3:6].copy()

    def reward(self, c_real, t):
        """eq. (12)-(13).  c_real [B,3] = realised CoM at time t[b].  Returns (r [B], landmarks used [B])."""
        c_real = np.asarray(c_real, dtype=np.float64)
        r = np.zeros(self.B)
        used = np.zeros(self.B, dtype=np.int32)
        for b in range(self.B):
            acc = 0.0
            for l in range(len(self.n)):
                pred = self.store.get((b, l, int(t[b])))
                if pred is None:
                    continue
                e = c_real[b] - pred
                acc += self.alpha[l] * sum(self.Qc[j] * e[j] * e[j] for j in range(3)) / (self.sigma_c * self.sigma_c)
                used[b] += 1
            r[b] = math.exp(-acc)
        return r, used
