"""float64 oracle of the paper's own 9-state centroidal model — TEST INFRASTRUCTURE ONLY.

PAPER.md:L41-57, eq. (1)-(4): xi = [c ; l_G ; k_G] in R^9 (CoM position, centroidal linear momentum, centroidal angular
momentum about the CoM), forward Euler with timestep dt:

    c_{k+1}   = c_k   + dt / m * l_{G,k}                                                        (2)
    l_{G,k+1} = l_{G,k} + dt (m g + sum_i f_{i,k})                                              (3)
    k_{G,k+1} = k_{G,k} + dt sum_i ((p_{i,k} - c_k) x f_{i,k} + tau_{i,k})                      (4)

Reading: the bilinear term (p_i - c_k) x f_i is resolved as in the 13-state model — the lever
r_{i,k} = p_{i,k} - c_k is DATA along the linearisation trajectory — so that (2)-(4) is the LTV system
xi_{k+1} = A xi_k + B_k u_k + e with

    A = [[I, dt/m I, 0], [0, I, 0], [0, 0, I]],   e = [0 ; dt m g ; 0],   g = (0, 0, -9.81)
    B_k: rows of l_G: dt I for every force;  rows of k_G: dt [r_{i,k}]x for the force, dt I for the moment of a wrench contact

and the input layout of the 13-state model (include/pinmpc.h): u = [f_1..f_nw | tau_1..tau_nw | f_{nw+1}..f_{nw+nf}].
The sum over the active set C_k is the sum over all contacts: an inactive contact has U_k = {0}.
Only tests/ may import this; it shares no code with paper_2606_05687_b200 and never imports it.
"""
from __future__ import annotations

import numpy as np

G = 9.81
NX = 9


def skew(r):
    return np.array([[0.0, -r[2], r[1]], [r[2], 0.0, -r[0]], [-r[1], r[0], 0.0]])


def assemble(n_wrench, n_force, dt, mass, foot_r):
    """mass [B], foot_r [B,N,nc,3] -> A [B,N,9,9], Bm [B,N,9,nu], e [B,N,9]."""
    mass = np.asarray(mass, dtype=np.float64); foot_r = np.asarray(foot_r, dtype=np.float64)
    B, N, nc, _ = foot_r.shape
    assert nc == n_wrench + n_force
    nu = 6 * n_wrench + 3 * n_force
    A = np.zeros((B, N, NX, NX)); Bm = np.zeros((B, N, NX, nu)); e = np.zeros((B, N, NX))
    for b in range(B):
        for k in range(N):
            A[b, k] = np.eye(NX)
            A[b, k, 0:3, 3:6] = dt / mass[b] * np.eye(3)
            e[b, k, 5] = -dt * mass[b] * G
            for i in range(nc):
                fc = 3 * i if i < n_wrench else 6 * n_wrench + 3 * (i - n_wrench)
                Bm[b, k, 3:6, fc:fc + 3] = dt * np.eye(3)
                Bm[b, k, 6:9, fc:fc + 3] = dt * skew(foot_r[b, k, i])
                if i < n_wrench:
                    mc = 3 * n_wrench + 3 * i
                    Bm[b, k, 6:9, mc:mc + 3] = dt * np.eye(3)
    return A, Bm, e


def pad13(A, Bm, e):
    """The same system embedded in 13 states (identity on the four padding states, no input, no offset)."""
    sh = A.shape[:-2]
    A13 = np.zeros(sh + (13, 13)); A13[..., :, :] = np.eye(13); A13[..., :9, :9] = A
    B13 = np.zeros(sh + (13, Bm.shape[-1])); B13[..., :9, :] = Bm
    e13 = np.zeros(sh + (13,)); e13[..., :9] = e
    return A13, B13, e13
