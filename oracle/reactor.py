"""CPU oracle of the 0-D constant-pressure reactor step -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It follows, step by step and with no reordering, the explicit time
stepping the paper uses its source term in (constant-pressure 0-D
auto-ignition advanced explicitly) with the scheme BASELINE.json configs[4] names (classic
RK4), on top of oracle.source_terms:

    dT/dt   = -sum_k h_k wdot_k / (rho cp)            (oracle.source_terms' second result)
    dY_k/dt = wdot_k W_k / rho,  rho = P / (Ru T sum_k Y_k / W_k),  P constant

    k1 = f(y),  k2 = f(p(y + dt/2 k1)),  k3 = f(p(y + dt/2 k2)),  k4 = f(p(y + dt k3))
    y <- p(y + dt/6 (k1 + 2 k2 + 2 k3 + k4))

p is the projection of DESIGN.md reading Q14 (the paper is silent on what an explicit
scheme should do outside its stability range, which is where BASELINE's dt = 1e-9 s is for
its synthetic rate constants): Y <- max(Y, 0); Y <- Y / sum(Y); T <- clip(T, 250, 5000).

Pins (tests/test_oracle_reactor.py): on a thermoneutral A <=> B mechanism with equal molar
masses the right-hand side is linear, so one step must multiply the distance from
equilibrium by exactly 1 + z + z^2/2 + z^3/6 + z^4/24, z = -(k_f + k_r) dt (the stability
polynomial of the scheme, computed at 50 digits); conservation of sum(Y) and of every
element by the unprojected update; fourth-order convergence against a tiny-step reference.
"""
from __future__ import annotations

import numpy as np

from . import source_terms

RU = 8314.46261815324  # J/(kmol K)
T_MIN, T_MAX = 250.0, 5000.0


def project(T, Y):
    """p: onto valid thermochemical states (reading Q14)."""
    Y = np.maximum(Y, 0.0)
    Y = Y / Y.sum(axis=0, keepdims=True)
    return np.minimum(np.maximum(T, T_MIN), T_MAX), Y


def rhs(omech, W, T, P, Y):
    """f(y) = (dT/dt [N], dY/dt [S, N]) of the constant-pressure reactor."""
    wdot, dTdt, _ = source_terms(omech, T, P, Y)
    rho = P / (RU * T * (Y / W[:, None]).sum(axis=0))
    return dTdt, wdot * W[:, None] / rho[None, :]


def rk4_step(omech, W, T, P, Y, dt, return_stages=False):
    """One step; returns (T_new, Y_new) and, if asked, the projected stage states."""
    T = np.asarray(T, dtype=np.float64)
    Y = np.asarray(Y, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64)
    k1 = rhs(omech, W, T, P, Y)
    T2, Y2 = project(T + 0.5 * dt * k1[0], Y + 0.5 * dt * k1[1])
    k2 = rhs(omech, W, T2, P, Y2)
    T3, Y3 = project(T + 0.5 * dt * k2[0], Y + 0.5 * dt * k2[1])
    k3 = rhs(omech, W, T3, P, Y3)
    T4, Y4 = project(T + dt * k3[0], Y + dt * k3[1])
    k4 = rhs(omech, W, T4, P, Y4)
    Tn = T + dt * (k1[0] / 6.0 + k2[0] / 3.0 + k3[0] / 3.0 + k4[0] / 6.0)
    Yn = Y + dt * (k1[1] / 6.0 + k2[1] / 3.0 + k3[1] / 3.0 + k4[1] / 6.0)
    out = project(Tn, Yn)
    if return_stages:
        return out, [(T2, Y2), (T3, Y3), (T4, Y4)], (Tn, Yn)
    return out


def integrate(omech, W, T, P, Y, dt, n_steps):
    for _ in range(int(n_steps)):
        T, Y = rk4_step(omech, W, T, P, Y, dt)
    return T, Y
