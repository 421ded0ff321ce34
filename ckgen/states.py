"""Seeded synthetic thermochemical states (inputs only, no kinetics).

Stand-ins for the cell states of the paper's 0-D ignition and 1-D detonation runs
(PAPER.md:185, 205-227), with the distributions BASELINE.json's `configs` state.
Layout is the library's SoA layout (batch dimension N_C leading every
column): T[N], P[N], Y[S][N], float64, C-contiguous.
"""
from __future__ import annotations

import numpy as np

from .mechanism import P_ATM

Y_FLOOR = 1.0e-20


def generate_states(S, N, seed, T_range, P_range_atm, dirichlet_alpha):
    """T ~ U[T_range] K, P ~ U[P_range_atm] atm (returned in Pa), Y ~ Dirichlet(alpha)
    floored at 1e-20 and renormalised. Returns (T[N], P[N], Y[S, N])."""
    rng = np.random.default_rng(seed)
    T = rng.uniform(T_range[0], T_range[1], size=N)
    P = rng.uniform(P_range_atm[0], P_range_atm[1], size=N) * P_ATM
    Y = np.empty((S, N))
    # Dirichlet(alpha) = normalised iid Gamma(alpha); drawn row by row to bound memory
    for k in range(S):
        Y[k] = rng.standard_gamma(dirichlet_alpha, size=N)
    Y /= Y.sum(axis=0, keepdims=True)
    np.maximum(Y, Y_FLOOR, out=Y)
    Y /= Y.sum(axis=0, keepdims=True)
    return T, P, Y
