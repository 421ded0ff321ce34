"""Seeded weights of an approximate ANN for log Kc (inputs only, no kinetics).

The paper replaces the exact equilibrium layer by a small trained network
(Eq. 12-14, Fig. 2): N_L hidden layers of N_H neurons on standardised
functions of temperature, a linear output layer of width N_R, standardised targets.  Its
trained weights are not available and training is out of scope, so this module
draws weights of the same shapes; timing (Fig. 10) and parity need no
trained values.  tests/ and bench.py may additionally fit the output layer by least squares.

It serves both the CPU oracle and the CUDA library and holds none of the method's
arithmetic: no forward pass, no activation function.
"""
from __future__ import annotations

import dataclasses

import numpy as np

RELU, ELU = 0, 1


@dataclasses.dataclass
class KcAnn:
    n_in: int            # 1: [ln T] (Architecture 2); 6: [ln T, T, T^2, T^3, T^4, 1/T] (Architecture 1)
    n_layers: int        # N_L hidden layers
    n_hidden: int        # N_H neurons per hidden layer
    activation: int      # RELU (Eq. 13) or ELU (Eq. 14)
    in_mean: np.ndarray  # [n_in]   standardisation of the inputs
    in_std: np.ndarray   # [n_in]
    W_in: np.ndarray     # [n_in, N_H]
    B: np.ndarray        # [N_L, N_H]
    W_hid: np.ndarray    # [N_L - 1, N_H (from), N_H (to)]
    W_out: np.ndarray    # [N_H, R]
    B_out: np.ndarray    # [R]
    out_mean: np.ndarray # [R]      de-standardisation of the outputs
    out_std: np.ndarray  # [R]


def temperature_features(T):
    """The exact layer's input features [ln T, T, T^2, T^3, T^4, 1/T]."""
    T = np.asarray(T, dtype=np.float64)
    return np.stack([np.log(T), T, T ** 2, T ** 3, T ** 4, 1.0 / T], axis=-1)


def random_kc_ann(R, n_layers, n_hidden, n_in=1, activation=ELU, seed=0, T_range=(900.0, 2800.0)):
    """Weights ~ N(0, 1/fan_in), biases ~ U[-0.5, 0.5]; inputs standardised with the mean and
    standard deviation of the features over a uniform temperature grid on T_range; output
    statistics out_mean ~ U[-20, 20], out_std ~ U[1, 10] (the size of log Kc in SI-kmol units)."""
    rng = np.random.default_rng(seed)
    feats = temperature_features(np.linspace(T_range[0], T_range[1], 4097))[:, :n_in]
    NH, NL = int(n_hidden), int(n_layers)
    return KcAnn(
        n_in=int(n_in), n_layers=NL, n_hidden=NH, activation=int(activation),
        in_mean=feats.mean(0), in_std=feats.std(0),
        W_in=rng.normal(0.0, 1.0 / np.sqrt(n_in), (n_in, NH)),
        B=rng.uniform(-0.5, 0.5, (NL, NH)),
        W_hid=rng.normal(0.0, 1.0 / np.sqrt(NH), (NL - 1, NH, NH)),
        W_out=rng.normal(0.0, 1.0 / np.sqrt(NH), (NH, R)),
        B_out=rng.uniform(-0.5, 0.5, R),
        out_mean=rng.uniform(-20.0, 20.0, R), out_std=rng.uniform(1.0, 10.0, R))
