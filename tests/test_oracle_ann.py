"""Pins the oracle's approximate-ANN log Kc path (Eq. 12-14) to things
fixed outside it:

* a worked two-layer example at 50 digits, elu and relu, with pre-activations of both signs
  (tests/golden/ann_closed_form.json; its script does not call the oracle);
* a network constructed to BE the exact equilibrium layer (Architecture 1 features passed
  through, output layer = the Gibbs weights of Eq. 10-11, non-trivial standardisation and a
  permutation as second hidden layer): the oracle must then return the exact path's source
  terms -- a transposed weight matrix, a swapped feature or a missed de-standardisation fails;
* a numpy restatement of Eq. 12 in the paper's batch-leading matrix form.
"""
import dataclasses
import json
import os

import numpy as np
import pytest

import ckgen
import oracle
from helpers import RU, exact_layer_as_ann, ann_forward_matrix_form
from test_oracle_closed_forms import two_species_mech

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "ann_closed_form.json")))


@pytest.mark.parametrize("kind", ["elu", "relu"])
def test_worked_two_layer_example(kind):
    mech = two_species_mech(W=(20, 20), a1=(3.5, 3.5), a6=(0, -5000), a7=(2, 3), nu_r=(1, 0), nu_p=(0, 1))
    ann = ckgen.KcAnn(
        n_in=1, n_layers=2, n_hidden=2, activation=ckgen.ELU if kind == "elu" else ckgen.RELU,
        in_mean=np.array([7.0]), in_std=np.array([0.5]), W_in=np.array([[0.8, -1.5]]),
        B=np.array([[0.1, 0.2], [-0.3, 0.4]]), W_hid=np.array([[[0.5, -2.0], [1.5, 0.25]]]),
        W_out=np.array([[1.25], [-0.75]]), B_out=np.array([0.5]), out_mean=np.array([4.0]),
        out_std=np.array([3.0]))
    om = oracle.OracleMechanism(mech, kc_ann=ann)
    det = oracle.cell_detail(om, 1000.0, 101325.0, np.array([0.75, 0.25]))
    g = GOLD[kind]
    assert abs(np.log(det["Kc"][0]) - float(g["lnKc"])) <= 1e-14 * abs(float(g["lnKc"]))
    assert abs(det["Q"][0] - float(g["q"])) <= 1e-13 * abs(float(g["q"]))
    assert abs(det["dTdt"] - float(g["dTdt"])) <= 1e-13 * abs(float(g["dTdt"]))
    # and it is not the exact layer's value (ln Kc = 6 for this mechanism)
    assert abs(np.log(det["Kc"][0]) - 6.0) > 0.1


@pytest.mark.parametrize("n_layers,activation", [(1, ckgen.RELU), (2, ckgen.ELU)])
def test_network_built_to_be_the_exact_layer(n_layers, activation):
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    mech = dataclasses.replace(mech, nasa_lo=mech.nasa_hi.copy())      # one NASA set: one network
    T, P, Y = ckgen.states(cfg, N=64)
    ann = exact_layer_as_ann(mech, n_layers=n_layers, activation=activation, seed=3)
    w0, d0, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    w1, d1, _ = oracle.source_terms(oracle.OracleMechanism(mech, kc_ann=ann), T, P, Y)
    # ln Kc of a few hundred summed in a different order: 1e-13 relative on Kc
    assert np.abs(w1 - w0).max(0).max() <= 1e-11 * np.abs(w0).max()
    assert (np.abs(w1 - w0) <= 1e-11 * np.abs(w0).max(0, keepdims=True)).all()
    assert (np.abs(d1 - d0) <= 1e-9 * np.abs(d0)).all()


@pytest.mark.parametrize("n_in,n_layers,n_hidden,activation", [(1, 1, 8, ckgen.ELU), (1, 3, 32, ckgen.ELU),
                                                               (6, 2, 8, ckgen.RELU), (1, 2, 5, ckgen.RELU)])
def test_matrix_form_restatement(n_in, n_layers, n_hidden, activation):
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    ann = ckgen.random_kc_ann(mech.n_reactions, n_layers, n_hidden, n_in=n_in, activation=activation, seed=11)
    T, P, Y = ckgen.states(cfg, N=32)
    lnKc = ann_forward_matrix_form(ann, T)                               # [N, R]
    om = oracle.OracleMechanism(mech, kc_ann=ann)
    for i in (0, 7, 31):
        det = oracle.cell_detail(om, T[i], P[i], Y[:, i])
        np.testing.assert_allclose(np.log(det["Kc"]), lnKc[i], rtol=1e-12, atol=1e-12)
        # Eq. 7 with the approximate constant: k_r = k_f / Kc~
        np.testing.assert_allclose(det["kr"], det["kf"] / np.exp(lnKc[i]), rtol=1e-11)
