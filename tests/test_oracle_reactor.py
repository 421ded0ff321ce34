"""Pins oracle/reactor.py (the explicit RK4 constant-pressure reactor step built on the
oracle's source term) to things fixed outside it:

* the stability polynomial of the classic 4-stage scheme on a linear case, at 50 digits
  (tests/golden/reactor_closed_form.json, written by make_reactor_closed_form.py, which
  does not call the oracle): a wrong stage coefficient or weight changes R(z);
* linear invariants of the unprojected update (sum Y and every element);
* the projection's definition (reading Q14);
* fourth-order convergence against a much smaller step on a tamed random mechanism.
"""
import json
import os

import numpy as np

import ckgen
import oracle
from oracle import reactor
from helpers import tame
from test_oracle_closed_forms import two_species_mech

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "reactor_closed_form.json")))


def thermoneutral_isomerisation():
    return two_species_mech(W=(20, 20), a1=(3.5, 3.5), a6=(0, 0), a7=(2, 3), nu_r=(1, 0), nu_p=(0, 1))


def test_stability_polynomial_of_the_scheme():
    mech = thermoneutral_isomerisation()
    om = oracle.OracleMechanism(mech)
    for case in GOLD["cases"]:
        dt = float(case["dt"])
        T, P, Y = np.array([1000.0]), np.array([101325.0]), np.array([[0.75], [0.25]])
        for want in case["Y_A_after_steps_1_2_3"]:
            T, Y = reactor.rk4_step(om, mech.mol_weight, T, P, Y, dt)
            assert T[0] == 1000.0                         # thermoneutral: dT/dt = 0 exactly
            assert abs(Y[0, 0] - float(want)) <= 2e-14, (dt, Y[0, 0], want)
            assert abs(Y.sum() - 1.0) <= 1e-15
        # and the scheme is NOT the exact flow: R(z) differs from e^z at this step size
        if dt >= 2e-8:
            y_eq = float(GOLD["Y_A_eq"])
            exact = y_eq + float(case["exp_z"]) ** 3 * (0.75 - y_eq)
            assert abs(Y[0, 0] - exact) > 1e-6


def test_projection_definition():
    T = np.array([100.0, 6000.0, 1200.0])
    Y = np.array([[0.5, -0.2, 2.0], [0.7, 0.6, 2.0], [-0.1, 0.2, 0.0]])
    Tp, Yp = reactor.project(T, Y)
    assert Tp.tolist() == [250.0, 5000.0, 1200.0]
    np.testing.assert_allclose(Yp[:, 0], [0.5 / 1.2, 0.7 / 1.2, 0.0], rtol=1e-15)
    np.testing.assert_allclose(Yp[:, 1], [0.0, 0.75, 0.25], rtol=1e-15)
    np.testing.assert_allclose(Yp[:, 2], [0.5, 0.5, 0.0], rtol=1e-15)


def test_unprojected_update_conserves_mass_and_elements():
    """RK schemes preserve linear invariants: sum_k Y_k and sum_k n_ek Y_k / W_k move only by
    rounding (the source term conserves them, tests/test_oracle_invariants.py)."""
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = tame(ckgen.mechanism(cfg.mech))
    om = oracle.OracleMechanism(mech)
    T, P, Y = ckgen.states(cfg, N=64)
    _, _, (Tn, Yn) = reactor.rk4_step(om, mech.mol_weight, T, P, Y, 1e-9, return_stages=True)
    assert np.abs(Yn.sum(0) - 1.0).max() <= 1e-14
    el0 = mech.elem_count.T @ (Y / mech.mol_weight[:, None])
    el1 = mech.elem_count.T @ (Yn / mech.mol_weight[:, None])
    assert np.abs(el1 - el0).max() <= 1e-14 * np.abs(el0).max()
    assert np.abs(Yn - Y).max() > 1e-9                      # something did happen


def test_fourth_order_convergence():
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = tame(ckgen.mechanism(cfg.mech))
    om = oracle.OracleMechanism(mech)
    T, P, Y = ckgen.states(cfg, N=16)
    t_end = 4e-6
    ref = reactor.integrate(om, mech.mol_weight, T, P, Y, t_end / 256, 256)
    errs = []
    for n in (4, 8, 16):
        Tn, Yn = reactor.integrate(om, mech.mol_weight, T, P, Y, t_end / n, n)
        errs.append(max(np.abs(Yn - ref[1]).max(), np.abs(Tn - ref[0]).max() / 2000.0))
    assert errs[0] > 1e-13, "the test problem is too easy to show an order: %r" % errs
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(3.5 < o < 4.8 for o in orders), (errs, orders)
