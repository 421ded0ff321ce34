"""Pins of the oracle's analytic Jacobian (oracle/ck_oracle_jac.c), d(wdot, dT/dt)/d(Y, T) at
constant P, to things other than itself:

* 50-digit derivatives of the single-reaction closed forms (tests/golden/
  jacobian_closed_form.json, mpmath differentiation of make_closed_forms.py's definition;
  elementary, recombination, three-body, Lindemann, 4- and 3-parameter Troe, two states each);
* central finite differences of oracle.source_terms (pinned by test_oracle_closed_forms /
  test_oracle_invariants) on the generated mechanisms, every column, both NASA ranges;
* Euler's theorem: the source term is homogeneous of degree 0 in Y (C_k depends on the mole
  fractions and P/(Ru T) only), hence sum_l Y_l J_il = 0 for every row;
* conservation: sum_i W_i J_il = 0 and sum_i n_ei J_il = 0 for every column (reactions are
  element balanced), the derivative of the invariants pinned in test_oracle_invariants.
A dropped chain-rule term, a wrong sign, a transposed index, a missing efficiency or Troe
derivative fails one of them.
"""
import json
import os

import numpy as np
import pytest

import ckgen
import oracle
from test_oracle_closed_forms import CASES, two_species_mech

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "jacobian_closed_form.json")))


@pytest.mark.parametrize("name", [k for k in GOLD if not k.startswith("_")])
def test_closed_form_jacobians(name):
    g = GOLD[name]
    mech = two_species_mech(**CASES[name.split("@")[0]])
    J = oracle.jacobian(oracle.OracleMechanism(mech), np.array([float(g["T"])]), np.array([float(g["P"])]),
                        np.array([[float(y)] for y in g["Y"]]))[0]
    ref = np.array([[float(v) for v in row] for row in g["J"]])
    # every entry to 1e-11 of its own size (they are all far from cancellation in these cases),
    # with the column's largest entry as floor for the few that are small differences
    tol = 1e-11 * np.abs(ref) + 1e-13 * np.abs(ref).max(axis=0, keepdims=True)
    assert (np.abs(J - ref) <= tol).all(), (name, J, ref)


def fd_jacobian(om, T, P, Y, rel=2e-6):
    """Central differences of the source-term oracle, one column at a time; N cells at once."""
    S, N = Y.shape
    J = np.empty((N, S + 1, S + 1))
    for l in range(S + 1):
        Tp, Tm, Yp, Ym = T.copy(), T.copy(), Y.copy(), Y.copy()
        if l < S:
            h = rel * np.maximum(Y[l], 1e-3)
            Yp[l] += h
            Ym[l] -= h
            # keep the lower point positive (the floor on C is not differentiated)
            assert (Ym[l] > 0).all()
        else:
            h = rel * T
            Tp, Tm = T + h, T - h
        wp, dp, _ = oracle.source_terms(om, Tp, P, Yp)
        wm, dm, _ = oracle.source_terms(om, Tm, P, Ym)
        J[:, :S, l] = ((wp - wm) / (2 * h)).T
        J[:, S, l] = (dp - dm) / (2 * h)
    return J


def column_scale(J):
    """Per cell and column: the largest species-row entry, and for the energy row its own size."""
    S = J.shape[1] - 1
    sc = np.empty_like(J)
    sc[:, :S, :] = np.abs(J[:, :S, :]).max(axis=1, keepdims=True)
    sc[:, S, :] = np.abs(J[:, S, :]).max(axis=1, keepdims=True)
    return sc


@pytest.mark.parametrize("cfg_name,N", [("tiny_1k", 24), ("mid_1m", 6), ("large_256k", 2)])
def test_finite_differences(cfg_name, N):
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    # Y far from the floor so that the lower finite-difference point stays physical
    Y = np.maximum(Y, 2e-3)
    Y /= Y.sum(0)
    T[: N // 3] = np.linspace(400.0, 990.0, N // 3)      # low NASA range too
    om = oracle.OracleMechanism(mech)
    J = oracle.jacobian(om, T, P, Y)
    Jfd = fd_jacobian(om, T, P, Y)
    err = np.abs(J - Jfd) / column_scale(J)
    assert err.max() < 2e-6, (cfg_name, err.max(), np.unravel_index(err.argmax(), err.shape))


@pytest.mark.parametrize("cfg_name", ["tiny_1k", "mid_1m"])
def test_euler_homogeneity_and_conservation(cfg_name):
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=40)
    T[:10] = np.linspace(500.0, 999.0, 10)
    J = oracle.jacobian(oracle.OracleMechanism(mech), T, P, Y)
    S = mech.n_species
    # Euler: sum_l Y_l J_il = 0, measured against sum_l |Y_l J_il|
    terms = J[:, :, :S] * Y.T[:, None, :]
    assert (np.abs(terms.sum(2)) <= 1e-10 * np.abs(terms).sum(2) + 1e-300).all()
    # conservation of mass and of every element, column by column
    weights = [mech.mol_weight] + [mech.elem_count[:, e].astype(float) for e in range(mech.elem_count.shape[1])]
    for w in weights:
        t = J[:, :S, :] * w[None, :, None]
        assert (np.abs(t.sum(1)) <= 1e-10 * np.abs(t).sum(1) + 1e-300).all()


def test_jacobian_does_not_depend_on_normalisation_scaling():
    """f(cY) = f(Y)  =>  J(cY) = J(Y)/c on the Y columns, unchanged on the T column."""
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=8)
    om = oracle.OracleMechanism(mech)
    J1, J2 = oracle.jacobian(om, T, P, Y), oracle.jacobian(om, T, P, 2.5 * Y)
    S = mech.n_species
    sc = column_scale(J1)
    assert (np.abs(J2[:, :, :S] * 2.5 - J1[:, :, :S]) <= 1e-11 * sc[:, :, :S]).all()
    assert (np.abs(J2[:, :, S] - J1[:, :, S]) <= 1e-11 * sc[:, :, S]).all()


def test_finite_differences_with_catalyst_real_nu_irreversible_and_lindemann():
    """The branches the generated mechanisms do not reach: a species on both sides of a reaction,
    a real-valued stoichiometric coefficient (pow), irreversible reactions, Lindemann falloff and
    the 3-parameter Troe form."""
    import dataclasses
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    nu_r, nu_p = mech.nu_reac.copy(), mech.nu_prod.copy()
    free = int(np.flatnonzero((nu_r[:, 0] == 0) & (nu_p[:, 0] == 0))[0])
    nu_r[free, 0] += 1.0
    nu_p[free, 0] += 1.0
    k = int(np.flatnonzero(nu_r[:, 1])[0])
    nu_r[k, 1] = 1.5
    rev = mech.reversible.copy()
    rev[::3] = 0
    typ = mech.rxn_type.copy()
    troe = mech.troe.copy()
    fo = np.flatnonzero(typ == 3)
    typ[fo[0]] = 2
    troe[fo[1:], 3] = np.inf
    mech = dataclasses.replace(mech, nu_reac=nu_r, nu_prod=nu_p, reversible=rev, rxn_type=typ, troe=troe)
    T, P, Y = ckgen.states(cfg, N=16)
    Y = np.maximum(Y, 2e-3)
    Y /= Y.sum(0)
    om = oracle.OracleMechanism(mech)
    J = oracle.jacobian(om, T, P, Y)
    err = np.abs(J - fd_jacobian(om, T, P, Y)) / column_scale(J)
    assert err.max() < 2e-6, err.max()
