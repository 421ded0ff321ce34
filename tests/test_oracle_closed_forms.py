"""Pins the oracle to hand-derivable single-reaction closed forms (north_star:
"hand-computed single-reaction closed forms").

Expected values come from tests/golden/closed_forms.json (50-digit mpmath evaluation of
the closed-form formulas, written by tests/golden/make_closed_forms.py, which does not
call the oracle) and, independently, from the numbers printed in SURVEY.md section 8(c).
A dropped term, wrong sign, transposed index or wrong unit in the oracle's Arrhenius,
NASA-7, Kc, concentration, third-body, falloff or energy step fails one of them.
"""
import json
import math
import os

import numpy as np
import pytest

import ckgen
import oracle

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))
INF = float("inf")


def two_species_mech(W, a1, a6, a7, nu_r, nu_p, rxn_type=0, E=(1.0, 1.0), k0=None,
                     troe=(0.0, 1.0, 1.0, 1.0)):
    S, R = 2, 1
    nasa = np.zeros((S, 7))
    nasa[:, 0], nasa[:, 5], nasa[:, 6] = a1, a6, a7
    return ckgen.Mechanism(
        elements=("X",), elem_count=np.array([[1], [1]]), mol_weight=np.array(W, float),
        nu_reac=np.array(nu_r, float).reshape(S, R), nu_prod=np.array(nu_p, float).reshape(S, R),
        ln_A=np.array([math.log(1e10)]), b=np.array([0.5]), Ea_over_R=np.array([1.0e4]),
        reversible=np.ones(R, np.uint8), nasa_lo=nasa.copy(), nasa_hi=nasa.copy(),
        T_mid=np.full(S, 1000.0), rxn_type=np.array([rxn_type], np.uint8),
        eff=np.array(E, float).reshape(S, R),
        ln_A0=np.array([math.log(k0) if k0 else 0.0]), b0=np.zeros(R), Ea0_over_R=np.zeros(R),
        troe=np.array([troe], float), p_ref=101325.0)


CASES = {
    "ex1_isomerisation": dict(W=(20, 20), a1=(3.5, 3.5), a6=(0, -5000), a7=(2, 3),
                              nu_r=(1, 0), nu_p=(0, 1)),
    "ex2_recombination": dict(W=(20, 40), a1=(3.5, 4.5), a6=(0, -12000), a7=(2, 1.5),
                              nu_r=(2, 0), nu_p=(0, 1)),
    "ex3_three_body": dict(W=(20, 20), a1=(3.5, 3.5), a6=(0, -5000), a7=(2, 3),
                           nu_r=(1, 0), nu_p=(0, 1), rxn_type=1, E=(2.0, 0.5)),
    "ex4_troe": dict(W=(20, 20), a1=(3.5, 3.5), a6=(0, -5000), a7=(2, 3), nu_r=(1, 0),
                     nu_p=(0, 1), rxn_type=3, E=(2.0, 0.5), k0=1e12,
                     troe=(0.6, 200.0, 1500.0, 5000.0)),
    "ex4_lindemann": dict(W=(20, 20), a1=(3.5, 3.5), a6=(0, -5000), a7=(2, 3), nu_r=(1, 0),
                          nu_p=(0, 1), rxn_type=2, E=(2.0, 0.5), k0=1e12),
    "ex4_troe3": dict(W=(20, 20), a1=(3.5, 3.5), a6=(0, -5000), a7=(2, 3), nu_r=(1, 0),
                      nu_p=(0, 1), rxn_type=3, E=(2.0, 0.5), k0=1e12,
                      troe=(0.6, 200.0, 1500.0, INF)),
}

# SURVEY.md section 8(c), "Closed forms, worked numbers" (an independent evaluation)
SURVEY_PRINTED = {
    "ex1_isomerisation": dict(lnKc=6.0, Kc=403.4287934927351, kf=14356718.36611194,
                              rho=0.2437319274940843, q=131111.2286646428,
                              dTdt=15369488696.94144),
    "ex2_recombination": dict(lnKc=-0.8619696084343845, Kc=0.42232943897116,
                              rho=0.2785507742789535, q=-57615.32005798444,
                              dTdt=-18818344435.36366),
    "ex3_three_body": dict(M=0.01980321910889435, q=2596.42438888227),
    "ex4_troe": dict(Pr=1379.369477333937, kf=12974090.93994502, q=118484.5283277418),
    "ex4_lindemann": dict(kf=14346317.73164279, q=131016.2459583329),
}


def run(name):
    mech = two_species_mech(**CASES[name])
    om = oracle.OracleMechanism(mech)
    Y = np.array([0.75, 0.25])
    det = oracle.cell_detail(om, 1000.0, 101325.0, Y)
    w, d, _ = oracle.source_terms(om, np.array([1000.0]), np.array([101325.0]), Y.reshape(2, 1))
    # the batched entry point and the detail entry point are the same computation
    assert np.array_equal(w[:, 0], det["wdot"]) and d[0] == det["dTdt"]
    return mech, det


@pytest.mark.parametrize("name", list(CASES))
def test_oracle_matches_50_digit_closed_form(name):
    mech, det = run(name)
    g = GOLD[name]
    rel = lambda a, b: abs(a - b) / max(abs(b), 1e-300)
    nu = (mech.nu_prod - mech.nu_reac)[:, 0]
    assert rel(det["rho"], float(g["rho"])) < 1e-14
    for k in range(2):
        assert rel(det["C"][k], float(g["C"][k])) < 1e-14
        assert rel(det["g_RT"][k], float(g["g_RT"][k])) < 1e-14
        assert rel(det["wdot"][k], float(g["wdot"][k])) < 1e-12
    assert abs(math.log(det["Kc"][0]) - float(g["lnKc"])) < 1e-13
    assert rel(det["kf"][0], float(g["kf"])) < 1e-13
    assert rel(det["Q"][0], float(g["q"])) < 1e-12
    assert rel(det["dTdt"], float(g["dTdt"])) < 1e-12
    if "M" in g:
        assert rel(det["M"][0], float(g["M"])) < 1e-14
    # Eq. 2 for a single reaction: wdot_k = nu_k q ; and mass is conserved
    assert np.allclose(det["wdot"], nu * det["Q"][0], rtol=1e-15)
    assert abs((mech.mol_weight * det["wdot"]).sum()) <= 1e-12 * np.abs(mech.mol_weight * det["wdot"]).sum()


@pytest.mark.parametrize("name", list(SURVEY_PRINTED))
def test_oracle_matches_numbers_printed_in_survey(name):
    _, det = run(name)
    exp = SURVEY_PRINTED[name]
    got = dict(lnKc=math.log(det["Kc"][0]), Kc=det["Kc"][0], kf=det["kf"][0], rho=det["rho"],
               q=det["Q"][0], dTdt=det["dTdt"], M=det["M"][0])
    if "Pr" in exp:
        om = oracle.OracleMechanism(two_species_mech(**{**CASES[name], "rxn_type": 0}))
        kinf = oracle.cell_detail(om, 1000.0, 101325.0, np.array([0.75, 0.25]))["kf"][0]
        got["Pr"] = 1e12 * det["M"][0] / kinf
    for key, val in exp.items():
        assert abs(got[key] - val) <= 2e-13 * abs(val) + 1e-15, (name, key, got[key], val)


def test_ex1_hand_values():
    """Numbers a reader can check on paper: ln Kc = 6 by construction
    (g_A - g_B = a6_A/T - a7_A - a6_B/T + a7_B = 0 - 2 + 5 + 3), sum(nu) = 0."""
    _, det = run("ex1_isomerisation")
    assert abs(math.log(det["Kc"][0]) - 6.0) < 1e-13
    kf = 1e10 * math.sqrt(1000.0) * math.exp(-10.0)
    assert abs(det["kf"][0] - kf) < 1e-13 * kf
    # dT/dt = 5000 * q * 20 / (3.5 rho): only B carries enthalpy (a6 = -5000 K), W = 20
    q, rho = det["Q"][0], det["rho"]
    assert abs(det["dTdt"] - 5000.0 * q * 20.0 / (3.5 * rho)) < 1e-12 * abs(det["dTdt"])


def test_troe_limits():
    """Pr -> 0: k -> k0 M F (low-pressure limit, F -> Fcent^(1/(1+f1^2)) with f1 -> 1/0.14
    in magnitude); Pr -> infinity: k -> k_inf (F -> 1 because f1 -> -1/0.14 ... bounded,
    so check through Lindemann where F = 1 exactly)."""
    Y = np.array([0.75, 0.25])
    base = CASES["ex4_lindemann"]
    for k0, expect in ((1e-6, "low"), (1e30, "high")):
        om = oracle.OracleMechanism(two_species_mech(**{**base, "k0": k0}))
        det = oracle.cell_detail(om, 1000.0, 101325.0, Y)
        kinf = 1e10 * math.sqrt(1000.0) * math.exp(-10.0)
        if expect == "low":
            assert abs(det["kf"][0] - k0 * det["M"][0]) < 1e-9 * k0 * det["M"][0]
        else:
            assert abs(det["kf"][0] - kinf) < 1e-9 * kinf
    # Troe with alpha = 1 and T** = inf: Fcent = exp(-T/T*), the one-term form
    om = oracle.OracleMechanism(two_species_mech(**{**CASES["ex4_troe"], "troe": (1.0, 200.0, 1500.0, INF)}))
    det = oracle.cell_detail(om, 1000.0, 101325.0, Y)
    Fc = math.exp(-1000.0 / 1500.0)
    lFc = math.log10(Fc)
    Pr = float(GOLD["ex4_troe"]["Pr"])
    c, n = -0.4 - 0.67 * lFc, 0.75 - 1.27 * lFc
    f1 = (math.log10(Pr) + c) / (n - 0.14 * (math.log10(Pr) + c))
    F = 10 ** (lFc / (1 + f1 * f1))
    kinf = float(GOLD["ex4_troe"]["k_inf"])
    assert abs(det["kf"][0] - kinf * Pr / (1 + Pr) * F) < 1e-13 * kinf


@pytest.mark.parametrize("name,k0", [("ex4_troe_low_pressure", 7.25e-4), ("ex4_troe_high_pressure", 7.25e20)])
def test_troe_pressure_limits_with_F_active(name, k0):
    """Troe falloff twelve decades into either pressure limit (Pr = 1e-12, 1e+12), F != 1 in both
    (PAPER.md:159 gives no formula; the textbook form at 50 digits, closed_forms.json).  The low
    limit is k = k0 M F to 1e-12, the high one k = k_inf F to 1e-12."""
    g = GOLD[name]
    mech = two_species_mech(**{**CASES["ex4_troe"], "k0": k0})
    det = oracle.cell_detail(oracle.OracleMechanism(mech), 1000.0, 101325.0, np.array([0.75, 0.25]))
    rel = lambda a, b: abs(a - b) / abs(b)
    assert rel(det["kf"][0], float(g["kf"])) < 1e-13
    assert rel(det["Q"][0], float(g["q"])) < 1e-12
    assert rel(det["dTdt"], float(g["dTdt"])) < 1e-12
    F, Pr, kinf, M = float(g["F"]), float(g["Pr"]), float(g["k_inf"]), float(g["M"])
    assert abs(F - 1.0) > 5e-4                                   # the factor is active
    if Pr < 1:
        assert rel(det["kf"][0], k0 * M * F) < 2e-12             # Pr/(1+Pr) -> Pr
    else:
        assert rel(det["kf"][0], kinf * F) < 2e-12               # Pr/(1+Pr) -> 1


def nasa7_mech():
    """Ex5 of tests/golden/make_closed_forms.py: A + 2 B <=> C, full NASA-7 sets (typed here
    as floats from the same table; the golden file holds the 50-digit results, not the inputs)."""
    lo = np.array([[3.2, 1.1e-3, -2.4e-6, 3.1e-9, -1.2e-12, -950.0, 0.7],
                   [2.9, 2.4e-3, -4.1e-6, 2.2e-9, -0.7e-12, 29100.0, 4.9],
                   [4.3, -0.6e-3, 8.8e-6, -9.1e-9, 3.2e-12, -17800.0, 3.4]])
    hi = np.array([[3.0, 0.8e-3, -0.11e-6, 0.02e-9, -0.002e-12, -830.0, -1.1],
                   [2.6, -0.03e-3, 0.05e-6, -0.01e-9, 0.001e-12, 29200.0, 4.8],
                   [4.6, 4.1e-3, -1.3e-6, 0.21e-9, -0.012e-12, -18000.0, 0.6]])
    S, R = 3, 1
    return ckgen.Mechanism(
        elements=("X",), elem_count=np.array([[2], [16], [34]]), mol_weight=np.array([2.0, 16.0, 34.0]),
        nu_reac=np.array([[1.0], [2.0], [0.0]]), nu_prod=np.array([[0.0], [0.0], [1.0]]),
        ln_A=np.array([math.log(3e11)]), b=np.array([-0.7]), Ea_over_R=np.array([6500.0]),
        reversible=np.ones(R, np.uint8), nasa_lo=lo, nasa_hi=hi, T_mid=np.full(S, 1000.0),
        rxn_type=np.zeros(R, np.uint8), eff=np.ones((S, R)), ln_A0=np.zeros(R), b0=np.zeros(R),
        Ea0_over_R=np.zeros(R), troe=np.ones((R, 4)), p_ref=101325.0)


@pytest.mark.parametrize("T", [800, 1000, 1600])
def test_full_nasa7_set_in_both_ranges(T):
    """Every NASA-7 coefficient non-zero, different sets below and above T_mid (PAPER.md:101-108,
    Eq. 10): cp/R, h/RT, s/R, g/RT, ln Kc, the rate and dT/dt against the 50-digit evaluation.
    A wrong divisor of a2..a5 in h or s, a swapped range or a missing a6/T, a7 fails here; T = 1000
    is exactly T_mid and must take the LOW set (reading Q4)."""
    g = GOLD["ex5_nasa7_T%d" % T]
    det = oracle.cell_detail(oracle.OracleMechanism(nasa7_mech()), float(T), 3 * 101325.0,
                             np.array([0.2, 0.5, 0.3]))
    rel = lambda a, b: abs(a - b) / max(abs(b), 1e-300)
    for k in range(3):
        for key in ("cp_R", "h_RT", "s_R", "g_RT", "C"):
            assert rel(det[key][k], float(g[key][k])) < 2e-14, (key, k)
        assert rel(det["wdot"][k], float(g["wdot"][k])) < 1e-12
    assert abs(math.log(det["Kc"][0]) - float(g["lnKc"])) < 2e-13
    assert rel(det["kf"][0], float(g["kf"])) < 1e-13
    assert rel(det["Q"][0], float(g["q"])) < 1e-12
    assert rel(det["cp_mass"], float(g["cp_mass"])) < 1e-14
    assert rel(det["dTdt"], float(g["dTdt"])) < 1e-12
    # the two sets really differ at these states (the test cannot pass with the ranges swapped)
    other = oracle.cell_detail(oracle.OracleMechanism(nasa7_mech()), float(T) + (400.0 if T <= 1000 else -800.0),
                               3 * 101325.0, np.array([0.2, 0.5, 0.3]))
    assert abs(other["cp_R"][2] - det["cp_R"][2]) > 0.05


def test_irreversible_has_no_reverse_rate():
    mech = two_species_mech(**CASES["ex1_isomerisation"])
    mech.reversible[:] = 0
    det = oracle.cell_detail(oracle.OracleMechanism(mech), 1000.0, 101325.0, np.array([0.75, 0.25]))
    g = GOLD["ex1_isomerisation"]
    assert det["qr"][0] == 0.0 and det["kr"][0] == 0.0
    assert abs(det["Q"][0] - float(g["k_inf"]) * float(g["C"][0])) < 1e-13 * det["Q"][0]
