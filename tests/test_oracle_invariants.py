"""Pins the oracle to what the mathematics fixes for any mechanism and state
(SURVEY.md section 8(c) "Invariants", "Detailed balance", "Special cases"), and to a
numpy restatement of the paper's matrix equations (tests/helpers.paper_matrix_form)."""
import dataclasses

import numpy as np
import pytest

import ckgen
import oracle
from helpers import RU, paper_matrix_form, parity_violations

SPECS = [ckgen.MECH_TINY, ckgen.MECH_MID]
CFG_OF = {"S9_R21": "tiny_1k", "S53_R325": "mid_1m", "S111_R784": "large_256k"}


def mech_and_states(spec, N, T_range=None):
    mech = ckgen.mechanism(spec)
    cfg = ckgen.CONFIGS[CFG_OF[spec.name]]
    if T_range is not None:
        cfg = dataclasses.replace(cfg, T_range=T_range)
    T, P, Y = ckgen.states(cfg, N=N)
    return mech, T, P, Y


@pytest.mark.parametrize("spec", SPECS + [ckgen.MECH_LARGE], ids=lambda s: s.name)
def test_mass_and_element_conservation(spec):
    """sum_k W_k wdot_k = 0 and sum_k n_ek wdot_k = 0: reactions are element balanced and
    W comes from the element counts, so Eq. 2 conserves both."""
    mech, T, P, Y = mech_and_states(spec, 256, T_range=(300.0, 3000.0))
    w, d, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    assert np.isfinite(w).all() and np.isfinite(d).all()
    for weights in [mech.mol_weight] + [mech.elem_count[:, e].astype(float)
                                        for e in range(mech.elem_count.shape[1])]:
        terms = weights[:, None] * w
        assert (np.abs(terms.sum(0)) <= 1e-12 * np.abs(terms).sum(0) + 1e-300).all()


@pytest.mark.parametrize("spec", SPECS, ids=lambda s: s.name)
def test_thermo_identities_by_finite_differences(spec):
    """d(g/RT)/dT = -(h/RT)/T, d(h/R)/dT = cp/R, d(s/R)/dT = (cp/R)/T: fixes every NASA-7
    divisor (1/2..1/5, 1/2..1/4) and the a6, a7 placement.  4th-order central differences
    (exact for these polynomials up to rounding); both temperature ranges."""
    mech = ckgen.mechanism(spec)
    om = oracle.OracleMechanism(mech)
    Y = np.full(mech.n_species, 1.0 / mech.n_species)
    for T in (450.0, 999.0, 1001.0, 1700.0, 3100.0):
        h = 0.25
        f = {dT: oracle.cell_detail(om, T + dT, 2e5, Y) for dT in (-2 * h, -h, 0.0, h, 2 * h)}

        def ddT(fun):
            v = {k: fun(f[k], T + k) for k in f}
            return (v[-2 * h] - 8 * v[-h] + 8 * v[h] - v[2 * h]) / (12 * h)

        c = f[0.0]
        np.testing.assert_allclose(ddT(lambda d, t: d["g_RT"]), -c["h_RT"] / T, rtol=2e-9, atol=1e-12)
        np.testing.assert_allclose(ddT(lambda d, t: d["h_RT"] * t), c["cp_R"], rtol=2e-9)
        np.testing.assert_allclose(ddT(lambda d, t: d["s_R"]), c["cp_R"] / T, rtol=2e-9, atol=1e-14)
        np.testing.assert_allclose(c["g_RT"], c["h_RT"] - c["s_R"], rtol=1e-15)


def test_range_switch_at_T_mid():
    """T <= T_mid takes the low range (reading Q4): make the two ranges differ
    grossly and look at cp on either side of and exactly at the switch."""
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    hi = mech.nasa_hi.copy()
    hi[:, 0] += 100.0
    mech = dataclasses.replace(mech, nasa_hi=hi)
    om = oracle.OracleMechanism(mech)
    Y = np.full(mech.n_species, 1.0 / mech.n_species)
    at = oracle.cell_detail(om, 1000.0, 1e5, Y)["cp_R"]
    below = oracle.cell_detail(om, np.nextafter(1000.0, 0), 1e5, Y)["cp_R"]
    above = oracle.cell_detail(om, np.nextafter(1000.0, 2000), 1e5, Y)["cp_R"]
    assert np.allclose(at, below, rtol=1e-12) and (above - at > 99.0).all()


@pytest.mark.parametrize("spec", SPECS, ids=lambda s: s.name)
def test_detailed_balance_at_constructed_equilibrium(spec):
    """With ln C_k = -g_k/RT + ln(p_ref/(Ru T)) + sum_e lambda_e n_ek every element-balanced
    reversible reaction has q_f = q_r, third bodies and falloff included."""
    mech = ckgen.mechanism(spec)
    om = oracle.OracleMechanism(mech)
    rng = np.random.default_rng(7)
    S = mech.n_species
    for T in (800.0, 1500.0, 2600.0):
        g = oracle.cell_detail(om, T, 1e5, np.full(S, 1.0 / S))["g_RT"]   # g depends on T only
        lam = rng.uniform(-3.0, 0.0, size=mech.elem_count.shape[1])
        lnC = -g + np.log(mech.p_ref / (RU * T)) + mech.elem_count @ lam
        # keep the largest concentration moderate by adding the same amount to every
        # lambda_e (a uniform shift of ln C itself would not be of the equilibrium form)
        n_atoms = mech.elem_count.sum(1).astype(float)
        lo, hi = -200.0, 200.0                      # bisection: max_k ln C_k = ln 1e-3
        for _ in range(100):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if (lnC + mid * n_atoms).max() < np.log(1e-3) else (lo, mid)
        lnC = lnC + lo * n_atoms
        C = np.exp(lnC)
        P = C.sum() * RU * T
        Y = C * mech.mol_weight / (C * mech.mol_weight).sum()
        det = oracle.cell_detail(om, T, P, Y)
        np.testing.assert_allclose(det["C"], C, rtol=1e-12)
        assert (np.abs(det["qf"] - det["qr"]) <= 1e-11 * det["qf"]).all()
        dnu = np.abs(mech.nu_prod - mech.nu_reac)
        phi = np.where(mech.rxn_type == 1, det["M"], 1.0)
        assert (np.abs(det["wdot"]) <= 1e-10 * (dnu @ (phi * det["qf"]))).all()


@pytest.mark.parametrize("spec", SPECS, ids=lambda s: s.name)
def test_Kc_and_kf_do_not_depend_on_pressure_or_composition(spec):
    mech = ckgen.mechanism(spec)
    elementary = np.flatnonzero(mech.rxn_type == 0)
    om = oracle.OracleMechanism(mech)
    _, T, P, Y = mech_and_states(spec, 2)
    a = oracle.cell_detail(om, 1234.5, P[0], Y[:, 0])
    b = oracle.cell_detail(om, 1234.5, 7.0 * P[1], Y[:, 1])
    np.testing.assert_allclose(a["Kc"], b["Kc"], rtol=1e-15)
    np.testing.assert_allclose(a["kf"][elementary], b["kf"][elementary], rtol=1e-15)


def test_power_law_Kc_when_only_a1_is_nonzero():
    """NASA a2..a7 = 0: g/RT = a1 (1 - ln T), so Kc = (p_ref/(Ru T))^dn * (T/e)^(sum nu a1)."""
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    lo = np.zeros_like(mech.nasa_lo)
    lo[:, 0] = np.linspace(2.5, 6.0, mech.n_species)
    mech = dataclasses.replace(mech, nasa_lo=lo, nasa_hi=lo.copy())
    det = oracle.cell_detail(oracle.OracleMechanism(mech), 1400.0, 1e5,
                             np.full(mech.n_species, 1.0 / mech.n_species))
    nu = mech.nu_prod - mech.nu_reac
    expect = (mech.p_ref / (RU * 1400.0)) ** nu.sum(0) * (1400.0 / np.e) ** (lo[:, 0] @ nu)
    np.testing.assert_allclose(det["Kc"], expect, rtol=1e-12)


@pytest.mark.parametrize("spec", SPECS, ids=lambda s: s.name)
def test_wdot_is_linear_in_third_body_concentration(spec):
    """Doubling every efficiency of the three-body reactions doubles their Q and leaves
    the others alone (Q7: M multiplies both directions)."""
    mech = ckgen.mechanism(spec)
    tb = mech.rxn_type == 1
    eff2 = mech.eff.copy()
    eff2[:, tb] *= 2.0
    _, T, P, Y = mech_and_states(spec, 1)
    a = oracle.cell_detail(oracle.OracleMechanism(mech), T[0], P[0], Y[:, 0])
    b = oracle.cell_detail(oracle.OracleMechanism(dataclasses.replace(mech, eff=eff2)), T[0], P[0], Y[:, 0])
    np.testing.assert_allclose(b["Q"][tb], 2.0 * a["Q"][tb], rtol=1e-14)
    np.testing.assert_array_equal(b["Q"][mech.rxn_type == 0], a["Q"][mech.rxn_type == 0])
    np.testing.assert_allclose(a["M"][tb], a["C"] @ mech.eff[:, tb], rtol=1e-14)


@pytest.mark.parametrize("spec", SPECS, ids=lambda s: s.name)
def test_all_irreversible_equals_forward_rates_only(spec):
    mech = ckgen.mechanism(spec)
    _, T, P, Y = mech_and_states(spec, 1)
    rev = oracle.cell_detail(oracle.OracleMechanism(mech), T[0], P[0], Y[:, 0])
    irr = oracle.cell_detail(oracle.OracleMechanism(
        dataclasses.replace(mech, reversible=np.zeros(mech.n_reactions, np.uint8))), T[0], P[0], Y[:, 0])
    assert (irr["qr"] == 0).all()
    np.testing.assert_array_equal(irr["qf"], rev["qf"])
    nu = mech.nu_prod - mech.nu_reac
    phi = np.where(mech.rxn_type == 1, rev["M"], 1.0)
    np.testing.assert_allclose(irr["wdot"], nu @ (phi * rev["qf"]), rtol=1e-12,
                               atol=1e-13 * np.abs(nu @ (phi * rev["qf"])).max())


@pytest.mark.parametrize("spec,N,T_range", [
    (ckgen.MECH_TINY, 512, None), (ckgen.MECH_TINY, 256, (300.0, 1100.0)),
    (ckgen.MECH_MID, 256, None), (ckgen.MECH_MID, 128, (300.0, 1100.0)),
    (ckgen.MECH_LARGE, 64, None)], ids=lambda x: getattr(x, "name", str(x)))
def test_oracle_agrees_with_paper_matrix_form(spec, N, T_range):
    """Two derivations of the same result: the oracle's product-form rate law (Eq. 3, 5, 7,
    8) and the paper's log-space matrix layers (Eq. 2, 4, 6, 10, 11) in dense numpy."""
    mech, T, P, Y = mech_and_states(spec, N, T_range)
    w, d, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    Om, dT = paper_matrix_form(mech, T, P, Y)
    wmax = np.abs(w).max(0)
    assert (np.abs(Om.T - w) <= 1e-11 * wmax[None, :]).all()
    assert (np.abs(dT - d) <= 1e-9 * np.abs(d) + 1e-12).all()


def test_non_integer_and_absent_species():
    """Real-valued nu goes through pow; Y = 0 acts as an absent species
    through the 1e-300 floor (reading Q9) and gives finite rates equal to the matrix form."""
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    nu_r = mech.nu_reac.copy()
    j = 0
    k = int(np.flatnonzero(nu_r[:, j])[0])
    nu_r[k, j] = 1.5
    mech2 = dataclasses.replace(mech, nu_reac=nu_r)
    _, T, P, Y = mech_and_states(ckgen.MECH_TINY, 8)
    Y = Y.copy()
    Y[2, :4] = 0.0
    Y /= Y.sum(0, keepdims=True)
    w, d, _ = oracle.source_terms(oracle.OracleMechanism(mech2), T, P, Y)
    Om, dT = paper_matrix_form(mech2, T, P, Y)
    assert np.isfinite(w).all()
    assert (np.abs(Om.T - w) <= 1e-11 * np.abs(w).max(0)[None, :]).all()


def test_non_positive_mass_fractions_are_absent_species():
    """Reading Q9 (PAPER.md:56 presumes C > 0): Y_k <= 0 is an absent
    species.  A small negative mass fraction gives exactly what Y_k = 0 gives, in W_mix, M, cp
    and the rates -- so the result does not depend on the size of the undershoot."""
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    om = oracle.OracleMechanism(mech)
    T, P, Y = ckgen.states(cfg, N=64)
    Y0, Yn = Y.copy(), Y.copy()
    Y0[2, :32] = 0.0
    Yn[2, :32] = -1e-9
    Y0[6, 16:48] = 0.0
    Yn[6, 16:48] = -3e-4
    w0, d0, _ = oracle.source_terms(om, T, P, Y0)
    wn, dn, _ = oracle.source_terms(om, T, P, Yn)
    assert np.array_equal(w0, wn) and np.array_equal(d0, dn)
    assert np.isfinite(w0).all() and np.isfinite(d0).all()


# ---------------------------------------------------------------------------------------------
# The 40-digit arbiter of DESIGN.md reading Q19 (helpers.mp_source_terms: mpmath, the paper's product
# form in the oracle's order of steps, no code shared with the oracle or with the log-matrix form).

@pytest.mark.parametrize("cfg_name,n", [("tiny_1k", 6), ("mid_1m", 3), ("large_256k", 1)])
def test_oracle_against_the_40_digit_product_form(cfg_name, n):
    """On ordinary cells the fp64 oracle is within 1 % of the north_star tolerance of the 40-digit value
    (every reaction type of the generated mechanisms is in these: third bodies, Troe falloff)."""
    from helpers import mp_source_terms
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=n)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    for i in range(n):
        w, d = mp_source_terms(mech, T[i], P[i], Y[:, i])
        w = np.array([float(x) for x in w])
        rw, rt = parity_violations(wr[:, i:i + 1], dr[i:i + 1], w[:, None], np.array([float(d)]))
        assert rw <= 1e-2 and rt <= 1e-2, (cfg_name, i, rw, rt)


def test_reading_q19_the_fp64_oracle_itself_breaks_the_dTdt_bound_where_the_energy_sum_cancels():
    """Cell 96243 of config 4 (S=111/R=784, 2^18 cells) has the most cancelling energy sum of the batch,
    kappa = sum|h_k wdot_k| / |sum h_k wdot_k| = 7.4e4.  There the fp64 oracle is 1.6e-10 (relative) away
    from the 40-digit value of dT/dt: more than the north_star's 1e-10, which is why a cell like this one is
    decided on the sum's own scale, (1e-10 + 1e-14 kappa) |dT/dt| -- and the oracle is well inside that.
    Its wdot, which does not cancel, is within 1 % of the tolerance."""
    from helpers import energy_kappa, mp_source_terms
    cfg = ckgen.CONFIGS["large_256k"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg)
    i = 96243
    Tc, Pc, Yc = T[i:i + 1], P[i:i + 1], np.ascontiguousarray(Y[:, i:i + 1])
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), Tc, Pc, Yc)
    kappa = float(energy_kappa(mech, Tc, wr)[0])
    assert 7e4 < kappa < 8e4
    w, d = mp_source_terms(mech, Tc[0], Pc[0], Yc[:, 0])
    rel = abs(dr[0] - float(d)) / abs(float(d))
    assert 1e-10 < rel < 0.5 * (1e-10 + 1e-14 * kappa), rel
    w = np.array([float(x) for x in w])
    rw, _ = parity_violations(wr, dr, w[:, None], dr)
    assert rw <= 1e-2
