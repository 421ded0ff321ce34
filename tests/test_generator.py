"""The seeded input generator: deterministic, element balanced, shaped as BASELINE.json's
configs say.  It holds no kinetics, so there is nothing to compare with the oracle here."""
import numpy as np
import pytest

import ckgen


@pytest.mark.parametrize("spec", [ckgen.MECH_TINY, ckgen.MECH_MID], ids=lambda s: s.name)
def test_mechanism_shape_balance_and_determinism(spec):
    m = ckgen.mechanism(spec)
    again = ckgen.generate_mechanism(spec.S, spec.R, spec.elements, spec.seed,
                                     spec.frac_three_body, spec.frac_falloff)
    for f in ("nu_reac", "nu_prod", "ln_A", "b", "Ea_over_R", "nasa_lo", "nasa_hi", "eff", "troe"):
        assert np.array_equal(getattr(m, f), getattr(again, f)), f
    assert m.nu_reac.shape == (spec.S, spec.R)
    nu = m.nu_prod - m.nu_reac
    assert np.abs(m.elem_count.T @ nu).max() == 0                       # element balanced
    assert ((m.nu_reac > 0) & (m.nu_prod > 0)).sum() == 0               # disjoint sides
    n_r, n_p = (m.nu_reac > 0).sum(0), (m.nu_prod > 0).sum(0)
    assert n_r.min() >= 1 and n_r.max() <= 3 and n_p.min() >= 1 and n_p.max() <= 3
    assert set(np.unique(m.nu_reac)) <= {0.0, 1.0, 2.0}
    cols = {(tuple(m.nu_reac[:, j]), tuple(m.nu_prod[:, j])) for j in range(spec.R)}
    assert len(cols) == spec.R                                          # distinct reactions
    n_tb, n_fo = ckgen.type_counts(spec.R, spec.frac_three_body, spec.frac_falloff)
    assert (m.rxn_type == 1).sum() == n_tb and (m.rxn_type == 3).sum() == n_fo
    assert np.log(1e6) <= m.ln_A.min() and m.ln_A.max() <= np.log(1e14)
    assert -2 <= m.b.min() and m.b.max() <= 2
    assert 0 <= m.Ea_over_R.min() and m.Ea_over_R.max() <= 2e5 / 8.31446261815324
    used = m.rxn_type != 0
    assert m.eff[:, used].min() >= 0.5 and m.eff[:, used].max() <= 5.0
    assert (m.eff[:, ~used] == 1).all()
    tro = m.troe[m.rxn_type == 3]
    assert 0.3 <= tro[:, 0].min() and tro[:, 0].max() <= 0.9
    assert 1e2 <= tro[:, 1:].min() and tro[:, 1:].max() <= 1e4
    aw = {"H": 1.008, "C": 12.011, "N": 14.007, "O": 15.999, "Ar": 39.95}
    W = m.elem_count @ np.array([aw[e] for e in m.elements])
    assert np.allclose(W, m.mol_weight)


def test_nasa_cp_range_and_continuity():
    m = ckgen.mechanism(ckgen.MECH_MID)
    P = np.polynomial.polynomial
    for k in range(m.n_species):
        lo, hi = m.nasa_lo[k], m.nasa_hi[k]
        cl = P.polyval(np.linspace(300, 1000, 50), lo[:5])
        ch = P.polyval(np.linspace(1000, 3500, 50), hi[:5])
        assert 2.5 - 1e-9 <= min(cl.min(), ch.min()) and max(cl.max(), ch.max()) <= 10 + 1e-9
        assert abs(P.polyval(1000.0, lo[:5]) - P.polyval(1000.0, hi[:5])) < 1e-9
        assert (np.abs(lo[:5]) > 0).all() and (np.abs(hi[:5]) > 0).all()


def test_states_distribution_layout_and_determinism():
    cfg = ckgen.CONFIGS["mid_1m"]
    T, P, Y = ckgen.states(cfg, N=4096)
    T2, P2, Y2 = ckgen.states(cfg, N=4096)
    assert np.array_equal(T, T2) and np.array_equal(P, P2) and np.array_equal(Y, Y2)
    assert Y.shape == (53, 4096) and Y.flags.c_contiguous and Y.dtype == np.float64
    assert 900 <= T.min() and T.max() <= 2800
    assert 101325 <= P.min() and P.max() <= 40 * 101325
    assert np.allclose(Y.sum(0), 1.0, atol=1e-14) and Y.min() >= 0.99e-20


@pytest.mark.parametrize("cfg_name", ["tiny_1k", "tiny_1m", "mid_1m", "large_256k", "mid_rk4"])
def test_log_rates_stay_inside_fp64_exp_range(cfg_name):
    """SURVEY.md section 8(c) tolerance notes / 8(d) NASA-7 bullet: the generator must keep
    max |ln q| < 650 (fp64 exp overflows at 709.8) on the configs' own states, or Eq. 4's exp
    activations would overflow in any implementation.  4096 states per config,
    the arguments of the two exps from the matrix-form restatement in tests/helpers.py."""
    from helpers import paper_matrix_form
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=4096)
    lqf, lqr = paper_matrix_form(mech, T, P, Y, return_log_rates=True)
    assert np.isfinite(lqf).all() and np.isfinite(lqr).all()
    worst = max(np.abs(lqf).max(), np.abs(lqr).max())
    print("%s: ln q_f in [%.1f, %.1f], ln q_r in [%.1f, %.1f]" % (cfg_name, lqf.min(), lqf.max(), lqr.min(), lqr.max()))
    assert worst < 650.0, worst


def test_config_table_matches_baseline_json():
    c = ckgen.CONFIGS
    assert (c["tiny_1k"].mech.S, c["tiny_1k"].mech.R, c["tiny_1k"].N) == (9, 21, 1024)
    assert c["tiny_1m"].N == 1 << 20
    assert (c["mid_1m"].mech.S, c["mid_1m"].mech.R, c["mid_1m"].N) == (53, 325, 1 << 20)
    assert (c["large_256k"].mech.S, c["large_256k"].mech.R, c["large_256k"].N) == (111, 784, 1 << 18)
    assert c["mid_rk4"].N == 65536 and c["mid_rk4"].T_range == (1100.0, 1500.0)
    assert ckgen.SWEEP_N == (256, 1024, 4096, 16384, 65536, 262144, 1048576, 4194304)
