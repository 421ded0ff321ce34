"""The reduced-precision variants of the rate layers (PAPER.md:277:
"adapting the ANN-based interpretation to single or half-precision environments") against the
fp64 oracle: ck_mech_desc.precision = CK_PREC_MIXED (exp mantissas from the fp32 special-function
unit) and CK_PREC_F32_RATES (ln C, gathers, Arrhenius and equilibrium layers in fp32 as well).
State, results, M = C E and the contraction of Eq. 2 stay fp64 in both, so no rate overflows.

These are NOT held to the north_star tolerance (that is the fp64 product's); the tests assert the
error bounds DESIGN.md section 15 derives from the arithmetic, measured the way the north_star
measures wdot -- relative to max_k |wdot_k| of the cell -- and, for dT/dt, relative to the scale
sum_k |h_k wdot_k| / (rho cp) of the energy sum (its terms cancel; reading Q19)."""
import dataclasses

import numpy as np
import pytest

import ckgen
import oracle
from helpers import energy_kappa, tame

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

# error bounds, per cell: (wdot relative to max_k|wdot_k|, dT/dt relative to the energy sum's scale)
BOUND = {1: (4e-6, 4e-6), 2: (5e-4, 5e-4)}


@pytest.fixture(scope="module")
def ck():
    import paper_2008_08483_b200 as ck
    assert torch.cuda.is_available()
    return ck


def run(ck, mech, T, P, Y, precision):
    dev = torch.device("cuda:0")
    N = T.shape[0]
    with ck.Mechanism(mech, precision=precision) as gm:
        assert gm.info("jit") == 1 and gm.info("precision") == precision
        Td, Pd, Yd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (T, P, Y))
        w = torch.full((mech.n_species, N), float("nan"), dtype=torch.float64, device=dev)
        d = torch.full((N,), float("nan"), dtype=torch.float64, device=dev)
        gm.source_terms(Td, Pd, Yd, w, d, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    return w.cpu().numpy(), d.cpu().numpy()


def errors(mech, T, w, d, wr, dr):
    """Per cell: max_k |d wdot_k| / max_k |wdot_k| and |d dT/dt| / (kappa |dT/dt|)."""
    e_w = np.abs(w - wr).max(0) / np.abs(wr).max(0)
    e_t = np.abs(d - dr) / (energy_kappa(mech, T, wr) * np.abs(dr))
    return e_w, e_t


@pytest.mark.parametrize("precision", [1, 2])
@pytest.mark.parametrize("cfg_name,N", [("tiny_1k", 1024), ("mid_1m", 3000), ("large_256k", 1100), ("mid_rk4", 777)])
def test_reduced_precision_error_on_the_configs_own_states(ck, cfg_name, N, precision):
    """Rates up to e^250 on these states: an fp32 *result* would overflow in every cell, the
    exponent-split variants do not; their error stays inside the derived bound on every cell."""
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    w, d = run(ck, mech, T, P, Y, precision)
    assert np.isfinite(w).all() and np.isfinite(d).all()
    e_w, e_t = errors(mech, T, w, d, wr, dr)
    print("%s precision %d: wdot err/max median %.2e max %.2e; dT/dt err/scale median %.2e max %.2e"
          % (cfg_name, precision, np.median(e_w), e_w.max(), np.median(e_t), e_t.max()))
    assert e_w.max() <= BOUND[precision][0] and e_t.max() <= BOUND[precision][1]
    # ... and the variant really is less precise than the product (it is not silently fp64)
    assert e_w.max() > 1e-9
    # conservation holds to fp64 rounding in every variant: Eq. 2 is contracted in fp64
    terms = mech.mol_weight[:, None] * w
    assert (np.abs(terms.sum(0)) <= 1e-11 * np.abs(terms).sum(0)).all()


@pytest.mark.parametrize("precision", [1, 2])
@pytest.mark.parametrize("spec", [ckgen.MECH_TINY, ckgen.MECH_MID, ckgen.MECH_LARGE], ids=lambda s: s.name)
def test_reduced_precision_error_on_tamed_mechanisms(ck, spec, precision):
    """Mechanisms with physically mild kinetics (|ln Kc| ~ 10, rates that fit fp32): the same bounds."""
    mech = tame(ckgen.mechanism(spec))
    cfg = {9: "tiny_1k", 53: "mid_1m", 111: "large_256k"}[spec.S]
    T, P, Y = ckgen.states(ckgen.CONFIGS[cfg], N=900)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    w, d = run(ck, mech, T, P, Y, precision)
    e_w, e_t = errors(mech, T, w, d, wr, dr)
    print("tamed %s precision %d: wdot err/max median %.2e max %.2e; dT/dt err/scale median %.2e max %.2e"
          % (spec.name, precision, np.median(e_w), e_w.max(), np.median(e_t), e_t.max()))
    assert e_w.max() <= BOUND[precision][0] and e_t.max() <= BOUND[precision][1]


def test_precision_zero_is_the_default_and_bad_values_are_rejected(ck, monkeypatch):
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=500)
    w0, d0 = run(ck, mech, T, P, Y, 0)
    with ck.Mechanism(mech) as gm:
        assert gm.info("precision") == 0
    for bad in (-1, 3):
        with pytest.raises(ck.CkError) as e:
            ck.Mechanism(mech, precision=bad)
        assert e.value.status == 1
    # fall-back kernel has no reduced-precision variant: refused, never silently fp64
    monkeypatch.setenv("CK_KERNEL", "generic")
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(mech, precision=1)
    assert e.value.status == 4
    monkeypatch.delenv("CK_KERNEL")
    # a ragged batch through the fp32-rates variant with cold accumulators and the pair shape
    for env in ({"CK_JIT_SREG": "3"}, {"CK_JIT_PAIR": "1"}):
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T[:77], P[:77], np.ascontiguousarray(Y[:, :77]))
        w, d = run(ck, mech, T[:77], P[:77], np.ascontiguousarray(Y[:, :77]), 2)
        e_w, e_t = errors(mech, T[:77], w, d, wr, dr)
        assert e_w.max() <= BOUND[2][0] and e_t.max() <= BOUND[2][1]
        for k in env:
            monkeypatch.delenv(k)
    assert np.isfinite(w0).all() and np.isfinite(d0).all()
