"""The all-DMMA small-mechanism kernel (CK_JIT_NU=dmma; csrc/ck_nu_kernel.cuh): Eq. 4's two
log-rate contractions, M = C E and Eq. 2 as dense DMMA.8x8x4 products, the
rate layers in the tensor fragment layout.  Same tolerance as the product's sparse kernel: the
north_star's, against the oracle."""
import dataclasses

import numpy as np
import pytest

import ckgen
import oracle
from helpers import parity_violations

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ck():
    import paper_2008_08483_b200 as ck
    assert torch.cuda.is_available()
    return ck


@pytest.fixture(autouse=True)
def nu_dmma(monkeypatch):
    monkeypatch.setenv("CK_JIT_NU", "dmma")


def check(ck, mech, T, P, Y, label):
    dev = torch.device("cuda:0")
    N = T.shape[0]
    with ck.Mechanism(mech) as gm:
        assert gm.info("all_dmma") == 1
        Td, Pd, Yd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (T, P, Y))
        w = torch.full((mech.n_species, N), float("nan"), dtype=torch.float64, device=dev)
        d = torch.full((N,), float("nan"), dtype=torch.float64, device=dev)
        gm.source_terms(Td, Pd, Yd, w, d, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        w2 = torch.empty_like(w)
        d2 = torch.empty_like(d)
        gm.source_terms(Td, Pd, Yd, w2, d2, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert torch.equal(w, w2) and torch.equal(d, d2)             # deterministic run to run
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    rw, rt = parity_violations(w.cpu().numpy(), d.cpu().numpy(), wr, dr)
    print("%s: worst wdot err/tol %.3g, dT/dt err/tol %.3g" % (label, rw, rt))
    assert rw <= 1.0 and rt <= 1.0, (label, rw, rt)


@pytest.mark.parametrize("N", [1, 31, 32, 33, 1024, 12289, 200001])
def test_parity_on_the_tiny_config(ck, N):
    cfg = ckgen.CONFIGS["tiny_1k"]
    check(ck, ckgen.mechanism(cfg.mech), *ckgen.states(cfg, N=N), label="all-DMMA N=%d" % N)


def test_every_reaction_on_its_own_and_both_temperature_ranges(ck):
    cfg = dataclasses.replace(ckgen.CONFIGS["tiny_1k"], T_range=(400.0, 2800.0))
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=200)
    T[:4] = [1000.0, np.nextafter(1000.0, 2000.0), 999.0, 1001.0]
    for j in range(mech.n_reactions):
        check(ck, mech.subset([j]), T, P, Y, "all-DMMA reaction %d (type %d)" % (j, mech.rxn_type[j]))


def test_irreversible_lindemann_real_nu_absent_species_distinct_T_mid(ck):
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    rev = mech.reversible.copy()
    rev[::3] = 0
    typ = mech.rxn_type.copy()
    typ[np.flatnonzero(typ == 3)[:1]] = 2                 # one Troe -> Lindemann
    nu_r = mech.nu_reac.copy()
    nu_r[int(np.flatnonzero(nu_r[:, 1])[0]), 1] = 1.5
    troe = mech.troe.copy()
    troe[np.flatnonzero(mech.rxn_type == 3)[-1], 3] = np.inf      # 3-parameter Troe
    rng = np.random.default_rng(3)
    T_mid = rng.choice([800.0, 1000.0, 1400.0, 2000.0], size=mech.n_species)
    m2 = dataclasses.replace(mech, reversible=rev, rxn_type=typ, nu_reac=nu_r, troe=troe, T_mid=T_mid)
    T, P, Y = ckgen.states(dataclasses.replace(cfg, T_range=(500.0, 2600.0)), N=700)
    Y = Y.copy()
    Y[1, :64] = 0.0
    Y[3, 32:96] = -1e-9
    Y[5, 200:260] = 1e-300
    check(ck, m2, T, P, Y, "all-DMMA variants")


def test_refused_where_it_does_not_apply(ck):
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(ckgen.mechanism(ckgen.MECH_MID))
    assert e.value.status == 4
