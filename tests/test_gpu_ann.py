"""The approximate-ANN log Kc layer (Eq. 12-14) on the device against the
oracle's, through the C ABI, under the north_star tolerance."""
import dataclasses

import numpy as np
import pytest

import ckgen
import oracle
from helpers import parity_violations, exact_layer_as_ann

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ck():
    import paper_2008_08483_b200 as ck
    assert torch.cuda.is_available()
    return ck


def gpu_run(ck, mech, ann, T, P, Y):
    dev = torch.device("cuda:0")
    N = T.shape[0]
    Td, Pd, Yd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (T, P, Y))
    w = torch.full((mech.n_species, N), float("nan"), dtype=torch.float64, device=dev)
    d = torch.full((N,), float("nan"), dtype=torch.float64, device=dev)
    with ck.Mechanism(mech, kc_ann=ann) as gm:
        assert gm.info("jit") == 1
        gm.source_terms(Td, Pd, Yd, w, d, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    return w.cpu().numpy(), d.cpu().numpy()


# LF 1/8 and 2/8, HF 3/32, both activations, both architectures, odd N_H
ARCHS = [(1, 1, 8, ckgen.ELU), (1, 2, 8, ckgen.ELU), (1, 3, 32, ckgen.ELU), (1, 2, 8, ckgen.RELU),
         (6, 2, 8, ckgen.RELU), (6, 1, 5, ckgen.ELU), (1, 3, 48, ckgen.ELU)]


@pytest.mark.parametrize("n_in,n_layers,n_hidden,activation", ARCHS)
@pytest.mark.parametrize("cfg_name,N", [("tiny_1k", 1024), ("mid_1m", 1537)])
def test_parity_with_random_weights(ck, cfg_name, N, n_in, n_layers, n_hidden, activation):
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    ann = ckgen.random_kc_ann(mech.n_reactions, n_layers, n_hidden, n_in=n_in, activation=activation,
                              seed=100 + n_hidden, T_range=cfg.T_range)
    T, P, Y = ckgen.states(cfg, N=N)
    w, d = gpu_run(ck, mech, ann, T, P, Y)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech, kc_ann=ann), T, P, Y)
    rw, rt = parity_violations(w, d, wr, dr)
    assert rw <= 1.0 and rt <= 1.0, (rw, rt)
    # the network really is in the path: the exact layer gives something else
    w0, _, _ = oracle.source_terms(oracle.OracleMechanism(mech), T[:8], P[:8], np.ascontiguousarray(Y[:, :8]))
    assert np.abs(w0 - wr[:, :8]).max() > 1e-6 * np.abs(w0).max()


def test_large_mechanism_with_cold_accumulators_and_ring(ck):
    cfg = ckgen.CONFIGS["large_256k"]
    mech = ckgen.mechanism(cfg.mech)
    ann = ckgen.random_kc_ann(mech.n_reactions, 2, 8, seed=5, T_range=cfg.T_range)
    T, P, Y = ckgen.states(cfg, N=600)
    w, d = gpu_run(ck, mech, ann, T, P, Y)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech, kc_ann=ann), T, P, Y)
    rw, rt = parity_violations(w, d, wr, dr)
    assert rw <= 1.0 and rt <= 1.0, (rw, rt)


def test_network_built_to_be_the_exact_layer_matches_the_exact_kernel(ck):
    """Two different device code paths (folded Gibbs polynomial vs hidden layers + folded output
    layer) of the same function."""
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    mech = dataclasses.replace(mech, nasa_lo=mech.nasa_hi.copy())
    ann = exact_layer_as_ann(mech, n_layers=2, activation=ckgen.ELU, seed=1)
    T, P, Y = ckgen.states(cfg, N=512)
    w1, d1 = gpu_run(ck, mech, ann, T, P, Y)
    w0, d0 = gpu_run(ck, mech, None, T, P, Y)
    assert (np.abs(w1 - w0) <= 1e-10 * np.abs(w0).max(0, keepdims=True)).all()
    assert (np.abs(d1 - d0) <= 1e-8 * np.abs(d0) + 1e-12).all()


def test_errors(ck, monkeypatch):
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    ann = ckgen.random_kc_ann(mech.n_reactions, 2, 8)
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(mech, kc_ann=dataclasses.replace(ann, in_std=np.array([0.0])))
    assert e.value.status == 1
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(mech, kc_ann=dataclasses.replace(ann, activation=7))
    assert e.value.status == 1
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(mech, kc_ann=ckgen.random_kc_ann(mech.n_reactions, 3, 64))     # 64 KB of weights
    assert e.value.status == 4
    monkeypatch.setenv("CK_KERNEL", "generic")
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(mech, kc_ann=ann)
    assert e.value.status == 4
