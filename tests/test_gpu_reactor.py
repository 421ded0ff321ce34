"""ck_rk4_integrate (explicit RK4 constant-pressure reactor, BASELINE.json configs[4])
against oracle/reactor.py, through the C ABI.

Trajectory parity is checked on tamed mechanisms (tests/helpers.py: tame) whose time
scales the step resolves; on the configuration's own synthetic mechanism, whose rate
constants put dt = 1e-9 s far outside explicit stability (reading Q14), parity is
stage-wise: ck_source_terms against the oracle on the states the integrator reaches.
"""
import numpy as np
import pytest

import ckgen
import oracle
from oracle import reactor
from helpers import parity_violations, tame

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ck():
    import paper_2008_08483_b200 as ck
    assert torch.cuda.is_available()
    return ck


@pytest.fixture(autouse=True, params=["fused", "separate"])
def stage_variant(request, monkeypatch):
    """Every test runs with the RK stage update fused into the specialised source-term kernel's
    epilogue (the default) and with the separate stage kernels (CK_RK4_FUSED=0, also what the
    generic kernel uses)."""
    monkeypatch.setenv("CK_RK4_FUSED", "1" if request.param == "fused" else "0")
    return request.param


def to_dev(*arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0") for a in arrays]


@pytest.mark.parametrize("use_graph", [False, True])
@pytest.mark.parametrize("cfg_name,N,steps", [("tiny_1k", 1000, 25), ("mid_rk4", 600, 6), ("mid_rk4", 333, 2)])
def test_trajectory_parity_on_tamed_mechanism(ck, cfg_name, N, steps, use_graph):
    cfg = ckgen.CONFIGS[cfg_name]
    mech = tame(ckgen.mechanism(cfg.mech))
    T, P, Y = ckgen.states(cfg, N=N)
    dt = 1e-9
    Tr, Yr = reactor.integrate(oracle.OracleMechanism(mech), mech.mol_weight, T, P, Y, dt, steps)
    assert np.abs(Yr - Y).max() > 1e-7 and np.abs(Tr - T).max() > 1e-4      # the state moved
    Td, Pd, Yd = to_dev(T, P, Y)
    with ck.Mechanism(mech) as gm:
        gm.rk4_integrate(Td, Pd, Yd, dt, steps, use_graph=use_graph,
                         stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    # the increments are what the integrator computes: compare them to 1e-9 relative
    dT, dTr = Td.cpu().numpy() - T, Tr - T
    dY, dYr = Yd.cpu().numpy() - Y, Yr - Y
    assert np.abs(dT - dTr).max() <= 1e-9 * np.abs(dTr).max() + 1e-13 * T.max()
    assert (np.abs(dY - dYr) <= 1e-9 * np.abs(dYr).max(0, keepdims=True) + 4e-16).all()
    assert np.abs(Yd.cpu().numpy().sum(0) - 1.0).max() <= 1e-14


def test_graph_and_plain_launches_agree_bitwise_and_steps_compose(ck):
    cfg = ckgen.CONFIGS["mid_rk4"]
    mech = tame(ckgen.mechanism(cfg.mech))
    T, P, Y = ckgen.states(cfg, N=2048)
    st = torch.cuda.current_stream().cuda_stream
    with ck.Mechanism(mech) as gm:
        Ta, Pa, Ya = to_dev(T, P, Y)
        gm.rk4_integrate(Ta, Pa, Ya, 1e-9, 5, use_graph=False, stream=st)
        Tb, Pb, Yb = to_dev(T, P, Y)
        gm.rk4_integrate(Tb, Pb, Yb, 1e-9, 2, use_graph=True, stream=st)
        gm.rk4_integrate(Tb, Pb, Yb, 1e-9, 3, use_graph=True, stream=st)     # cached graph
        torch.cuda.synchronize()
        assert torch.equal(Ta, Tb) and torch.equal(Ya, Yb)
        gm.rk4_integrate(Tb, Pb, Yb, 1e-9, 0, stream=st)                      # no-op
        with pytest.raises(ck.CkError):
            gm.rk4_integrate(Tb, Pb, Yb, -1.0, 1, stream=st)


def test_config5_stagewise_parity_on_the_synthetic_mechanism(ck):
    """BASELINE.json configs[4] as written (S=53/R=325, dt = 1e-9 s, T0 ~ U[1100, 1500] K):
    the integrator must stay finite and on valid states, and the source term must match the
    oracle on the states it reaches (sample of 64 cells after 1, 10 and 100 steps)."""
    cfg = ckgen.CONFIGS["mid_rk4"]
    mech = ckgen.mechanism(cfg.mech)
    om = oracle.OracleMechanism(mech)
    N = 4096
    T, P, Y = ckgen.states(cfg, N=N)
    Td, Pd, Yd = to_dev(T, P, Y)
    st = torch.cuda.current_stream().cuda_stream
    w = torch.empty((mech.n_species, N), dtype=torch.float64, device="cuda:0")
    d = torch.empty(N, dtype=torch.float64, device="cuda:0")
    idx = np.random.default_rng(5).choice(N, 64, replace=False)
    with ck.Mechanism(mech) as gm:
        # one step against the oracle's step: the projection decides most of the result here
        (T1, Y1) = reactor.rk4_step(om, mech.mol_weight, T[idx], P[idx], np.ascontiguousarray(Y[:, idx]), 1e-9)
        done = 0
        for upto in (1, 10, 100):
            gm.rk4_integrate(Td, Pd, Yd, 1e-9, upto - done, stream=st)
            done = upto
            gm.source_terms(Td, Pd, Yd, w, d, stream=st)
            torch.cuda.synchronize()
            Th, Yh = Td.cpu().numpy(), Yd.cpu().numpy()
            assert np.isfinite(Th).all() and np.isfinite(Yh).all()
            assert Th.min() >= 250.0 and Th.max() <= 5000.0 and Yh.min() >= 0.0
            assert np.abs(Yh.sum(0) - 1.0).max() <= 1e-14
            if upto == 1:
                assert np.abs(Th[idx] - T1).max() <= 1e-9 * 5000.0
                assert np.abs(Yh[:, idx] - Y1).max() <= 1e-9
            wr, dr, _ = oracle.source_terms(om, Th[idx], P[idx], np.ascontiguousarray(Yh[:, idx]))
            rw, rt = parity_violations(w[:, idx].cpu().numpy(), d[idx].cpu().numpy(), wr, dr)
            assert rw <= 1.0 and rt <= 1.0, (upto, rw, rt)


def test_config5_as_written_65536_cells_1000_steps(ck):
    """BASELINE.json configs[4] at its full size (65 536 cells, 1000 steps of dt = 1e-9 s; PAPER.md:183-185,
    SURVEY reading Q14): after 1, 10, 100 and 1000 steps every state is finite and valid, and the source
    term of EVERY cell of the batch -- the cells the projection has clamped (T at 250 or 5000 K, a Y at
    exactly 0) included, they are counted and printed -- matches the oracle evaluated on the same state.
    dT/dt of cells whose energy sum cancels is decided as everywhere else (reading Q19)."""
    from helpers import dTdt_conditioned_violations, mp_dTdt
    cfg = ckgen.CONFIGS["mid_rk4"]
    mech = ckgen.mechanism(cfg.mech)
    om = oracle.OracleMechanism(mech)
    N = cfg.N
    assert N == 65536
    T, P, Y = ckgen.states(cfg)
    Td, Pd, Yd = to_dev(T, P, Y)
    st = torch.cuda.current_stream().cuda_stream
    w = torch.empty((mech.n_species, N), dtype=torch.float64, device="cuda:0")
    d = torch.empty(N, dtype=torch.float64, device="cuda:0")
    with ck.Mechanism(mech) as gm:
        done = 0
        for upto in (1, 10, 100, 1000):
            gm.rk4_integrate(Td, Pd, Yd, 1e-9, upto - done, stream=st)
            done = upto
            gm.source_terms(Td, Pd, Yd, w, d, stream=st)
            torch.cuda.synchronize()
            Th, Yh = Td.cpu().numpy(), Yd.cpu().numpy()
            assert np.isfinite(Th).all() and np.isfinite(Yh).all()
            assert Th.min() >= 250.0 and Th.max() <= 5000.0 and Yh.min() >= 0.0
            assert np.abs(Yh.sum(0) - 1.0).max() <= 1e-14
            clamped_T = (Th == 250.0) | (Th == 5000.0)
            clamped_Y = (Yh == 0.0).any(0)
            wr, dr, _ = oracle.source_terms(om, Th, P, Yh)
            wg, dg = w.cpu().numpy(), d.cpu().numpy()
            rw, rt = parity_violations(wg, dg, wr, dr)
            print("step %d: %d cells with T at a bound, %d with a species at exactly 0; worst wdot err/tol %.3g, "
                  "worst dT/dt err/tol %.3g" % (upto, clamped_T.sum(), clamped_Y.sum(), rw, rt))
            assert rw <= 1.0, (upto, rw)
            if rt > 1.0:
                over, kappa, ratio = dTdt_conditioned_violations(mech, Th, dg, wr, dr)
                assert over.size <= max(1, N // 20000), (upto, over.size)
                exact = mp_dTdt(mech, Th[over], P[over], Yh[:, over])      # 40 digits, the oracle's product form
                e_gpu = np.abs((dg[over] - exact) / exact).astype(float)
                print("step %d: %d cells over the north_star dT/dt bound by cancellation, kappa %.3g .. %.3g, "
                      "err / Q19 bound %.3g" % (upto, over.size, kappa.min(), kappa.max(), ratio.max()))
                assert kappa.min() > 1e3 and ratio.max() <= 1.0, (upto, kappa.min(), ratio.max())
                assert (e_gpu <= 1e-10 + 1e-14 * kappa).all()


def test_large_mechanism_one_step(ck):
    """S=111: cold accumulators and the species permutation through the fused stage epilogue."""
    cfg = ckgen.CONFIGS["large_256k"]
    mech = tame(ckgen.mechanism(cfg.mech))
    T, P, Y = ckgen.states(cfg, N=300)
    Tr, Yr = reactor.integrate(oracle.OracleMechanism(mech), mech.mol_weight, T, P, Y, 1e-9, 2)
    Td, Pd, Yd = to_dev(T, P, Y)
    with ck.Mechanism(mech) as gm:
        gm.rk4_integrate(Td, Pd, Yd, 1e-9, 2, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    dY, dYr = Yd.cpu().numpy() - Y, Yr - Y
    assert np.abs(dYr).max() > 1e-8
    assert (np.abs(dY - dYr) <= 1e-9 * np.abs(dYr).max(0, keepdims=True) + 4e-16).all()
    assert np.abs((Td.cpu().numpy() - T) - (Tr - T)).max() <= 1e-9 * np.abs(Tr - T).max() + 1e-13 * T.max()
