"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element,
with the north_star tolerance:
   |d wdot_k| <= 1e-10 max_k|wdot_k| + 1e-12 |wdot_k|,  |d dT/dt| <= 1e-10 |dT/dt| + 1e-12 K/s.
"""
import dataclasses

import numpy as np
import pytest

import ckgen
import oracle
from helpers import RU, dTdt_conditioned_violations, mp_dTdt, parity_violations

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ck():
    import paper_2008_08483_b200 as ck
    assert torch.cuda.is_available()
    return ck


@pytest.fixture(autouse=True, params=["auto", "generic"])
def kernel_variant(request, monkeypatch):
    """Every test runs twice: with the mechanism-specialised (NVRTC) kernel that
    ck_mech_create picks by default, and with the generic table-driven kernel."""
    monkeypatch.setenv("CK_KERNEL", request.param)
    return request.param


def test_variant_selection(ck, kernel_variant):
    for spec in (ckgen.MECH_TINY, ckgen.MECH_MID, ckgen.MECH_LARGE):
        with ck.Mechanism(ckgen.mechanism(spec)) as gm:
            assert gm.info("jit") == (1 if kernel_variant == "auto" else 0)
            if kernel_variant == "auto":
                # S=111 does not fit 2 registers per species: hot/cold accumulator split
                assert (gm.info("s_reg") < spec.S) == (spec is ckgen.MECH_LARGE)
                # ... and that shape runs two threads per cell
                assert gm.info("pair") == (1 if spec is ckgen.MECH_LARGE else 0)


@pytest.mark.parametrize("s_reg", [0, 7, 30])
def test_cold_accumulators_on_small_mechanisms(ck, monkeypatch, kernel_variant, s_reg):
    """The shared-memory (cold) accumulator path and the species permutation that comes with
    it, forced on mechanisms that would otherwise keep every accumulator in registers."""
    if kernel_variant != "auto":
        pytest.skip("specialised kernel only")
    monkeypatch.setenv("CK_JIT_SREG", str(s_reg))
    monkeypatch.setenv("CK_JIT_PAIR", "0")      # one thread per cell (the pair shape has its own test)
    for cfg_name, N in (("tiny_1k", 1024), ("mid_1m", 777)):
        cfg = ckgen.CONFIGS[cfg_name]
        mech = ckgen.mechanism(cfg.mech)
        with ck.Mechanism(mech) as gm:
            assert gm.info("jit") == 1 and gm.info("s_reg") == min(s_reg, mech.n_species)
        assert_parity(ck, mech, *ckgen.states(cfg, N=N), label="%s s_reg=%d" % (cfg_name, s_reg))


@pytest.mark.parametrize("s_reg", [None, 0, 3, 12])
def test_two_threads_per_cell_on_small_mechanisms(ck, monkeypatch, kernel_variant, s_reg):
    """The two-threads-per-cell shape of the specialised kernel (CK_PAIR: halves of a cell's pair
    take alternate reaction blocks and alternate species and exchange rates through shared
    memory), forced on mechanisms that would not need it, with all accumulators in registers
    and with some or all of them in the shared-memory (cold) columns; ragged batches so that
    partly filled and idle warp pairs occur."""
    if kernel_variant != "auto":
        pytest.skip("specialised kernel only")
    monkeypatch.setenv("CK_JIT_PAIR", "1")
    if s_reg is not None:
        monkeypatch.setenv("CK_JIT_SREG", str(s_reg))
    for cfg_name, N in (("tiny_1k", 1024), ("tiny_1k", 77), ("mid_1m", 777), ("mid_1m", 129)):
        cfg = ckgen.CONFIGS[cfg_name]
        mech = ckgen.mechanism(cfg.mech)
        with ck.Mechanism(mech) as gm:
            assert gm.info("jit") == 1 and gm.info("pair") == 1
        assert_parity(ck, mech, *ckgen.states(cfg, N=N), label="pair %s s_reg=%s N=%d" % (cfg_name, s_reg, N))


def gpu_run(ck, mech, T, P, Y, gm=None):
    """T, P, Y numpy -> (wdot[S,N], dTdt[N]) numpy via ck_source_terms on device buffers."""
    own = gm is None
    gm = gm or ck.Mechanism(mech)
    dev = torch.device("cuda:0")
    N = T.shape[0]
    Td = torch.from_numpy(np.ascontiguousarray(T)).to(dev)
    Pd = torch.from_numpy(np.ascontiguousarray(P)).to(dev)
    Yd = torch.from_numpy(np.ascontiguousarray(Y)).to(dev)
    w = torch.full((mech.n_species, N), float("nan"), dtype=torch.float64, device=dev)
    d = torch.full((N,), float("nan"), dtype=torch.float64, device=dev)
    gm.source_terms(Td, Pd, Yd, w, d, N=N, stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    if own:
        gm.close()
    return w.cpu().numpy(), d.cpu().numpy()


def assert_parity(ck, mech, T, P, Y, label=""):
    w, d = gpu_run(ck, mech, T, P, Y)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    rw, rt = parity_violations(w, d, wr, dr)
    assert rw <= 1.0, "%s wdot error is %.3g x tolerance" % (label, rw)
    if rt > 1.0:
        # report the conditioning of the energy sum rather than loosening the bound
        i = int(np.argmax(np.abs(d - dr) / (1e-10 * np.abs(dr) + 1e-12)))
        om = oracle.OracleMechanism(mech)
        det = oracle.cell_detail(om, T[i], P[i], Y[:, i])
        hw = det["h_RT"] * det["wdot"]
        kappa = np.abs(hw).sum() / max(abs(hw.sum()), 1e-300)
        raise AssertionError("%s dT/dt error is %.3g x tolerance at cell %d (kappa = %.3g)"
                             % (label, rt, i, kappa))
    return w, d, wr, dr


# ---------------------------------------------------------------- the five configs, small N

@pytest.mark.parametrize("cfg_name,N", [("tiny_1k", 1024), ("mid_1m", 2000), ("large_256k", 700),
                                        ("mid_rk4", 515)])
def test_config_parity_all_cells(ck, cfg_name, N):
    """Every cell, sizes spanning several 128-cell tiles and a ragged tail."""
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    assert_parity(ck, mech, T, P, Y, cfg_name)


def full_batch_parity(ck, mech, T, P, Y, label, variants=("auto", "generic"), host_chunks=()):
    """Every cell of a batch against the oracle (which runs once, in chunks of 65536 cells so that
    its memory stays bounded), for each kernel variant: finiteness, mass and element conservation
    on the device over all cells, then element by element under the north_star tolerance.
    host_chunks: also ck_source_terms_host with these CK_HOST_CHUNKS values, against the oracle.
    Returns the worst (wdot, dT/dt) error / tolerance over all variants."""
    import os
    N = T.shape[0]
    S = mech.n_species
    dev = torch.device("cuda:0")
    om = oracle.OracleMechanism(mech)
    wr = np.empty((S, N))
    dr = np.empty(N)
    for c0 in range(0, N, 65536):
        c1 = min(N, c0 + 65536)
        wr[:, c0:c1], dr[c0:c1], _ = oracle.source_terms(om, T[c0:c1], P[c0:c1], np.ascontiguousarray(Y[:, c0:c1]))
    assert np.isfinite(wr).all() and np.isfinite(dr).all()
    Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
    weights = [mech.mol_weight] + [mech.elem_count[:, e].astype(float) for e in range(mech.elem_count.shape[1])]
    worst_w = worst_t = 0.0
    saved = os.environ.get("CK_KERNEL")
    try:
        for variant in variants:
            os.environ["CK_KERNEL"] = variant
            with ck.Mechanism(mech) as gm:
                assert gm.info("jit") == (1 if variant == "auto" else 0)
                w = torch.full((S, N), float("nan"), dtype=torch.float64, device=dev)
                d = torch.full((N,), float("nan"), dtype=torch.float64, device=dev)
                gm.source_terms(Td, Pd, Yd, w, d, stream=torch.cuda.current_stream().cuda_stream)
                torch.cuda.synchronize()
                assert torch.isfinite(w).all() and torch.isfinite(d).all()
                for wt in weights:
                    terms = torch.from_numpy(wt).to(dev)[:, None] * w
                    assert (terms.sum(0).abs() <= 1e-11 * terms.abs().sum(0) + 1e-300).all()
                    del terms
                results = [("device", w.cpu().numpy(), d.cpu().numpy())]
                del w, d
                for chunks in (host_chunks if variant == "auto" else ()):
                    os.environ["CK_HOST_CHUNKS"] = str(chunks)      # (read by ck_mech_create)
                    try:
                        with ck.Mechanism(mech) as gh:
                            wh, dh = gh.source_terms_host(T, P, Y)
                    finally:
                        del os.environ["CK_HOST_CHUNKS"]
                    results.append(("host, %d chunks" % chunks, wh, dh))
            for what, wg, dg in results:
                rw, rt = parity_violations(wg, dg, wr, dr)
                print("%s [%s, %s]: N=%d all cells, worst wdot err/tol %.3g, worst dT/dt err/tol %.3g"
                      % (label, variant, what, N, rw, rt))
                assert rw <= 1.0, (label, variant, what, rw, rt)
                if rt > 1.0:
                    # Cells over the north_star bound on dT/dt ALONE: the energy sum cancels there
                    # (reading Q19).  They must be few, ill-conditioned (kappa > 1e3), inside
                    # the bound taken on the sum's own scale, and no farther from a 40-digit
                    # evaluation in the oracle's product form (helpers.mp_dTdt) than that bound allows (the fp64 oracle is itself off by ~1e-15 kappa).
                    over, kappa, ratio = dTdt_conditioned_violations(mech, T, dg, wr, dr)
                    # (few first: that also bounds the work of the long-double arbiter, which then takes
                    #  EVERY such cell, not a sample of them)
                    assert over.size <= max(1, N // 20000), (label, variant, what, over.size)
                    exact = mp_dTdt(mech, T[over], P[over], Y[:, over])      # 40 digits, the oracle's product form
                    e_gpu = np.abs((dg[over] - exact) / exact).astype(float)
                    e_orc = np.abs((dr[over] - exact) / exact).astype(float)
                    print("%s [%s, %s]: %d of %d cells over the north_star dT/dt bound, all by cancellation: "
                          "kappa %.3g .. %.3g, worst err / Q19 bound %.3g; against a 40-digit evaluation: GPU rel err "
                          "%.3g, fp64 oracle rel err %.3g (worst of all %d)"
                          % (label, variant, what, over.size, N, kappa.min(), kappa.max(), ratio.max(),
                             e_gpu.max(), e_orc.max(), e_gpu.size))
                    assert kappa.min() > 1e3 and ratio.max() <= 1.0, \
                        (label, variant, what, over.size, kappa.min(), ratio.max())
                    assert (e_gpu <= 1e-10 + 1e-14 * kappa).all()
                worst_w, worst_t = max(worst_w, rw), max(worst_t, rt)
    finally:
        if saved is None:
            os.environ.pop("CK_KERNEL", None)
        else:
            os.environ["CK_KERNEL"] = saved
    return worst_w, worst_t


@pytest.mark.parametrize("cfg_name", ["tiny_1m", "mid_1m", "large_256k"])
def test_full_size_parity_every_cell(ck, kernel_variant, cfg_name):
    """BASELINE.json's full sizes (configs 2-4: 2^20, 2^20, 2^18 cells) in the launch
    configuration bench.py times: EVERY cell against the oracle, both kernel variants, plus the
    pipelined host entry point with 1, 8 and 16 chunks (north_star: "matching the oracle ... on
    all five configs"; parity over all N cells of every config)."""
    if kernel_variant != "auto":
        pytest.skip("both variants are covered inside the test (the oracle runs once)")
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg)
    full_batch_parity(ck, mech, T, P, Y, cfg_name, host_chunks=(1, 8, 16))


@pytest.mark.parametrize("N", ckgen.SWEEP_N)
def test_sweep_sizes_parity_every_cell(ck, kernel_variant, N):
    """BASELINE.json configs[4], sweep part: N = 2^8, 2^10, ..., 2^22 cells at S=53/R=325 (the
    sizes bench.py --sweep times): every cell of every size against the
    oracle.  2^22 cells are 3.66 GB of state in and out, rows past 2^31 bytes."""
    if kernel_variant != "auto":
        pytest.skip("specialised kernel (the one the sweep times); the generic one runs at 2^8..2^16")
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    full_batch_parity(ck, mech, T, P, Y, "sweep N=2^%d" % (N.bit_length() - 1),
                      variants=("auto", "generic") if N <= 65536 else ("auto",))


# ---------------------------------------------------------------- every reaction on its own

@pytest.mark.parametrize("spec", [ckgen.MECH_TINY, ckgen.MECH_MID], ids=lambda s: s.name)
def test_single_reaction_mechanisms(ck, spec):
    """Each reaction as a mechanism of its own: with one reaction the north_star tolerance
    is a relative 1e-10 on that reaction's rate, so no reaction hides behind a larger one.
    Covers elementary, three-body and Troe records and both temperature ranges."""
    mech = ckgen.mechanism(spec)
    cfg = ckgen.CONFIGS["tiny_1k" if spec is ckgen.MECH_TINY else "mid_1m"]
    cfg = dataclasses.replace(cfg, T_range=(600.0, 2800.0))
    T, P, Y = ckgen.states(cfg, N=160)
    R = mech.n_reactions
    picks = range(R) if R <= 32 else np.unique(np.concatenate(
        [np.flatnonzero(mech.rxn_type == 3)[:6], np.flatnonzero(mech.rxn_type == 1)[:6],
         np.flatnonzero(mech.rxn_type == 0)[:12]]))
    for j in picks:
        assert_parity(ck, mech.subset([j]), T, P, Y, "%s reaction %d" % (spec.name, j))


# ---------------------------------------------------------------- edge cases

@pytest.mark.parametrize("N", [1, 31, 127, 128, 129, 257, 383, 384, 385, 769])
def test_ragged_sizes(ck, N):
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    assert_parity(ck, mech, T, P, Y, "N=%d" % N)


def test_empty_batch_is_a_noop(ck):
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    gm = ck.Mechanism(mech)
    ck.ck_source_terms(gm.handle, 0, 0, 0, 0, 0, 0)      # N == 0: pointers are not touched
    gm.close()


def test_temperature_at_below_and_across_T_mid(ck):
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(dataclasses.replace(cfg, T_range=(300.0, 1100.0)), N=300)
    T[:8] = 1000.0                                   # exactly T_mid: low range (reading Q4)
    T[8:16] = np.nextafter(1000.0, 2000.0)
    assert_parity(ck, mech, T, P, Y, "T around T_mid")


@pytest.mark.parametrize("cfg_name", ["tiny_1k", "mid_1m", "large_256k"])
def test_wide_temperature_and_pressure_range(ck, cfg_name):
    """The whole fitted temperature range of the NASA-7 data (300-3500 K, and beyond to 4500 K)
    and four decades of pressure, far outside the configs' own state distributions: both
    temperature ranges, rates from underflow to 1e+100 and beyond."""
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    N = 600
    _, _, Y = ckgen.states(cfg, N=N)
    rng = np.random.default_rng(99)
    T = rng.uniform(300.0, 4500.0, N)
    P = 10.0 ** rng.uniform(3.5, 7.5, N)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    ok = np.isfinite(wr).all(0) & np.isfinite(dr)          # (the oracle's product form overflows first)
    print("%s wide T, P: %d of %d cells dropped (the ORACLE is not finite there)" % (cfg_name, int((~ok).sum()), N))
    assert ok.mean() > 0.9
    assert_parity(ck, mech, T[ok], P[ok], np.ascontiguousarray(Y[:, ok]), "%s wide T, P" % cfg_name)


def test_distinct_T_mid_per_species(ck):
    """Several temperature ranges: the folded equilibrium layer keeps one coefficient row
    per range delimited by the distinct T_mid values."""
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    rng = np.random.default_rng(3)
    T_mid = rng.choice([800.0, 1000.0, 1400.0, 2000.0], size=mech.n_species)
    mech = dataclasses.replace(mech, T_mid=T_mid)
    T, P, Y = ckgen.states(dataclasses.replace(cfg, T_range=(500.0, 2600.0)), N=640)
    T[:4] = [800.0, 1000.0, 1400.0, 2000.0]
    assert_parity(ck, mech, T, P, Y, "distinct T_mid")


def test_absent_species_and_tiny_mass_fractions(ck):
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=256)
    Y = Y.copy()
    Y[1, :64] = 0.0
    Y[3, 32:96] = 0.0
    Y[5, 200:] = 1e-300
    Y /= Y.sum(0, keepdims=True)
    assert_parity(ck, mech, T, P, Y, "absent species")


def test_negative_mass_fractions(ck):
    """Y_k <= 0 is an absent species (reading Q9): the small negative mass fractions a caller's own
    integrator produces enter W_mix, cp, M = C E and C as 0 on the device as in the oracle --
    three-body and falloff rates would differ if M were built from the raw values."""
    for cfg_name in ("tiny_1k", "mid_1m"):
        cfg = ckgen.CONFIGS[cfg_name]
        mech = ckgen.mechanism(cfg.mech)
        T, P, Y = ckgen.states(cfg, N=300)
        Y = Y.copy()
        rng = np.random.default_rng(5)
        neg = rng.random(Y.shape) < 0.15
        Y[neg] = -10.0 ** rng.uniform(-14, -3, size=int(neg.sum()))
        Y[0, :8] = -0.0
        assert_parity(ck, mech, T, P, Y, "%s negative Y" % cfg_name)


def test_irreversible_lindemann_and_real_valued_nu(ck):
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    rev = mech.reversible.copy()
    rev[::3] = 0
    typ = mech.rxn_type.copy()
    typ[typ == 3] = 2                                   # Troe -> Lindemann
    nu_r = mech.nu_reac.copy()
    k = int(np.flatnonzero(nu_r[:, 1])[0])
    nu_r[k, 1] = 1.5
    mech2 = dataclasses.replace(mech, reversible=rev, rxn_type=typ, nu_reac=nu_r)
    T, P, Y = ckgen.states(cfg, N=200)
    assert_parity(ck, mech2, T, P, Y, "irreversible/lindemann/real nu")
    # 3-parameter Troe (T** = +INF)
    troe = mech.troe.copy()
    troe[:, 3] = np.inf
    assert_parity(ck, dataclasses.replace(mech, troe=troe), T, P, Y, "Troe 3-parameter")


def test_species_on_both_sides(ck):
    """A + B -> A + C style reactions: nu' and nu'' overlap, the net list is shorter."""
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    nu_r, nu_p = mech.nu_reac.copy(), mech.nu_prod.copy()
    free = int(np.flatnonzero((nu_r[:, 0] == 0) & (nu_p[:, 0] == 0))[0])
    nu_r[free, 0] += 1.0
    nu_p[free, 0] += 1.0
    assert_parity(ck, dataclasses.replace(mech, nu_reac=nu_r, nu_prod=nu_p),
                  *ckgen.states(cfg, N=130), label="catalyst species")


def test_detailed_balance_on_the_device(ck):
    """At a constructed equilibrium the net rates vanish to rounding:
    |wdot_k| <= 1e-10 sum_j |nu_kj| phi_j q_f,j."""
    mech = ckgen.mechanism(ckgen.MECH_MID)
    om = oracle.OracleMechanism(mech)
    S = mech.n_species
    Ts = np.array([800.0, 1500.0, 2600.0])
    Ps, Ys, bounds = [], [], []
    rng = np.random.default_rng(7)
    for T in Ts:
        g = oracle.cell_detail(om, T, 1e5, np.full(S, 1.0 / S))["g_RT"]
        lam = rng.uniform(-3.0, 0.0, size=mech.elem_count.shape[1])
        lnC = -g + np.log(mech.p_ref / (RU * T)) + mech.elem_count @ lam
        n_atoms = mech.elem_count.sum(1).astype(float)
        lo, hi = -200.0, 200.0
        for _ in range(100):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if (lnC + mid * n_atoms).max() < np.log(1e-3) else (lo, mid)
        C = np.exp(lnC + lo * n_atoms)
        P = C.sum() * RU * T
        Y = C * mech.mol_weight / (C * mech.mol_weight).sum()
        det = oracle.cell_detail(om, T, P, Y)
        phi = np.where(mech.rxn_type == 1, det["M"], 1.0)
        bounds.append(1e-10 * (np.abs(mech.nu_prod - mech.nu_reac) @ (phi * det["qf"])))
        Ps.append(P)
        Ys.append(Y)
    w, d = gpu_run(ck, mech, Ts, np.array(Ps), np.ascontiguousarray(np.array(Ys).T))
    assert (np.abs(w) <= np.array(bounds).T + 1e-300).all()


def test_deterministic_and_host_entry_point(ck):
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=5000)
    gm = ck.Mechanism(mech)
    w1, d1 = gpu_run(ck, mech, T, P, Y, gm)
    w2, d2 = gpu_run(ck, mech, T, P, Y, gm)
    assert np.array_equal(w1, w2) and np.array_equal(d1, d2)         # bitwise run to run
    wh, dh = gm.source_terms_host(T, P, Y)
    assert np.array_equal(wh, w1) and np.array_equal(dh, d1)         # same kernels, host buffers
    Tp, Pp, Yp = (torch.from_numpy(a).pin_memory() for a in (T, P, Y))
    wp = torch.empty((mech.n_species, 5000), dtype=torch.float64).pin_memory()
    dp = torch.empty(5000, dtype=torch.float64).pin_memory()
    gm.source_terms_host(Tp, Pp, Yp, wp, dp)
    assert np.array_equal(wp.numpy(), w1) and np.array_equal(dp.numpy(), d1)
    gm.close()


@pytest.mark.parametrize("chunks", [None, 1, 3, 16])
def test_host_entry_point_pipelined(ck, monkeypatch, kernel_variant, chunks):
    """ck_source_terms_host splits big batches into chunks of cells pipelined over copy-in /
    compute / copy-out streams: a ragged batch big enough to be split (and forced chunk counts)
    must give, cell for cell, the bits of one ck_source_terms call over the whole batch on the
    tiny mechanism (the per-cell arithmetic does not depend on the tiling), and results that
    were already in the output buffers beyond the batch must stay untouched."""
    if kernel_variant != "auto":
        pytest.skip("same host code for both kernels")
    if chunks is not None:
        monkeypatch.setenv("CK_HOST_CHUNKS", str(chunks))
    cfg = ckgen.CONFIGS["tiny_1m"]
    mech = ckgen.mechanism(cfg.mech)
    N = 3 * 65536 + 4097
    T, P, Y = ckgen.states(cfg, N=N)
    with ck.Mechanism(mech) as gm:
        w1, d1 = gpu_run(ck, mech, T, P, Y, gm)
        Tp, Pp, Yp = (torch.from_numpy(a).pin_memory() for a in (T, P, Y))
        wp = torch.full((mech.n_species, N), -7.0, dtype=torch.float64).pin_memory()
        dp = torch.full((N,), -7.0, dtype=torch.float64).pin_memory()
        for _ in range(2):      # second call reuses streams, events and staging
            gm.source_terms_host(Tp, Pp, Yp, wp, dp)
        assert np.array_equal(wp.numpy(), w1) and np.array_equal(dp.numpy(), d1)
        wh, dh = gm.source_terms_host(T, P, Y)      # pageable memory
        assert np.array_equal(wh, w1) and np.array_equal(dh, d1)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T[-4097:], P[-4097:], np.ascontiguousarray(Y[:, -4097:]))
    rw, rt = parity_violations(w1[:, -4097:], d1[-4097:], wr, dr)
    assert rw <= 1.0 and rt <= 1.0


@pytest.mark.parametrize("cfg_name,N", [("mid_1m", 2048), ("mid_1m", 40000), ("tiny_1k", 3000), ("large_256k", 1500)])
def test_concurrent_calls_on_two_streams_share_one_handle(ck, cfg_name, N):
    """ck_source_terms is re-entrant for distinct output buffers.  Two
    streams launch on ONE handle at the same time, over and over, with different inputs and
    outputs (grids small enough to be resident side by side at the small N); every result must
    match the oracle and be bitwise what a call alone gives -- the blocks of overlapping launches
    each take their own slot of the M = C E scratch (third-body and falloff rates would be
    corrupted otherwise)."""
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    S = mech.n_species
    dev = torch.device("cuda:0")
    om = oracle.OracleMechanism(mech)
    batches = [ckgen.states(cfg, N=N, seed_offset=o) for o in (0, 1)]
    refs = [oracle.source_terms(om, *b)[:2] for b in batches]
    with ck.Mechanism(mech) as gm:
        alone = [gpu_run(ck, mech, *b, gm) for b in batches]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        bufs = []
        for b, st in zip(batches, streams):
            with torch.cuda.stream(st):
                Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in b)
                w = torch.empty((S, N), dtype=torch.float64, device=dev)
                d = torch.empty((N,), dtype=torch.float64, device=dev)
            bufs.append((Td, Pd, Yd, w, d))
        torch.cuda.synchronize()
        for rep in range(25):
            for (Td, Pd, Yd, w, d), st in zip(bufs, streams):
                gm.source_terms(Td, Pd, Yd, w, d, stream=st.cuda_stream)
        torch.cuda.synchronize()
        for (Td, Pd, Yd, w, d), (wa, da), (wr, dr) in zip(bufs, alone, refs):
            wg, dg = w.cpu().numpy(), d.cpu().numpy()
            assert np.array_equal(wg, wa) and np.array_equal(dg, da)
            rw, rt = parity_violations(wg, dg, wr, dr)
            assert rw <= 1.0 and rt <= 1.0, (cfg_name, rw, rt)


@pytest.mark.parametrize("N_a,N_b", [(2048, 40000), (3000, 8000), (4736, 4737), (9472, 9473), (777, 300000)])
def test_concurrent_calls_of_different_shapes_share_one_handle(ck, kernel_variant, N_a, N_b):
    """The kernel shapes built on one handle (8 and 4 threads per cell for small batches, thread <-> cell
    beyond) share the M = C E scratch and its busy flags, so slot s has to be the same bytes in all of
    them: two streams launch calls that select DIFFERENT shapes on one handle at the same time, over and
    over; every result is bitwise what the call gives alone (and that one matches the oracle)."""
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    S = mech.n_species
    dev = torch.device("cuda:0")
    om = oracle.OracleMechanism(mech)
    batches = [ckgen.states(cfg, N=n, seed_offset=o) for o, n in enumerate((N_a, N_b))]
    with ck.Mechanism(mech) as gm:
        if kernel_variant == "auto":
            assert gm.info("small_batch_max") == 9472
        alone = [gpu_run(ck, mech, *b, gm) for b in batches]
        for b, (wa, da) in zip(batches, alone):
            n = min(b[0].shape[0], 4000)          # (the oracle on a sample; full batches have their own tests)
            wr, dr, _ = oracle.source_terms(om, b[0][:n], b[1][:n], np.ascontiguousarray(b[2][:, :n]))
            rw, rt = parity_violations(wa[:, :n], da[:n], wr, dr)
            assert rw <= 1.0 and rt <= 1.0, (N_a, N_b, rw, rt)
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        bufs = []
        for b, st in zip(batches, streams):
            with torch.cuda.stream(st):
                Td, Pd, Yd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in b)
                w = torch.empty((S, b[0].shape[0]), dtype=torch.float64, device=dev)
                d = torch.empty((b[0].shape[0],), dtype=torch.float64, device=dev)
            bufs.append((Td, Pd, Yd, w, d))
        torch.cuda.synchronize()
        # the shorter call is repeated more often so that both streams stay busy for about as long
        reps = [max(1, int(25 * max(N_a, N_b) / max(n, 8192))) for n in (N_a, N_b)]
        for rep in range(max(reps)):
            for (Td, Pd, Yd, w, d), st, r in zip(bufs, streams, reps):
                if rep < r:
                    gm.source_terms(Td, Pd, Yd, w, d, stream=st.cuda_stream)
        torch.cuda.synchronize()
        for (Td, Pd, Yd, w, d), (wa, da) in zip(bufs, alone):
            assert np.array_equal(w.cpu().numpy(), wa) and np.array_equal(d.cpu().numpy(), da)


def test_source_terms_beside_rk4_on_one_handle(ck, kernel_variant):
    """ck_rk4_integrate's stage kernels take their M = C E slots from the same scratch and flags as
    ck_source_terms: a reactor run on one stream and source-term calls of a small-batch shape on another,
    on ONE handle, both give the bits they give alone."""
    from helpers import tame
    cfg = ckgen.CONFIGS["mid_rk4"]
    mech = tame(ckgen.mechanism(cfg.mech))
    S = mech.n_species
    dev = torch.device("cuda:0")
    N_rk, N_st, steps, dt = 20000, 3000, 12, 1e-9
    Tr, Pr, Yr = ckgen.states(cfg, N=N_rk, seed_offset=3)
    Ts, Ps, Ys = ckgen.states(cfg, N=N_st, seed_offset=4)
    put = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    with ck.Mechanism(mech) as gm:
        w_alone, d_alone = gpu_run(ck, mech, Ts, Ps, Ys, gm)
        T1, P1, Y1 = put(Tr), put(Pr), put(Yr)
        gm.rk4_integrate(T1, P1, Y1, dt, steps, use_graph=False)
        torch.cuda.synchronize()
        T_alone, Y_alone = T1.cpu().numpy(), Y1.cpu().numpy()
        assert np.isfinite(T_alone).all() and np.isfinite(Y_alone).all()
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        T2, P2, Y2 = put(Tr), put(Pr), put(Yr)
        Td, Pd, Yd = put(Ts), put(Ps), put(Ys)
        w = torch.empty((S, N_st), dtype=torch.float64, device=dev)
        d = torch.empty((N_st,), dtype=torch.float64, device=dev)
        torch.cuda.synchronize()
        gm.rk4_integrate(T2, P2, Y2, dt, steps, use_graph=False, stream=sa.cuda_stream)
        for rep in range(40):
            gm.source_terms(Td, Pd, Yd, w, d, stream=sb.cuda_stream)
        torch.cuda.synchronize()
        assert np.array_equal(T2.cpu().numpy(), T_alone) and np.array_equal(Y2.cpu().numpy(), Y_alone)
        assert np.array_equal(w.cpu().numpy(), w_alone) and np.array_equal(d.cpu().numpy(), d_alone)


@pytest.mark.parametrize("N", [1, 31, 32, 33, 256, 1000, 4096, 4736, 4737, 9472, 9473, 18944, 18945])
def test_small_batch_shape_is_selected_and_matches_the_oracle(ck, kernel_variant, N):
    """Below one wave of 32-cell tiles (N <= 32 x 148) ck_source_terms runs the small-batch shape of
    the specialised kernel: 8 threads per cell taking alternate reaction blocks, partial accumulators
    summed in a fixed order (the flat region of the paper's Fig. 9).  Parity on
    the auto-selected shape on both sides of the switch, ragged tiles included, bitwise run to run;
    with it turned off the same cells agree to the tolerance (another summation order)."""
    if kernel_variant != "auto":
        pytest.skip("specialised kernel only")
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    with ck.Mechanism(mech) as gm:
        assert gm.info("small_batch_max") == 64 * 148     # (2 threads per cell do not fit shared memory at S=53)
        w1, d1 = gpu_run(ck, mech, T, P, Y, gm)
        w2, d2 = gpu_run(ck, mech, T, P, Y, gm)
    assert np.array_equal(w1, w2) and np.array_equal(d1, d2)
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y)
    rw, rt = parity_violations(w1, d1, wr, dr)
    assert rw <= 1.0 and rt <= 1.0, (N, rw, rt)


def test_small_batch_shape_variants(ck, kernel_variant, monkeypatch):
    """4 and 2 threads per cell (CK_JIT_SPLIT), the fp32-rates precision in the small-batch shape,
    several temperature ranges, and mechanisms that do not get the shape (few reactions, S > 103)."""
    if kernel_variant != "auto":
        pytest.skip("specialised kernel only")
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    rng = np.random.default_rng(11)
    mech_r = dataclasses.replace(mech, T_mid=rng.choice([800.0, 1000.0, 1400.0], size=mech.n_species))
    T, P, Y = ckgen.states(dataclasses.replace(cfg, T_range=(500.0, 2700.0)), N=777)
    for split, cells in (("8", 32), ("4", 64), ("2", 0)):
        monkeypatch.setenv("CK_JIT_SPLIT", split)
        with ck.Mechanism(mech) as gm:
            assert gm.info("small_batch_max") == cells * 148
        assert_parity(ck, mech, T, P, Y, "split %s" % split)
        assert_parity(ck, mech_r, T, P, Y, "split %s, four temperature ranges" % split)
    monkeypatch.setenv("CK_JIT_SPLIT", "0")
    with ck.Mechanism(mech) as gm:
        assert gm.info("small_batch_max") == 0
    monkeypatch.delenv("CK_JIT_SPLIT")
    with ck.Mechanism(ckgen.mechanism(ckgen.MECH_TINY)) as gm:
        assert gm.info("small_batch_max") == 0           # 21 reactions: the walk is short
    with ck.Mechanism(ckgen.mechanism(ckgen.MECH_LARGE)) as gm:
        assert gm.info("small_batch_max") == 0           # accumulators do not fit one thread's registers
    with ck.Mechanism(mech, precision=2) as gm:
        assert gm.info("small_batch_max") == 128 * 148    # (rate table in fp32: half the size)


@pytest.mark.parametrize("cfg_name,N", [("mid_1m", 148 * 256 * 2 + 4321), ("large_256k", 148 * 128 + 777), ("tiny_1k", 70001)])
def test_every_tile_size_gives_the_same_bits(ck, kernel_variant, monkeypatch, cfg_name, N):
    """A cell's arithmetic does not depend on the tile it falls into or on how many tiles a block
    walks: the specialised kernel with its tile size forced to 32, 64, 96, 160, ... cells (CK_JIT_TILE;
    other grids, other numbers of tiles per block, other interleavings of the bulk loads, the
    mbarrier phases, the pair barriers and the M-scratch slots) returns, bit for bit, what the
    balanced default returns.  Stresses the hand-offs the parity tests only see in one schedule."""
    if kernel_variant != "auto":
        pytest.skip("specialised kernel only")
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    dev = torch.device("cuda:0")
    Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
    st = torch.cuda.current_stream().cuda_stream

    def run(gm):
        w = torch.full((mech.n_species, N), float("nan"), dtype=torch.float64, device=dev)
        d = torch.full((N,), float("nan"), dtype=torch.float64, device=dev)
        gm.source_terms(Td, Pd, Yd, w, d, stream=st)
        torch.cuda.synchronize()
        return w, d

    with ck.Mechanism(mech) as gm:
        assert gm.info("jit") == 1
        w0, d0 = run(gm)
        assert torch.isfinite(w0).all() and torch.isfinite(d0).all()
        cells = gm.info("threads") // (2 if gm.info("pair") else 1)
    for tile in (32, 64, 96, 160, 224, 256):
        if tile > cells:
            continue
        monkeypatch.setenv("CK_JIT_TILE", str(tile))           # (read by ck_mech_create, not by the call)
        with ck.Mechanism(mech) as gm:
            for _ in range(2):
                w, d = run(gm)
                assert torch.equal(w, w0) and torch.equal(d, d0), (cfg_name, tile)
    monkeypatch.delenv("CK_JIT_TILE")


@pytest.mark.parametrize("knob,value", [("CK_JIT_KC", "none"), ("CK_JACJ_EXP", "1"), ("CK_JACJ_TIMING", "1")])
def test_result_changing_knobs_are_refused_without_the_ablation_switch(ck, monkeypatch, kernel_variant, knob, value):
    """Environment knobs that make a kernel compute something other than the source term or the Jacobian
    (measurement-only ablations) are refused by ck_mech_create unless CK_ALLOW_ABLATION=1 is set as well,
    and a handle built with them says so through ck_mech_info 18 ("ablation")."""
    if kernel_variant != "auto":
        pytest.skip("the knobs exist only in the specialised kernels")
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    with ck.Mechanism(mech) as gm:
        assert gm.info("ablation") == 0
    monkeypatch.setenv(knob, value)
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(mech)
    assert e.value.status == 1 and "CK_ALLOW_ABLATION" in str(e.value)
    if knob != "CK_JACJ_TIMING":            # (that one makes the kernel print: not built here)
        monkeypatch.setenv("CK_ALLOW_ABLATION", "1")
        with ck.Mechanism(mech) as gm:
            assert gm.info("ablation") == 1


def test_error_codes(ck):
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    gm = ck.Mechanism(mech)
    with pytest.raises(ck.CkError) as e:
        ck.ck_source_terms(gm.handle, 0, 0, 0, 16, 0, 0)
    assert e.value.status == 1
    with pytest.raises(ck.CkError) as e:
        ck.ck_source_terms(gm.handle, 8, 8, 8, -1, 8, 8)
    assert e.value.status == 1
    with pytest.raises(ck.CkError) as e:
        ck.ck_source_terms(None, 8, 8, 8, 4, 8, 8)
    assert e.value.status == 1
    gm.close()
    bad = dataclasses.replace(mech, rxn_type=np.full(mech.n_reactions, 9, np.uint8))
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(bad)
    assert e.value.status == 4
    bad = dataclasses.replace(mech, mol_weight=-mech.mol_weight)
    with pytest.raises(ck.CkError) as e:
        ck.Mechanism(bad)
    assert e.value.status == 1
