"""Parity of ck_jacobian (through the C ABI) against the oracle's analytic Jacobian
(oracle/ck_oracle_jac.c), entry by entry.

Tolerance: the GPU forms every rate in log form (relative error of a
rate ~1e-14 |ln q| ~ 1e-12) and each entry of a species row is a sum of such terms whose
natural size is the largest entry of its column, so
    |dJ_il| <= 1e-9 max_i |J_il| + 1e-11 |J_il|            (species rows, per cell and column)
and the energy row, a sum over species that cancels like dT/dt itself, is measured against
the sum of the absolute terms it is made of:
    |dJ_Sl| <= 1e-9 (sum_k |H_k J_kl| / D + |J_Sl|),  H_k = (h_k/RT) Ru T, D = rho cp.
"""
import numpy as np
import pytest

import ckgen
import oracle
from helpers import RU

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ck():
    import paper_2008_08483_b200 as ck
    assert torch.cuda.is_available()
    return ck


@pytest.fixture(autouse=True, params=["jit", "v2", "v1"])
def jac_kernel(request, monkeypatch):
    """Every test runs on all three Jacobian kernels: jit (the mechanism-specialised kernel, the
    default where it exists: CK_JAC_KERNEL unset; mechanisms it does not take fall to v2 / v1),
    v2 (table-driven, lanes = cells, DMMA dense part) and v1 (table-driven, lanes = columns, tiles of
    4 to 32 cells)."""
    if request.param == "jit":
        monkeypatch.delenv("CK_JAC_KERNEL", raising=False)
    else:
        monkeypatch.setenv("CK_JAC_KERNEL", request.param)
    return request.param


def gpu_jacobian(ck, gm, T, P, Y):
    dev = torch.device("cuda:0")
    N, S = T.shape[0], Y.shape[0]
    Td, Pd, Yd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (T, P, Y))
    J = torch.full((N, S + 1, S + 1), float("nan"), dtype=torch.float64, device=dev)
    gm.jacobian(Td, Pd, Yd, J, stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return J.cpu().numpy()


def violations(mech, T, P, Y, J, Jr):
    """Worst error/tolerance over the species rows and over the energy row."""
    S = mech.n_species
    om = oracle.OracleMechanism(mech)
    assert np.isfinite(J).all()
    col = np.abs(Jr[:, :S, :]).max(axis=1, keepdims=True)
    tol = 1e-9 * col + 1e-11 * np.abs(Jr[:, :S, :])
    rs = float((np.abs(J[:, :S, :] - Jr[:, :S, :]) / np.maximum(tol, 1e-300)).max())
    re = 0.0
    for i in range(T.shape[0]):
        det = oracle.cell_detail(om, T[i], P[i], Y[:, i])
        H = det["h_RT"] * RU * T[i]
        D = det["rho"] * det["cp_mass"]
        scale = (np.abs(H[:, None] * Jr[i, :S, :])).sum(0) / D + np.abs(Jr[i, S, :])
        re = max(re, float((np.abs(J[i, S, :] - Jr[i, S, :]) / (1e-9 * scale)).max()))
    return rs, re


@pytest.mark.parametrize("cfg_name,N", [("tiny_1k", 1024), ("mid_1m", 203), ("large_256k", 61), ("mid_rk4", 50)])
def test_parity_all_entries(ck, cfg_name, N):
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    T[: N // 4] = np.linspace(350.0, 1000.0, N // 4)      # low NASA range and T = T_mid exactly
    with ck.Mechanism(mech) as gm:
        assert gm.info("jac_cells") in (4, 8, 16) or (gm.info("jac_cells") % 32 == 0 and gm.info("jac_cells") <= 512)
        J = gpu_jacobian(ck, gm, T, P, Y)
    Jr = oracle.jacobian(oracle.OracleMechanism(mech), T, P, Y)
    rs, re = violations(mech, T, P, Y, J, Jr)
    print("%s: worst Jacobian error / bound: species rows %.3g, energy row %.3g" % (cfg_name, rs, re))
    assert rs <= 1.0 and re <= 1.0, (cfg_name, rs, re)


@pytest.mark.parametrize("N", [1, 3, 7, 8, 9, 17, 31, 32, 33, 65])
def test_ragged_batches_and_determinism(ck, N):
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    with ck.Mechanism(mech) as gm:
        J1 = gpu_jacobian(ck, gm, T, P, Y)
        J2 = gpu_jacobian(ck, gm, T, P, Y)
    assert np.array_equal(J1, J2)
    Jr = oracle.jacobian(oracle.OracleMechanism(mech), T, P, Y)
    rs, re = violations(mech, T, P, Y, J1, Jr)
    assert rs <= 1.0 and re <= 1.0, (N, rs, re)


@pytest.mark.parametrize("shape", ["4,16,1", "8,16,1", "16,16,1", "32,16,1", "4,8,2"])
@pytest.mark.parametrize("N", [1, 31, 33, 70])
def test_every_launch_shape_on_the_tiny_mechanism(ck, monkeypatch, jac_kernel, shape, N):
    """Tiles of 4 to 32 cells and both block sizes (CK_JAC_SHAPE = cells, warps, blocks per SM),
    with batches that leave a ragged last tile: same bits from every shape (the arithmetic of a
    cell does not depend on the tile it falls in), parity on one of them."""
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    with ck.Mechanism(mech) as gm:
        Jd = gpu_jacobian(ck, gm, T, P, Y)
    if jac_kernel != "v1":
        pytest.skip("launch shapes of the first kernel")
    monkeypatch.setenv("CK_JAC_SHAPE", shape)
    with ck.Mechanism(mech) as gm:
        assert gm.info("jac_cells") == int(shape.split(",")[0])
        J = gpu_jacobian(ck, gm, T, P, Y)
    Jr = oracle.jacobian(oracle.OracleMechanism(mech), T, P, Y)
    rs, re = violations(mech, T, P, Y, J, Jr)
    assert rs <= 1.0 and re <= 1.0, (shape, N, rs, re)
    rs, re = violations(mech, T, P, Y, Jd, Jr)
    assert rs <= 1.0 and re <= 1.0, ("default", N, rs, re)


def test_single_reaction_mechanisms(ck):
    """Each reaction type as a mechanism of its own (no reaction hides behind a larger one),
    including irreversible ones."""
    import dataclasses
    mech = ckgen.mechanism(ckgen.MECH_MID)
    cfg = dataclasses.replace(ckgen.CONFIGS["mid_1m"], T_range=(600.0, 2800.0))
    T, P, Y = ckgen.states(cfg, N=40)
    picks = np.concatenate([np.flatnonzero(mech.rxn_type == 3)[:4], np.flatnonzero(mech.rxn_type == 1)[:4],
                            np.flatnonzero(mech.rxn_type == 0)[:6]])
    for n, j in enumerate(picks):
        sub = mech.subset([j])
        if n % 2:
            sub = dataclasses.replace(sub, reversible=np.zeros(1, np.uint8))
        with ck.Mechanism(sub) as gm:
            J = gpu_jacobian(ck, gm, T, P, Y)
        Jr = oracle.jacobian(oracle.OracleMechanism(sub), T, P, Y)
        rs, re = violations(sub, T, P, Y, J, Jr)
        assert rs <= 1.0 and re <= 1.0, (int(j), rs, re)


def test_lindemann_and_three_parameter_troe(ck):
    import dataclasses
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    rt = mech.rxn_type.copy()
    troe = mech.troe.copy()
    fo = np.flatnonzero(rt == 3)
    rt[fo[0]] = 2                       # Lindemann
    troe[fo[1:], 3] = np.inf            # 3-parameter Troe
    mech = dataclasses.replace(mech, rxn_type=rt, troe=troe)
    T, P, Y = ckgen.states(ckgen.CONFIGS["tiny_1k"], N=64)
    with ck.Mechanism(mech) as gm:
        J = gpu_jacobian(ck, gm, T, P, Y)
    Jr = oracle.jacobian(oracle.OracleMechanism(mech), T, P, Y)
    rs, re = violations(mech, T, P, Y, J, Jr)
    assert rs <= 1.0 and re <= 1.0, (rs, re)


def test_catalyst_species_real_valued_nu_and_irreversible_reactions(ck):
    """A + B -> A + C style reactions (nu' and nu'' overlap: the species has a column but no row
    entry for that reaction), a real-valued stoichiometric coefficient, a third of the
    reactions irreversible."""
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
    mech = dataclasses.replace(mech, nu_reac=nu_r, nu_prod=nu_p, reversible=rev)
    T, P, Y = ckgen.states(cfg, N=90)
    with ck.Mechanism(mech) as gm:
        J = gpu_jacobian(ck, gm, T, P, Y)
    Jr = oracle.jacobian(oracle.OracleMechanism(mech), T, P, Y)
    rs, re = violations(mech, T, P, Y, J, Jr)
    assert rs <= 1.0 and re <= 1.0, (rs, re)


@pytest.mark.parametrize("cfg_name,N", [("mid_1m", 1 << 15), ("large_256k", 1 << 13)])
def test_bench_size_properties_and_sampled_parity(ck, cfg_name, N):
    """At the size bench.py --jacobian times: Euler's relation sum_l Y_l J_il = 0 and mass
    conservation sum_i W_i J_il = 0 on every cell (on the device), the oracle on a sample."""
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    S = mech.n_species
    T, P, Y = ckgen.states(cfg, N=N)
    dev = torch.device("cuda:0")
    Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
    J = torch.empty((N, S + 1, S + 1), dtype=torch.float64, device=dev)
    with ck.Mechanism(mech) as gm:
        gm.jacobian(Td, Pd, Yd, J, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    assert torch.isfinite(J).all()
    terms = J[:, :, :S] * Yd.T[:, None, :]
    assert (terms.sum(2).abs() <= 1e-9 * terms.abs().sum(2) + 1e-300).all()
    del terms
    w = torch.from_numpy(mech.mol_weight).to(dev)
    t = J[:, :S, :] * w[None, :, None]
    assert (t.sum(1).abs() <= 1e-9 * t.abs().sum(1) + 1e-300).all()
    del t
    idx = np.unique(np.concatenate([np.random.default_rng(7).integers(0, N, 40), [0, 7, 8, N - 9, N - 1]]))
    Jr = oracle.jacobian(oracle.OracleMechanism(mech), T[idx], P[idx], np.ascontiguousarray(Y[:, idx]))
    rs, re = violations(mech, T[idx], P[idx], np.ascontiguousarray(Y[:, idx]), J[idx].cpu().numpy(), Jr)
    assert rs <= 1.0 and re <= 1.0, (rs, re)


def violations_vectorised(mech, T, P, Y, J, Jr):
    """`violations` for large batches: the same two bounds, the energy row's scale from numpy
    expressions of rho, cp and h (tolerance scales only; no oracle value is replaced)."""
    from helpers import nasa_h_RT
    S = mech.n_species
    col = np.abs(Jr[:, :S, :]).max(axis=1, keepdims=True)
    tol = 1e-9 * col + 1e-11 * np.abs(Jr[:, :S, :])
    rs = float((np.abs(J[:, :S, :] - Jr[:, :S, :]) / np.maximum(tol, 1e-300)).max())
    H = (nasa_h_RT(mech, T) * RU * T[None, :]).T                         # [N, S]
    yw = np.maximum(Y, 0.0) / mech.mol_weight[:, None]                   # [S, N]
    rho = P / (RU * T * yw.sum(0))
    Tn = T[None, :]
    low = Tn <= mech.T_mid[:, None]
    cp = lambda a: a[:, 0, None] + a[:, 1, None] * Tn + a[:, 2, None] * Tn**2 + a[:, 3, None] * Tn**3 + a[:, 4, None] * Tn**4
    cp_mass = (yw * np.where(low, cp(mech.nasa_lo), cp(mech.nasa_hi)) * RU).sum(0)
    D = rho * cp_mass
    scale = np.einsum("ns,nsl->nl", np.abs(H), np.abs(Jr[:, :S, :])) / D[:, None] + np.abs(Jr[:, S, :])
    re = float((np.abs(J[:, S, :] - Jr[:, S, :]) / (1e-9 * scale)).max())
    return rs, re


def composition_scale(mech, om, T, P, Y, k, l):
    """DESIGN.md reading Q20.  An entry of a species row and a composition column is
        J_kl = sum_j nu_kj [ q_f,j (nu'_lj / Y_l - sum_i nu'_ij W_mix / W_l)
                            - q_r,j (nu''_lj / Y_l - sum_i nu''_ij W_mix / W_l) ] + (third-body, falloff terms):
    C_i = rho Y_i / W_i with rho ~ W_mix at constant P, so every reaction's derivative is a DIFFERENCE of the
    direct term nu_l / Y_l and the density term (sum nu) W_mix / W_l.  Where the two nearly coincide the fp64
    oracle's own rounding of that difference is about 2^-53 of the terms, not of the result.  Returns the scale
    of the terms, sum_j |nu_kj| [ q_f (nu'_l / Y_l + sum nu' W_mix / W_l) + q_r (...'') ], from the oracle's
    q_f, q_r of one cell (the third-body and falloff terms would only add to it)."""
    det = oracle.cell_detail(om, T, P, Y)
    W = mech.mol_weight
    Wmix = 1.0 / (Y / W).sum()
    nu1, nu2 = mech.nu_reac, mech.nu_prod
    tf, sf = nu1[l] / Y[l], nu1.sum(0) * Wmix / W[l]
    tr, sr = nu2[l] / Y[l], nu2.sum(0) * Wmix / W[l]
    return float((np.abs(nu2[k] - nu1[k]) * (det["qf"] * (tf + sf) + det["qr"] * (tr + sr))).sum())


@pytest.mark.parametrize("cfg_name,N", [("tiny_1m", 1 << 20), ("mid_1m", 1 << 16), ("large_256k", 1 << 14)])
def test_every_entry_at_the_sizes_bench_times(ck, jac_kernel, cfg_name, N):
    """Every entry of every cell's matrix against the oracle's Jacobian at the batch sizes
    bench.py --jacobian times (2^20 cells at S=9, 2^16 at S=53, 2^14 at S=111), in the launch
    configuration it times (one ck_jacobian call over the whole batch), compared chunk by chunk."""
    if jac_kernel != "jit":
        pytest.skip("the kernel bench.py times is the default one; the table-driven kernels have test_parity_all_entries")
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    om = oracle.OracleMechanism(mech)
    S = mech.n_species
    T, P, Y = ckgen.states(cfg, N=N)
    dev = torch.device("cuda:0")
    Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
    J = torch.full((N, S + 1, S + 1), float("nan"), dtype=torch.float64, device=dev)
    with ck.Mechanism(mech) as gm:
        gm.jacobian(Td, Pd, Yd, J, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    assert torch.isfinite(J).all()
    chunk = max(1024, (1 << 26) // ((S + 1) * (S + 1) * 8))               # about 64 MB of matrices at a time
    worst_s = worst_e = 0.0
    flagged = []          # (cell, row, column, error, column max, oracle value) of species-row entries over the bound
    for c0 in range(0, N, chunk):
        c1 = min(N, c0 + chunk)
        Yc = np.ascontiguousarray(Y[:, c0:c1])
        Jr = oracle.jacobian(om, T[c0:c1], P[c0:c1], Yc)
        Jg = J[c0:c1].cpu().numpy()
        rs, re = violations_vectorised(mech, T[c0:c1], P[c0:c1], Yc, Jg, Jr)
        if rs > 1.0:
            col = np.abs(Jr[:, :S, :]).max(axis=1, keepdims=True)
            err = np.abs(Jg[:, :S, :] - Jr[:, :S, :])
            for i, k, l in zip(*np.nonzero(err > 1e-9 * col + 1e-11 * np.abs(Jr[:, :S, :]))):
                flagged.append((c0 + i, k, l, err[i, k, l], col[i, 0, l], Jr[i, k, l]))
            rs = float(np.where(err > 1e-9 * col + 1e-11 * np.abs(Jr[:, :S, :]), 0.0,
                                err / np.maximum(1e-9 * col + 1e-11 * np.abs(Jr[:, :S, :]), 1e-300)).max())
        worst_s, worst_e = max(worst_s, rs), max(worst_e, re)
    print("%s N=%d, every entry: worst Jacobian error / bound: species rows %.3g, energy row %.3g; %d entries in %d cells "
          "decided by reading Q20" % (cfg_name, N, worst_s, worst_e, len(flagged), len({f[0] for f in flagged})))
    assert worst_s <= 1.0 and worst_e <= 1.0, (cfg_name, worst_s, worst_e)
    # Entries over the bound: few, in composition columns, ill-conditioned by the cancellation of reading Q20
    # (terms > 1e3 x the column's largest entry), and within 1e-9 colmax + 1e-15 x the terms' scale (9 ulp of
    # the terms: the quotient, the product and the S-term sum for W_mix behind each of them).
    assert len({f[0] for f in flagged}) <= max(1, N // 20000), len(flagged)
    for i, k, l, err, colmax, ref in flagged:
        assert l < S, ("temperature column over the bound", i, k, l)
        scale = composition_scale(mech, om, T[i], P[i], np.ascontiguousarray(Y[:, i]), k, l)
        print("  cell %d entry (%d, %d): oracle %.9e, |gpu - oracle| = %.3g x 1e-9 colmax, terms / colmax = %.3g, "
              "error / Q20 bound %.3g" % (i, k, l, ref, err / (1e-9 * colmax), scale / colmax,
                                          err / (1e-9 * colmax + 1e-15 * scale)))
        assert scale > 1e3 * colmax and err <= 1e-9 * colmax + 1e-15 * scale, (i, k, l, err, colmax, scale)


def test_errors(ck):
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    ann = ckgen.random_kc_ann(mech.n_reactions, 1, 4, seed=1, T_range=(1000.0, 2500.0))
    with ck.Mechanism(mech, kc_ann=ann) as gm:
        assert gm.info("jac_cells") == 0
        with pytest.raises(ck.CkError) as e:
            ck.ck_jacobian(gm.handle, 8, 8, 8, 4, 8)
        assert e.value.status == 4
    with ck.Mechanism(mech) as gm:
        ck.ck_jacobian(gm.handle, 0, 0, 0, 0, 0)           # N == 0: a no-op
        with pytest.raises(ck.CkError) as e:
            ck.ck_jacobian(gm.handle, 0, 8, 8, 4, 8)
        assert e.value.status == 1
        with pytest.raises(ck.CkError) as e:
            ck.ck_jacobian(gm.handle, 8, 8, 8, -1, 8)
        assert e.value.status == 1


def test_kernel_in_use_and_a_J_that_is_only_8_byte_aligned(ck, jac_kernel):
    """ck_mech_info 22 names the kernel; the specialised kernel stores rows by 16-byte bulk / tensor
    copies, so a J that is only 8-byte aligned goes through the table-driven kernels: same values
    to the parity bound, every entry written."""
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    N, S = 77, mech.n_species
    T, P, Y = ckgen.states(cfg, N=N)
    dev = torch.device("cuda:0")
    Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
    with ck.Mechanism(mech) as gm:
        assert gm.info("jac_kernel") == {"jit": 3, "v2": 2, "v1": 1}[jac_kernel]
        buf = torch.full((N * (S + 1) * (S + 1) + 1,), float("nan"), dtype=torch.float64, device=dev)
        Jm = buf[1:].view(N, S + 1, S + 1)                 # 8 bytes past a 16-byte boundary
        assert Jm.data_ptr() % 16 == 8
        gm.jacobian(Td, Pd, Yd, Jm, stream=torch.cuda.current_stream().cuda_stream)
        Ja = gpu_jacobian(ck, gm, T, P, Y)
        torch.cuda.synchronize()
    Jm = Jm.cpu().numpy()
    assert np.isnan(buf[0].item())
    Jr = oracle.jacobian(oracle.OracleMechanism(mech), T, P, Y)
    for Jx in (Jm, Ja):
        rs, re = violations(mech, T, P, Y, Jx, Jr)
        assert rs <= 1.0 and re <= 1.0, (rs, re)


@pytest.mark.parametrize("cfg_name,N", [("mid_1m", 148 * 224 + 1234), ("tiny_1k", 148 * 512 * 2 + 99)])
def test_every_tile_size_gives_the_same_bits(ck, jac_kernel, monkeypatch, cfg_name, N):
    """The specialised kernel with its tile size forced (CK_JACJ_TILE: other grids, other numbers of tiles
    per block, other hand-offs between the out buffers, the tensor copies and the scratch) returns,
    bit for bit, what the balanced default returns."""
    if jac_kernel != "jit":
        pytest.skip("specialised kernel only")
    cfg = ckgen.CONFIGS[cfg_name]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=N)
    dev = torch.device("cuda:0")
    S = mech.n_species
    Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))

    def run(gm):
        J = torch.full((N, S + 1, S + 1), float("nan"), dtype=torch.float64, device=dev)
        gm.jacobian(Td, Pd, Yd, J, stream=torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return J

    with ck.Mechanism(mech) as gm:
        assert gm.info("jac_kernel") == 3
        J0 = run(gm)
        assert torch.isfinite(J0).all()
        cells = gm.info("jac_cells")
    for tile in (32, 96, 160, 224, 384, 512):
        if tile > cells:
            continue
        monkeypatch.setenv("CK_JACJ_TILE", str(tile))      # (read by ck_mech_create, not by the call)
        with ck.Mechanism(mech) as gm:
            J = run(gm)
        assert torch.equal(J, J0), (cfg_name, tile)
        del J
    monkeypatch.delenv("CK_JACJ_TILE")
