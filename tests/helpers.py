"""Shared test helpers: the north_star parity tolerance and a numpy restatement of the
paper's matrix equations (a second, independent derivation used to pin the oracle)."""
import numpy as np

RU = 8314.46261815324  # J/(kmol K)


def parity_violations(wdot, dTdt, wdot_ref, dTdt_ref):
    """north_star tolerance (BASELINE.json):
       |d wdot_k| <= 1e-10 * max_k |wdot_k| + 1e-12 * |wdot_k|   per cell
       |d dT/dt|  <= 1e-10 * |dT/dt| + 1e-12 K/s
    Returns (worst wdot ratio err/tol, worst dTdt ratio err/tol); both must be <= 1."""
    wmax = np.abs(wdot_ref).max(axis=0, keepdims=True)
    tol_w = 1e-10 * wmax + 1e-12 * np.abs(wdot_ref)
    err_w = np.abs(wdot - wdot_ref)
    tol_t = 1e-10 * np.abs(dTdt_ref) + 1e-12
    err_t = np.abs(dTdt - dTdt_ref)
    # tol_w can be 0 only if the whole reference column is 0; then err must be 0 too
    rw = np.where(tol_w > 0, err_w / np.where(tol_w > 0, tol_w, 1.0), np.where(err_w > 0, np.inf, 0.0))
    rt = err_t / tol_t
    if not (np.isfinite(wdot).all() and np.isfinite(dTdt).all()):
        return np.inf, np.inf
    return float(rw.max()) if rw.size else 0.0, float(rt.max()) if rt.size else 0.0


def nasa_h_RT(mech, T):
    """h_k/RT [S, N] from the NASA-7 sets, low set for T <= T_mid."""
    T = np.asarray(T, dtype=np.float64)[None, :]

    def h(a):
        return (a[:, 0, None] + a[:, 1, None] * T / 2 + a[:, 2, None] * T**2 / 3 + a[:, 3, None] * T**3 / 4
                + a[:, 4, None] * T**4 / 5 + a[:, 5, None] / T)
    return np.where(T <= mech.T_mid[:, None], h(mech.nasa_lo), h(mech.nasa_hi))


def energy_kappa(mech, T, wdot_ref):
    """kappa = sum_k |h_k wdot_k| / |sum_k h_k wdot_k| per cell: the condition number of the energy
    sum in dT/dt = -sum_k h_k wdot_k / (rho cp) (tolerance notes)."""
    hw = nasa_h_RT(mech, T) * wdot_ref
    return np.abs(hw).sum(0) / np.maximum(np.abs(hw.sum(0)), 1e-300)


def dTdt_conditioned_violations(mech, T, dTdt, wdot_ref, dTdt_ref):
    """DESIGN.md reading Q19.  The north_star bound |d dT/dt| <= 1e-10 |dT/dt| + 1e-12 K/s is purely
    relative, but dT/dt is a sum of S terms h_k wdot_k that cancel: with condition number kappa a
    relative error eps of the rates becomes kappa * eps in dT/dt, and the fp64 ORACLE itself is then
    off the exact value by more than the bound (measured: 1.65e-10 at kappa = 7.4e4, against a
    long-double evaluation).  For cells that break the north_star bound on dT/dt ALONE the decision is
    taken against the sum's own scale, as the north_star does for wdot (relative to max_k |wdot_k|):
        |d dT/dt| <= 1e-10 |dT/dt| + 1e-12 + 1e-14 sum_k |h_k wdot_k| / (rho cp)
                   = (1e-10 + 1e-14 kappa) |dT/dt| + 1e-12.
    Returns (indices of the cells over the north_star bound, their kappa, their error / that bound)."""
    err = np.abs(dTdt - dTdt_ref)
    over = np.flatnonzero(err > 1e-10 * np.abs(dTdt_ref) + 1e-12)
    if over.size == 0:
        return over, np.zeros(0), np.zeros(0)
    kappa = energy_kappa(mech, T[over], wdot_ref[:, over])
    bound = (1e-10 + 1e-14 * kappa) * np.abs(dTdt_ref[over]) + 1e-12
    return over, kappa, err[over] / bound


def longdouble_dTdt(mech, T, P, Y):
    """dT/dt of a few cells in 80-bit extended precision (numpy longdouble through the matrix-form
    restatement below): the arbiter where the fp64 oracle's own rounding is of the size of the
    tolerance.  Returns float64 values rounded from the long-double result."""
    import dataclasses
    L = np.longdouble
    ml = dataclasses.replace(mech, **{
        f.name: getattr(mech, f.name).astype(L) for f in dataclasses.fields(mech)
        if isinstance(getattr(mech, f.name), np.ndarray) and getattr(mech, f.name).dtype == np.float64})
    _, dT = paper_matrix_form(ml, np.asarray(T).astype(L), np.asarray(P).astype(L), np.asarray(Y).astype(L), ru=L(RU))
    return dT


def mp_source_terms(mech, T, P, Y, dps=40):
    """One cell's (wdot[S], dT/dt) at `dps` decimal digits with mpmath, in the PRODUCT form of the paper's
    equations and in the oracle's order of steps (PAPER.md:56 concentrations; Eq. 5 Arrhenius; Eq. 8 Kc;
    PAPER.md:157-159 third bodies, Lindemann / Troe; Eq. 7 k_r = k_f / Kc; Eq. 3 mass action; Eq. 2; the
    constant-pressure energy equation): the arbiter for cells where the fp64 oracle's own rounding is of the
    size of the tolerance (reading Q19).  A third derivation, beside the fp64 C oracle and the
    log-matrix numpy form below; it shares no code with either.  Returns mpmath numbers."""
    from mpmath import mp, mpf, exp, log, log10
    old = mp.dps
    mp.dps = dps
    try:
        S, R = mech.n_species, mech.n_reactions
        Ru = mpf(RU)
        T, P = mpf(float(T)), mpf(float(P))
        W = [mpf(float(x)) for x in mech.mol_weight]
        Yk = [mpf(float(y)) if y > 0 else mpf(0) for y in Y]                      # reading Q9
        inv_Wmix = sum(Yk[k] / W[k] for k in range(S))
        rho = P / (Ru * T * inv_Wmix)
        C = [max(rho * Yk[k] / W[k], mpf("1e-300")) for k in range(S)]
        lnT = log(T)
        cp_R, h_RT, g_RT = [], [], []
        for k in range(S):
            a = [mpf(float(x)) for x in (mech.nasa_lo[k] if float(T) <= mech.T_mid[k] else mech.nasa_hi[k])]
            cp_R.append(a[0] + a[1] * T + a[2] * T**2 + a[3] * T**3 + a[4] * T**4)
            h = a[0] + a[1] * T / 2 + a[2] * T**2 / 3 + a[3] * T**3 / 4 + a[4] * T**4 / 5 + a[5] / T
            s_ = a[0] * lnT + a[1] * T + a[2] * T**2 / 2 + a[3] * T**3 / 3 + a[4] * T**4 / 4 + a[6]
            h_RT.append(h)
            g_RT.append(h - s_)
        arrh = lambda lnA, b, EaR: exp(mpf(float(lnA))) * T**mpf(float(b)) * exp(-mpf(float(EaR)) / T)
        wdot = [mpf(0)] * S
        for j in range(R):
            kf = arrh(mech.ln_A[j], mech.b[j], mech.Ea_over_R[j])
            reac = [(k, mpf(float(mech.nu_reac[k, j]))) for k in np.flatnonzero(mech.nu_reac[:, j])]
            prod = [(k, mpf(float(mech.nu_prod[k, j]))) for k in np.flatnonzero(mech.nu_prod[:, j])]
            dnu_sum = sum(n for _, n in prod) - sum(n for _, n in reac)
            dG = sum(n * g_RT[k] for k, n in prod) - sum(n * g_RT[k] for k, n in reac)
            Kc = exp(-dG) * (mpf(float(mech.p_ref)) / (Ru * T))**dnu_sum
            typ = int(mech.rxn_type[j])
            phi = mpf(1)
            if typ != 0:
                M = sum(mpf(float(mech.eff[k, j])) * C[k] for k in range(S))
                if typ == 1:
                    phi = M
                else:
                    k0 = arrh(mech.ln_A0[j], mech.b0[j], mech.Ea0_over_R[j])
                    Pr = k0 * M / kf
                    F = mpf(1)
                    if typ == 3:
                        al, T3, T1, T2 = (float(x) for x in mech.troe[j])
                        Fc = (1 - mpf(al)) * exp(-T / mpf(T3)) + mpf(al) * exp(-T / mpf(T1))
                        if np.isfinite(T2):
                            Fc += exp(-mpf(T2) / T)
                        lFc = log10(Fc)
                        c = mpf("-0.4") - mpf("0.67") * lFc
                        n = mpf("0.75") - mpf("1.27") * lFc
                        lPr = log10(max(Pr, mpf("1e-300")))
                        f1 = (lPr + c) / (n - mpf("0.14") * (lPr + c))
                        F = mpf(10)**(lFc / (1 + f1 * f1))
                    kf = kf * (Pr / (1 + Pr)) * F
            kr = kf / Kc if mech.reversible[j] else mpf(0)
            qf, qr = kf, kr
            for k, n in reac:
                qf *= C[k]**n
            for k, n in prod:
                qr *= C[k]**n
            Q = phi * (qf - qr)
            for k, n in prod:
                wdot[k] += n * Q
            for k, n in reac:
                wdot[k] -= n * Q
        cp = sum(Yk[k] * cp_R[k] * Ru / W[k] for k in range(S))
        hw = sum(h_RT[k] * Ru * T * wdot[k] for k in range(S))
        return wdot, -hw / (rho * cp)
    finally:
        mp.dps = old


def mp_dTdt(mech, T, P, Y, dps=40):
    """dT/dt of the cells T[n], P[n], Y[S, n] from mp_source_terms, rounded to float64."""
    return np.array([float(mp_source_terms(mech, T[i], P[i], Y[:, i], dps)[1]) for i in range(len(T))])


def energy_condition_number(mech, T, wdot_ref, h_RT):
    """kappa = sum|h_k wdot_k| / |sum h_k wdot_k| per cell."""
    hw = h_RT * RU * T[None, :] * wdot_ref
    return np.abs(hw).sum(0) / np.maximum(np.abs(hw.sum(0)), 1e-300)


def paper_matrix_form(mech, T, P, Y, return_log_rates=False, ru=RU):
    """Literal numpy evaluation of the paper's ANN-form equations, dense matrices,
    batch dimension leading.  Returns (Omega[N,S], dTdt[N]); with
    return_log_rates the arguments of Eq. 4's two exps instead: (ln Q_f[N,R], ln Q_r[N,R]).

    Eq. 6    log Kf = X_f W_f + B_f
    Eq. 10  G = X_G W_G + B_G, alpha from NASA-7 by range
    Eq. 11  log Kc = -(G - log(p_ref/(Ru T))) nu
    Sec 2.4 log M added to log Kf, M = C E; falloff non-matrix
    Eq. 4       Q_net = exp(log C nu' + log Kf) - exp(log C nu'' + log Kr)
    Eq. 2    Omega = Q_net nu^T
    """
    S, R = mech.n_species, mech.n_reactions
    T = np.asarray(T) if np.asarray(T).dtype == np.longdouble else np.asarray(T, dtype=np.float64)
    N = T.shape[0]
    Yc = np.ascontiguousarray(Y.T)                      # [N, S]
    W = mech.mol_weight
    nu1, nu2 = mech.nu_reac, mech.nu_prod               # [S, R]
    nu = nu2 - nu1

    # concentrations
    Wmix = 1.0 / (Yc / W).sum(1)
    rho = P * Wmix / (ru * T)
    C = np.maximum(rho[:, None] * Yc / W, 1e-300)       # [N, S]
    logC = np.log(C)

    # Eq. 6
    X_f = np.stack([np.log(T), 1.0 / T], axis=1)        # [N, 2]
    W_f = np.stack([mech.b, -mech.Ea_over_R], axis=0)   # [2, R]
    logKf = X_f @ W_f + mech.ln_A[None, :]

    # Eq. 10: alpha (7 x S) per temperature range, g/RT = h/RT - s/R collected on X_G
    X_G = np.stack([np.log(T), T, T**2, T**3, T**4, 1.0 / T], axis=1)     # [N, 6]

    def alpha(a):                                       # a: [S, 7] NASA a1..a7
        Wg = np.stack([-a[:, 0], -a[:, 1] / 2, -a[:, 2] / 6, -a[:, 3] / 12, -a[:, 4] / 20,
                       a[:, 5]], axis=0)                # [6, S]
        Bg = a[:, 0] - a[:, 6]                          # [S]
        return Wg, Bg

    Wg_lo, Bg_lo = alpha(mech.nasa_lo)
    Wg_hi, Bg_hi = alpha(mech.nasa_hi)
    low = T[:, None] <= mech.T_mid[None, :]             # [N, S]
    G = np.where(low, X_G @ Wg_lo + Bg_lo, X_G @ Wg_hi + Bg_hi)

    # Eq. 11 with the standard-concentration term in the bias
    logKc = -(G - np.log(mech.p_ref / (ru * T))[:, None]) @ nu            # [N, R]

    # Sec. 2.4: third bodies and falloff
    tb = mech.rxn_type == 1
    fo = (mech.rxn_type == 2) | (mech.rxn_type == 3)
    M = C @ mech.eff                                     # [N, R]
    logKf = logKf + np.where(tb[None, :], np.log(M), 0.0)
    if fo.any():
        W_0 = np.stack([mech.b0, -mech.Ea0_over_R], axis=0)
        logK0 = X_f @ W_0 + mech.ln_A0[None, :]
        Pr = np.exp(logK0 - logKf) * M
        al, T3, T1, T2 = (mech.troe[:, i][None, :] for i in range(4))
        with np.errstate(divide="ignore", invalid="ignore"):
            Fc = (1 - al) * np.exp(-T[:, None] / T3) + al * np.exp(-T[:, None] / T1) \
                + np.exp(-T2 / T[:, None])
            lFc = np.log10(Fc)
            c = -0.4 - 0.67 * lFc
            n = 0.75 - 1.27 * lFc
            lPr = np.log10(np.maximum(Pr, 1e-300))
            f1 = (lPr + c) / (n - 0.14 * (lPr + c))
            logF = np.log(10.0) * lFc / (1 + f1 * f1)
        logF = np.where((mech.rxn_type == 3)[None, :], logF, 0.0)
        logKf = np.where(fo[None, :], logKf + np.log(Pr / (1 + Pr)) + logF, logKf)
    logKr = logKf - logKc                                # Eq. 7 in log space

    if return_log_rates:
        return logC @ nu1 + logKf, logC @ nu2 + logKr
    # Eq. 4 and Eq. 2
    Qf = np.exp(logC @ nu1 + logKf)
    Qr = np.exp(logC @ nu2 + logKr) * mech.reversible[None, :]
    Omega = (Qf - Qr) @ nu.T                             # [N, S]

    # energy equation (north_star step 6)
    def cp_h(a):
        cp = a[:, 0] + X_G[:, 1:2] * a[:, 1] + X_G[:, 2:3] * a[:, 2] + X_G[:, 3:4] * a[:, 3] \
            + X_G[:, 4:5] * a[:, 4]
        h = a[:, 0] + X_G[:, 1:2] * a[:, 1] / 2 + X_G[:, 2:3] * a[:, 2] / 3 \
            + X_G[:, 3:4] * a[:, 3] / 4 + X_G[:, 4:5] * a[:, 4] / 5 + X_G[:, 5:6] * a[:, 5]
        return cp, h
    cp_lo, h_lo = cp_h(mech.nasa_lo)
    cp_hi, h_hi = cp_h(mech.nasa_hi)
    cp_R = np.where(low, cp_lo, cp_hi)
    h_RT = np.where(low, h_lo, h_hi)
    cp_mass = (Yc * cp_R * ru / W).sum(1)
    dTdt = -(h_RT * ru * T[:, None] * Omega).sum(1) / (rho * cp_mass)
    return Omega, dTdt


def tame(mech, seed=0):
    """A copy of a generated mechanism with physically mild kinetics, for tests that follow a
    state in time (input construction only, no kinetics): species enthalpies and entropies
    proportional to their element counts plus a small random part (element-balanced
    reactions then have |ln Kc| of order 10 instead of several hundred), one NASA-7 set for
    both temperature ranges, pre-exponential factors lowered by 1e8 and temperature exponents
    quartered, so that time scales are far longer than 1e-9 s."""
    import dataclasses
    rng = np.random.default_rng(seed)
    S = mech.n_species
    n_el = mech.elem_count.shape[1]
    h_el = rng.uniform(-4000.0, 4000.0, n_el)
    s_el = rng.uniform(5.0, 15.0, n_el)
    nasa = mech.nasa_lo.copy()
    nasa[:, 5] = mech.elem_count @ h_el + rng.uniform(-2000.0, 2000.0, S)
    nasa[:, 6] = mech.elem_count @ s_el + rng.uniform(-2.0, 2.0, S)
    return dataclasses.replace(mech, nasa_lo=nasa, nasa_hi=nasa.copy(),
                               ln_A=mech.ln_A - np.log(1e8), b=mech.b / 4.0,
                               ln_A0=mech.ln_A0 - np.log(1e8), b0=mech.b0 / 4.0)


def ann_forward_matrix_form(ann, T):
    """Eq. 12 literally, batch dimension leading: X_{l+1} = sigma(X_l W_l +
    B_l), standardised input features and de-standardised linear output.
    Returns log Kc~ [N, R]."""
    import ckgen
    act = (lambda z: np.maximum(z, 0.0)) if ann.activation == ckgen.RELU else \
        (lambda z: np.where(z >= 0.0, z, np.expm1(np.minimum(z, 0.0))))
    X = (ckgen.temperature_features(T)[:, :ann.n_in] - ann.in_mean) / ann.in_std
    X = act(X @ ann.W_in + ann.B[0])
    for l in range(1, ann.n_layers):
        X = act(X @ ann.W_hid[l - 1] + ann.B[l])
    return (X @ ann.W_out + ann.B_out) * ann.out_std + ann.out_mean


def exact_layer_as_ann(mech, n_layers=1, activation=1, seed=0):
    """A KcAnn that reproduces the exact equilibrium layer of a mechanism whose two NASA sets
    coincide (input construction from Eq. 10-11 of the paper): Architecture 1
    features pass through the hidden layers unchanged (they are all positive, so relu and elu
    act as the identity; a second hidden layer permutes them) and the output layer carries
    ln Kc_j = -sum_k nu_kj (g_k/RT - ln(p_ref/(Ru T))) on [ln T, T, T^2, T^3, T^4, 1/T].
    Standardisations are non-trivial and undone by the weights."""
    import ckgen
    rng = np.random.default_rng(seed)
    a = mech.nasa_hi
    S, R = mech.n_species, mech.n_reactions
    nu = mech.nu_prod - mech.nu_reac                                     # [S, R]
    # g'_k = g_k/RT - ln(p_ref/(Ru T)) = coef_k . X_G + bias_k
    coef = np.stack([1.0 - a[:, 0], -a[:, 1] / 2, -a[:, 2] / 6, -a[:, 3] / 12, -a[:, 4] / 20, a[:, 5]], axis=0)  # [6, S]
    bias = a[:, 0] - a[:, 6] - np.log(mech.p_ref / RU)                   # [S]
    Wk = -(coef @ nu)                                                    # [6, R]  ln Kc on the features
    bk = -(bias @ nu)                                                    # [R]
    in_mean = rng.uniform(0.5, 2.0, 6) * np.array([7.0, 1e3, 1e6, 1e9, 1e12, 1e-3])
    in_std = rng.uniform(0.5, 2.0, 6) * np.array([0.3, 5e2, 1e6, 1e9, 1e12, 3e-4])
    out_mean, out_std = rng.uniform(-20, 20, R), rng.uniform(1, 10, R)
    W_in, B0 = np.diag(in_std), in_mean.copy()                           # hidden 1 = raw features
    B = np.zeros((n_layers, 6))
    B[0] = B0
    perm = np.arange(6)
    W_hid = np.zeros((n_layers - 1, 6, 6))
    for l in range(n_layers - 1):
        p = rng.permutation(6)
        W_hid[l][np.arange(6), p] = 1.0                                  # neuron `from` -> neuron p[from]
        new = np.empty(6, dtype=int)
        new[p] = perm
        perm = new                                                       # hidden[to] holds feature perm[to]
    W_out = (Wk[perm] / out_std[None, :])
    B_out = (bk - out_mean) / out_std
    return ckgen.KcAnn(n_in=6, n_layers=n_layers, n_hidden=6, activation=activation, in_mean=in_mean,
                       in_std=in_std, W_in=W_in, B=B, W_hid=W_hid, W_out=W_out, B_out=B_out,
                       out_mean=out_mean, out_std=out_std)
