"""Writes tests/golden/closed_forms.json: hand-derivable single-reaction worked examples
(plus Ex5: the full NASA-7 set in both temperature ranges),
evaluated at 50 significant digits with mpmath.

This script calls neither oracle/ nor the CUDA library.  Each example is a single
reaction between constant-cp species (NASA a2..a5 = 0), for which every quantity has a
closed form one can type into a calculator:

  g_k/RT = a1 (1 - ln T) + a6/T - a7                 (h/RT = a1 + a6/T, s/R = a1 ln T + a7)
  ln Kc  = -sum_k nu_k g_k/RT + (sum_k nu_k) ln(p_ref/(Ru T))        (Eq. 8)
  k_f    = A T^b exp(-(Ea/R)/T)                                      (Eq. 5)
  q      = k_f prod C^nu' - (k_f/Kc) prod C^nu''                     (Eq. 3)
  1/Wmix = sum Y/W, rho = P Wmix/(Ru T), C = rho Y/W
  three-body: q *= M, M = sum E_k C_k
  falloff (textbook Lindemann/Troe): k_f -> k_inf Pr/(1+Pr) F, Pr = k_0 M/k_inf
  dT/dt  = -sum_k (h_k/RT) Ru T wdot_k / (rho cp),  cp = sum Y_k a1_k Ru/W_k

The values were cross-checked against the numbers printed in SURVEY.md section 8(c)
(an independent 50-digit evaluation); tests/test_oracle_closed_forms.py asserts both.

Run:  python tests/golden/make_closed_forms.py
"""
import json
import os

from mpmath import mp, mpf, exp, log, log10, inf

mp.dps = 50
RU = mpf("8314.46261815324")


def single_reaction(W, a1, a6, a7, nu_r, nu_p, lnA, b, EaR, Y, T, P, p_ref,
                    kind="elementary", E=None, k0=None, troe=None):
    W = [mpf(x) for x in W]; a1 = [mpf(x) for x in a1]; a6 = [mpf(x) for x in a6]
    a7 = [mpf(x) for x in a7]; Y = [mpf(x) for x in Y]
    T = mpf(T); P = mpf(P); p_ref = mpf(p_ref)
    n = len(W)
    g = [a1[k] * (1 - log(T)) + a6[k] / T - a7[k] for k in range(n)]
    h_RT = [a1[k] + a6[k] / T for k in range(n)]
    nu = [mpf(nu_p[k]) - mpf(nu_r[k]) for k in range(n)]
    lnKc = -sum(nu[k] * g[k] for k in range(n)) + sum(nu) * log(p_ref / (RU * T))
    Kc = exp(lnKc)
    kf = exp(mpf(lnA)) * T ** mpf(b) * exp(-mpf(EaR) / T)
    Wmix = 1 / sum(Y[k] / W[k] for k in range(n))
    rho = P * Wmix / (RU * T)
    C = [rho * Y[k] / W[k] for k in range(n)]
    out = {"g_RT": g, "lnKc": lnKc, "Kc": Kc, "k_inf": kf, "rho": rho, "C": C}
    phi = mpf(1)
    if kind != "elementary":
        M = sum(mpf(E[k]) * C[k] for k in range(n))
        out["M"] = M
        if kind == "three_body":
            phi = M
        else:
            Pr = mpf(k0) * M / kf
            F = mpf(1)
            out["Pr"] = Pr
            if kind == "troe":
                alpha, T3, T1, T2 = troe
                Fc = (1 - mpf(alpha)) * exp(-T / mpf(T3)) + mpf(alpha) * exp(-T / mpf(T1))
                if T2 != inf:
                    Fc += exp(-mpf(T2) / T)
                c = mpf("-0.4") - mpf("0.67") * log10(Fc)
                nn = mpf("0.75") - mpf("1.27") * log10(Fc)
                f1 = (log10(Pr) + c) / (nn - mpf("0.14") * (log10(Pr) + c))
                F = mpf(10) ** (log10(Fc) / (1 + f1 * f1))
                out.update({"Fcent": Fc, "c": c, "n": nn, "f1": f1, "F": F})
            kf = kf * Pr / (1 + Pr) * F
    out["kf"] = kf
    qf = kf
    qr = kf / Kc
    for k in range(n):
        qf *= C[k] ** mpf(nu_r[k])
        qr *= C[k] ** mpf(nu_p[k])
    q = phi * (qf - qr)
    wdot = [nu[k] * q for k in range(n)]
    cp = sum(Y[k] * a1[k] * RU / W[k] for k in range(n))
    dTdt = -sum(h_RT[k] * RU * T * wdot[k] for k in range(n)) / (rho * cp)
    out.update({"q": q, "wdot": wdot, "dTdt": dTdt,
                "mass_residual": sum(W[k] * wdot[k] for k in range(n))})
    return out


def nasa7_reaction(W, lo, hi, T_mid, nu_r, nu_p, lnA, b, EaR, Y, T, P, p_ref):
    """One reversible elementary reaction between species with the FULL NASA-7 set (a1..a7 all
    non-zero, a different set below and above T_mid; Eq. 10):
      cp/R = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
      h/RT = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T
      s/R  = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7,   g/RT = h/RT - s/R
    low set for T <= T_mid.  Everything else as in single_reaction()."""
    n = len(W)
    W = [mpf(x) for x in W]; Y = [mpf(x) for x in Y]
    T = mpf(T); P = mpf(P); p_ref = mpf(p_ref)
    a = [[mpf(x) for x in (lo[k] if T <= mpf(T_mid[k]) else hi[k])] for k in range(n)]
    cp_R = [a[k][0] + a[k][1] * T + a[k][2] * T**2 + a[k][3] * T**3 + a[k][4] * T**4 for k in range(n)]
    h_RT = [a[k][0] + a[k][1] * T / 2 + a[k][2] * T**2 / 3 + a[k][3] * T**3 / 4 + a[k][4] * T**4 / 5
            + a[k][5] / T for k in range(n)]
    s_R = [a[k][0] * log(T) + a[k][1] * T + a[k][2] * T**2 / 2 + a[k][3] * T**3 / 3 + a[k][4] * T**4 / 4
           + a[k][6] for k in range(n)]
    g = [h_RT[k] - s_R[k] for k in range(n)]
    nu = [mpf(nu_p[k]) - mpf(nu_r[k]) for k in range(n)]
    lnKc = -sum(nu[k] * g[k] for k in range(n)) + sum(nu) * log(p_ref / (RU * T))
    kf = exp(mpf(lnA)) * T ** mpf(b) * exp(-mpf(EaR) / T)
    Wmix = 1 / sum(Y[k] / W[k] for k in range(n))
    rho = P * Wmix / (RU * T)
    C = [rho * Y[k] / W[k] for k in range(n)]
    qf = kf
    qr = kf / exp(lnKc)
    for k in range(n):
        qf *= C[k] ** mpf(nu_r[k])
        qr *= C[k] ** mpf(nu_p[k])
    q = qf - qr
    wdot = [nu[k] * q for k in range(n)]
    cp = sum(Y[k] * cp_R[k] * RU / W[k] for k in range(n))
    dTdt = -sum(h_RT[k] * RU * T * wdot[k] for k in range(n)) / (rho * cp)
    return {"cp_R": cp_R, "h_RT": h_RT, "s_R": s_R, "g_RT": g, "lnKc": lnKc, "kf": kf, "rho": rho,
            "C": C, "q": q, "wdot": wdot, "cp_mass": cp, "dTdt": dTdt}


def as_json(d):
    f = lambda x: [f(y) for y in x] if isinstance(x, list) else mp.nstr(x, 20)
    return {k: f(v) for k, v in d.items()}


COMMON = dict(T=1000, P=101325, p_ref=101325, lnA=log(mpf("1e10")), b="0.5", EaR=10000)

EXAMPLES = {
    # Ex1  A <=> B
    "ex1_isomerisation": dict(W=[20, 20], a1=["3.5", "3.5"], a6=[0, -5000], a7=[2, 3],
                              nu_r=[1, 0], nu_p=[0, 1], Y=["0.75", "0.25"], **COMMON),
    # Ex2  2A <=> B  (sign and size of the (p_ref/RT)^sum(nu) term)
    "ex2_recombination": dict(W=[20, 40], a1=["3.5", "4.5"], a6=[0, -12000], a7=[2, "1.5"],
                              nu_r=[2, 0], nu_p=[0, 1], Y=["0.75", "0.25"], **COMMON),
    # Ex3  Ex1 as a three-body reaction, E = (2.0, 0.5)
    "ex3_three_body": dict(W=[20, 20], a1=["3.5", "3.5"], a6=[0, -5000], a7=[2, 3],
                           nu_r=[1, 0], nu_p=[0, 1], Y=["0.75", "0.25"], kind="three_body",
                           E=[2, "0.5"], **COMMON),
    # Ex4  Ex1 as falloff, k0 = 1e12, Troe (0.6, 200, 1500, 5000); Lindemann; 3-parameter
    "ex4_troe": dict(W=[20, 20], a1=["3.5", "3.5"], a6=[0, -5000], a7=[2, 3],
                     nu_r=[1, 0], nu_p=[0, 1], Y=["0.75", "0.25"], kind="troe",
                     E=[2, "0.5"], k0="1e12", troe=("0.6", 200, 1500, 5000), **COMMON),
    "ex4_lindemann": dict(W=[20, 20], a1=["3.5", "3.5"], a6=[0, -5000], a7=[2, 3],
                          nu_r=[1, 0], nu_p=[0, 1], Y=["0.75", "0.25"], kind="lindemann",
                          E=[2, "0.5"], k0="1e12", **COMMON),
    "ex4_troe3": dict(W=[20, 20], a1=["3.5", "3.5"], a6=[0, -5000], a7=[2, 3],
                      nu_r=[1, 0], nu_p=[0, 1], Y=["0.75", "0.25"], kind="troe",
                      E=[2, "0.5"], k0="1e12", troe=("0.6", 200, 1500, inf), **COMMON),
}


# Ex5  A + 2 B <=> C with every NASA-7 coefficient non-zero and different low / high sets
# (numbers of the size of real thermodynamic fits), evaluated below and above T_mid = 1000 K.
# Pins the divisors 2, 3, 4, 5 of h and 2, 3, 4 of s and the range switch of the oracle.
NASA_FULL = dict(
    W=[2, 16, 34],
    lo=[["3.2", "1.1e-3", "-2.4e-6", "3.1e-9", "-1.2e-12", "-950", "0.7"],
        ["2.9", "2.4e-3", "-4.1e-6", "2.2e-9", "-0.7e-12", "29100", "4.9"],
        ["4.3", "-0.6e-3", "8.8e-6", "-9.1e-9", "3.2e-12", "-17800", "3.4"]],
    hi=[["3.0", "0.8e-3", "-0.11e-6", "0.02e-9", "-0.002e-12", "-830", "-1.1"],
        ["2.6", "-0.03e-3", "0.05e-6", "-0.01e-9", "0.001e-12", "29200", "4.8"],
        ["4.6", "4.1e-3", "-1.3e-6", "0.21e-9", "-0.012e-12", "-18000", "0.6"]],
    T_mid=[1000, 1000, 1000], nu_r=[1, 2, 0], nu_p=[0, 0, 1], lnA=log(mpf("3e11")), b="-0.7",
    EaR=6500, Y=["0.2", "0.5", "0.3"], P=3 * 101325, p_ref=101325)

# Ex4 again with the Troe factor active far into both pressure limits (Pr ~ 1e-12 and 1e+12):
# k -> k0 M F(Pr -> 0) and k -> k_inf F(Pr -> inf); log10 F -> log10 Fcent / (1 + 1/0.14^2) in
# both limits (f1 -> -1/0.14), so F stays != 1 and a wrong constant of the Troe form shows.
_TROE = dict(W=[20, 20], a1=["3.5", "3.5"], a6=[0, -5000], a7=[2, 3], nu_r=[1, 0], nu_p=[0, 1],
             Y=["0.75", "0.25"], kind="troe", E=[2, "0.5"], troe=("0.6", 200, 1500, 5000), **COMMON)
EXAMPLES["ex4_troe_low_pressure"] = dict(k0="7.25e-4", **_TROE)
EXAMPLES["ex4_troe_high_pressure"] = dict(k0="7.25e20", **_TROE)


def main():
    out = {"_source": "tests/golden/make_closed_forms.py (mpmath, 50 digits); cases from "
                      "SURVEY.md section 8(c) Ex1-Ex4; formulas: PAPER.md Eq. 2, 3, 5, 7, 8"}
    for name, kw in EXAMPLES.items():
        out[name] = as_json(single_reaction(**kw))
    for T in (800, 1000, 1600):      # below, exactly at (low set, reading Q4) and above T_mid
        out["ex5_nasa7_T%d" % T] = as_json(nasa7_reaction(T=T, **NASA_FULL))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "closed_forms.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
