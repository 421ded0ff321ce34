"""Writes tests/golden/ann_closed_form.json: one worked example of the approximate ANN for
log Kc (Eq. 12-14, Architecture 2) inside the single-reaction closed form
Ex1 of make_closed_forms.py, at 50 digits with mpmath.  Calls neither oracle/ nor the CUDA
library.

Network: input x0 = (ln T - 7) / 0.5; two hidden layers of two neurons,
  z1 = x0 * [0.8, -1.5] + [0.1, 0.2],            h1 = sigma(z1)
  z2 = h1 @ [[0.5, -2.0], [1.5, 0.25]] + [-0.3, 0.4],  h2 = sigma(z2)     (row = from, column = to)
  y  = h2 @ [1.25, -0.75] + 0.5,                  ln Kc~ = 3 y + 4.
At T = 1000 K x0 < 0, so pre-activations of both signs occur: elu and relu differ.
Then A <=> B as in Ex1 with Kc replaced by Kc~ (Eq. 7): q = k_f (C_A - C_B / Kc~).

Run:  python tests/golden/make_ann_closed_form.py
"""
import json
import os

from mpmath import mp, mpf, exp, log

mp.dps = 50
RU = mpf("8314.46261815324")


def sigma(kind, z):
    if kind == "relu":
        return z if z > 0 else mpf(0)
    return z if z >= 0 else exp(z) - 1


def main():
    T, P = mpf(1000), mpf(101325)
    out = {"_source": "tests/golden/make_ann_closed_form.py (mpmath, 50 digits); PAPER.md Eq. 12-14, 7, 5, 3"}
    for kind in ("elu", "relu"):
        x0 = (log(T) - 7) / mpf("0.5")
        z1 = [x0 * mpf("0.8") + mpf("0.1"), x0 * mpf("-1.5") + mpf("0.2")]
        h1 = [sigma(kind, z) for z in z1]
        W2 = [[mpf("0.5"), mpf("-2.0")], [mpf("1.5"), mpf("0.25")]]
        z2 = [h1[0] * W2[0][0] + h1[1] * W2[1][0] - mpf("0.3"), h1[0] * W2[0][1] + h1[1] * W2[1][1] + mpf("0.4")]
        h2 = [sigma(kind, z) for z in z2]
        y = h2[0] * mpf("1.25") + h2[1] * mpf("-0.75") + mpf("0.5")
        lnKc = 3 * y + 4
        kf = mpf("1e10") * T ** mpf("0.5") * exp(-mpf(10000) / T)
        Y = [mpf("0.75"), mpf("0.25")]
        W = mpf(20)
        rho = P * W / (RU * T)
        C = [rho * y_ / W for y_ in Y]
        q = kf * (C[0] - C[1] / exp(lnKc))
        # thermo of Ex1: cp/R = 3.5 both, h/RT = 3.5 + a6/T with a6 = (0, -5000)
        cp = mpf("3.5") * RU / W
        dTdt = -((mpf("3.5")) * RU * T * (-q) + (mpf("3.5") - 5) * RU * T * q) / (rho * cp)
        out[kind] = {"x0": mp.nstr(x0, 20), "z1": [mp.nstr(z, 20) for z in z1], "z2": [mp.nstr(z, 20) for z in z2],
                     "lnKc": mp.nstr(lnKc, 20), "q": mp.nstr(q, 20), "dTdt": mp.nstr(dTdt, 20)}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "ann_closed_form.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
