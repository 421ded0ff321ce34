"""Writes tests/golden/reactor_closed_form.json: the explicit RK4 step of the constant-
pressure reactor on a case where it has a closed form, at 50 digits with mpmath.

Calls neither oracle/ nor the CUDA library.

Case: A <=> B, W_A = W_B = 20 kg/kmol, both species cp/R = 3.5 and the same enthalpy
(a6 = 0: thermoneutral, so dT/dt = 0 and rho is constant), s_B - s_A = R (a7 = 2, 3), so
Kc = e; k_f = 1e10 T^0.5 exp(-1e4/T) at T = 1000 K (Eq. 5), k_r = k_f / Kc
(Eq. 7).  With C_k = rho Y_k / W the reactor equation
    dY_A/dt = W wdot_A / rho = -(k_f Y_A - k_r Y_B),   Y_B = 1 - Y_A
is linear: d(Y_A - Y*)/dt = -(k_f + k_r)(Y_A - Y*), Y* = k_r / (k_f + k_r).  One step of
the classic 4-stage Runge-Kutta scheme multiplies Y_A - Y* by its stability polynomial
    R(z) = 1 + z + z^2/2 + z^3/6 + z^4/24,   z = -(k_f + k_r) dt
exactly (any wrong stage coefficient or weight changes a coefficient of R), while the
exact flow multiplies it by e^z.

Run:  python tests/golden/make_reactor_closed_form.py
"""
import json
import os

from mpmath import mp, mpf, exp

mp.dps = 50


def main():
    T = mpf(1000)
    kf = mpf("1e10") * T ** mpf("0.5") * exp(-mpf(10000) / T)
    kr = kf / exp(mpf(1))
    y_eq = kr / (kf + kr)
    out = {"_source": "tests/golden/make_reactor_closed_form.py (mpmath, 50 digits); "
                      "PAPER.md Eq. 5, 7, 8; classic RK4 stability polynomial",
           "kf": mp.nstr(kf, 20), "kr": mp.nstr(kr, 20), "Y_A_eq": mp.nstr(y_eq, 20), "cases": []}
    for dt in ("1e-9", "2e-8", "5e-8"):   # projection inactive: every stage keeps Y > 0
        z = -(kf + kr) * mpf(dt)
        R = 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24
        y = mpf("0.75")
        ys = []
        for _ in range(3):
            y = y_eq + R * (y - y_eq)
            ys.append(mp.nstr(y, 20))
        out["cases"].append({"dt": dt, "z": mp.nstr(z, 20), "R": mp.nstr(R, 20),
                             "exp_z": mp.nstr(exp(z), 20), "Y_A_after_steps_1_2_3": ys})
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "reactor_closed_form.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
