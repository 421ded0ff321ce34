"""Writes tests/golden/jacobian_closed_form.json: derivatives of the single-reaction worked
examples of make_closed_forms.py with respect to
(Y_0, Y_1, T) at constant P, by mpmath's high-order numerical differentiation at 60 digits
(accurate to > 25 digits).  The function differentiated is the 50-digit restatement of the
source-term definition in make_closed_forms.py (Eq. 2, 3, 5, 7, 8 and Sec. 2.4);
this script calls neither oracle/ nor the CUDA library.

Run:  python tests/golden/make_jacobian_closed_form.py
"""
import json
import os
import sys

from mpmath import mp, mpf, diff

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from make_closed_forms import EXAMPLES, single_reaction  # noqa: E402

mp.dps = 60


def outputs(kw, Y0, Y1, T):
    a = dict(kw)
    a["Y"] = [Y0, Y1]
    a["T"] = T
    r = single_reaction(**a)
    return [r["wdot"][0], r["wdot"][1], r["dTdt"]]


def jacobian(kw):
    x0 = [mpf(kw["Y"][0]), mpf(kw["Y"][1]), mpf(kw["T"])]
    J = [[None] * 3 for _ in range(3)]
    for i in range(3):
        for l in range(3):
            def f(v, i=i, l=l):
                x = list(x0)
                x[l] = v
                return outputs(kw, *x)[i]
            J[i][l] = diff(f, x0[l])
    return J


def main():
    out = {"_source": "tests/golden/make_jacobian_closed_form.py (mpmath diff, 60 digits) of the "
                      "single-reaction closed forms of make_closed_forms.py; rows wdot_0, wdot_1, "
                      "dT/dt; columns Y_0, Y_1, T; constant P"}
    # a second state for each case: other mass fractions that do not sum to one (the Jacobian
    # treats the Y_l as independent) and a temperature in the low NASA range is not needed here
    # (constant-cp species), but T = 1350 K moves every exponential
    for name, kw in EXAMPLES.items():
        for tag, over in (("", {}), ("@1350K", {"T": 1350, "Y": ["0.3", "0.6"], "P": 303975})):
            a = dict(kw)
            a.update(over)
            J = jacobian(a)
            out[name + tag] = {"T": str(a["T"]), "P": str(a["P"]), "Y": [str(y) for y in a["Y"]],
                               "J": [[mp.nstr(v, 25) for v in row] for row in J]}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "jacobian_closed_form.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
