"""Writes tests/golden/dpie_golden.txt.  Calls only oracle/ (Form Q quadrature, mpmath, 40 digits).

The cases (lenses L1..L4, pixels) are those SURVEY.md 8(c) pin 1 proposes; the VALUES are regenerated here from the
definition-by-quadrature (oracle/form_q.py), not copied: the survey's table (computed at survey time from the
complex-log form) is kept in the last two columns only as an independent cross-check, and this script fails if the
two disagree beyond 1e-18 (the table prints 20 digits).  Not from the paper (the paper prints no gradient value).

    python tests/golden/make_golden.py
"""
import os
import sys

import mpmath as mp

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))
from oracle import form_q  # noqa: E402

mp.mp.dps = 40

L = {
    "L1": (1.5, -0.75, 0.3, 0.5, 0.25, 20.0, 4.0),
    "L2": (0.0, 0.0, 0.0, 0.0, 0.5, 30.0, 2.0),
    "L3": (-10.0, 5.0, 1e-6, 2.5, 0.05, 10.0, 7.0),
    "L4": (2.0, 3.0, 0.6, 1.25, 8.0, 800.0, 25.0),
}
CASES = [
    ("L1", (4.0, 2.0), "1.6270970858737468782", "2.4988079578139617908"),
    ("L1", (1.51, -0.73), "0.026620775633982545205", "0.16538707205496459025"),
    ("L1", (-60.0, 35.0), "-0.72894909093990482944", "0.47422135806004960738"),
    ("L2", (3.0, 4.0), "1.0033932591626880057", "1.3378576788835840076"),
    ("L3", (-9.5, 5.25), "5.5790155599188464345", "2.789511765941331946"),
    ("L3", (-10.001, 5.002), "-0.069964705282291245163", "0.13992969117616329204"),
    ("L4", (-40.0, 55.0), "-14.526077044994419609", "9.6873737652113731799"),
    ("L4", (2.5, 2.5), "1.4255963501181430133", "-0.68150270584961467259"),
    ("L1+L2+L3+L4", (4.0, 2.0), "11.157988886150978416", "0.75874550803859845931"),
]


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "dpie_golden.txt")
    lines = ["# dPIE deflection golden values: oracle/form_q.py (1-D quadrature of the surface density, eq. 2-4 P:60-66),",
             "# mpmath 40 digits; written by tests/golden/make_golden.py; NOT from the paper (it prints none).",
             "# lens rows: name xc yc ellipticity angle rcore rcut b0", ]
    for k, v in L.items():
        lines.append("lens %s %s" % (k, " ".join(repr(x) for x in v)))
    lines.append("# case rows: lenses theta1 theta2 gradPsi1 gradPsi2")
    for names, (t1, t2), s1, s2 in CASES:
        lenses = [L[n] for n in names.split("+")]
        g1, g2 = form_q.gradient_point(lenses, t1, t2)
        # cross-check against the survey table with the DECIMAL parameters it was computed from (repr of the
        # fp64 value = the decimal literal); the stored values use the fp64 inputs the C++ oracle receives.
        dec = [tuple(mp.mpf(repr(x)) for x in row) for row in lenses]
        h1, h2 = form_q.gradient_point(dec, mp.mpf(repr(t1)), mp.mpf(repr(t2)))
        d = max(abs(h1 - mp.mpf(s1)), abs(h2 - mp.mpf(s2)))
        print(names, t1, t2, mp.nstr(g1, 25), mp.nstr(g2, 25), "diff vs survey table", mp.nstr(d, 3))
        assert d < mp.mpf(10) ** -18, "quadrature disagrees with the survey-time complex-log value"
        lines.append("case %s %r %r %s %s" % (names, t1, t2, mp.nstr(g1, 25), mp.nstr(g2, 25)))
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
