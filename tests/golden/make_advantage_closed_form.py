#!/usr/bin/env python
"""Writes tests/golden/advantage_closed_form.txt: closed-form values of Eq. 1 for binary
rewards, evaluated with 40-digit `decimal` arithmetic.  Calls nothing but the standard library (not the
oracle, not the CUDA path).

    python tests/golden/make_advantage_closed_form.py [--check]

k ones among G rewards in {0, 1}: p = k/G, the population variance is p(1-p), the sample variance (ddof = 1,
DESIGN.md R1) is p(1-p) G/(G-1); A_one = (1-p)/(sigma+eps), A_zero = -p/(sigma+eps) (eps outside the root, R3).
"""
import os
import sys
from decimal import Decimal, getcontext

getcontext().prec = 40
PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "advantage_closed_form.txt")
# (G, k, ddof, eps as written in the file)
CASES = [(8, 4, 0, "0"), (4, 1, 0, "0"), (8, 2, 0, "0"), (16, 8, 1, "0"), (8, 4, 0, "1e-6"), (8, 1, 0, "1e-6"),
         (8, 3, 1, "1e-6"), (16, 5, 0, "1e-6")]
HEADER = """\
# Closed-form values of Eq. 1 (PAPER.md:86-90) for binary rewards: k ones among G.
# p = k/G; sigma = sqrt(p(1-p)) * (sqrt(G/(G-1)) if ddof==1 else 1)   [DESIGN.md reading R1]
# A_one = (1-p)/(sigma+eps); A_zero = -p/(sigma+eps).  Evaluated with 40-digit decimal arithmetic
# (python `decimal`, not the oracle).  Columns: G k ddof eps A_one A_zero
"""


def fmt(x: Decimal) -> str:
    return f"{x:.17E}"


def lines():
    out = []
    for G, k, ddof, eps in CASES:
        p = Decimal(k) / Decimal(G)
        var = p * (1 - p)
        if ddof == 1:
            var = var * Decimal(G) / Decimal(G - 1)
        sigma = var.sqrt()
        den = sigma + Decimal(eps)
        out.append(f"{G} {k} {ddof} {eps} {fmt((1 - p) / den)} {fmt(-p / den)}")
    return out


def main():
    text = HEADER + "\n".join(lines()) + "\n"
    if "--check" in sys.argv:
        with open(PATH) as f:
            ok = f.read() == text
        print("advantage_closed_form.txt", "matches" if ok else "DIFFERS")
        return 0 if ok else 1
    with open(PATH, "w") as f:
        f.write(text)
    return 0


if __name__ == "__main__":
    sys.exit(main())
