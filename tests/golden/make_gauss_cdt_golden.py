#!/usr/bin/env python
"""Writes tests/golden/gauss_cdt_table1.txt: the 24-entry 16-bit cumulative table of O12 (S21)

    C[j] = floor(65536 * Phi((j - 12 + 1/2) / sigma) + 1/2),  j = 0..23,

for the four Gaussian widths of the paper's Table 1 (sigma = 2.3, 1.7, 1.2, 1.0), computed with the
standard library only (`decimal`, 60 significant digits) from the everywhere-convergent series

    Phi(x) = 1/2 + phi(x) * sum_{n >= 0} x^(2n+1) / (2n+1)!!,   phi(x) = exp(-x^2/2) / sqrt(2 pi).

It calls nothing of oracle/ or of the CUDA path: the file pins the INTEGER table both sides must produce (both
evaluate the formula in double with libm's erfc, so a shared rounding accident would otherwise go unseen).  The
script also reports the distance of every 65536*Phi + 1/2 from the nearest integer, i.e. how far each entry is
from flipping; the smallest is written into the file's header.

    python tests/golden/make_gauss_cdt_golden.py
"""
from decimal import Decimal, getcontext
from pathlib import Path

getcontext().prec = 60
SIGMAS = ["1.0", "1.2", "1.7", "2.3"]
TAU = 12


def pi_dec() -> Decimal:
    # Machin: pi = 16 atan(1/5) - 4 atan(1/239)
    def atan_inv(n: int) -> Decimal:
        x = Decimal(1) / n
        x2, term, total, k = x * x, x, x, 1
        while abs(term) > Decimal(10) ** -70:
            term = -term * x2
            k += 2
            total += term / k
        return total
    return 16 * atan_inv(5) - 4 * atan_inv(239)


def Phi(x: Decimal) -> Decimal:
    phi = (-(x * x) / 2).exp() / (2 * pi_dec()).sqrt()
    term, total, n = x, x, 0
    while abs(term) > Decimal(10) ** -70:
        n += 1
        term = term * x * x / (2 * n + 1)
        total += term
    return Decimal(1) / 2 + phi * total


def main():
    lines = ["# 16-bit CDT of the rounded Gaussian (O12 / DESIGN.md S21) for Table 1's sigmas (P:L94-102).",
             "# Written by tests/golden/make_gauss_cdt_golden.py (python `decimal`, 60 digits; no oracle, no CUDA).",
             "# sigma_<value> = C[0] ... C[23]"]
    margin = Decimal(1)
    body = []
    for sg in SIGMAS:
        sigma = Decimal(sg)
        row = []
        for j in range(2 * TAU):
            y = 65536 * Phi((Decimal(j) - TAU + Decimal(1) / 2) / sigma) + Decimal(1) / 2
            c = int(y.to_integral_value(rounding="ROUND_FLOOR"))
            frac = y - c
            margin = min(margin, frac, 1 - frac)
            row.append(c)
        body.append(f"sigma_{sg} = " + " ".join(map(str, row)))
    lines.append(f"# smallest distance of 65536*Phi + 1/2 from an integer over all entries: {margin:.3E} "
                 "(double evaluation errs by ~1e-11: no entry can flip)")
    out = Path(__file__).resolve().parent / "gauss_cdt_table1.txt"
    out.write_text("\n".join(lines + body) + "\n")
    print(out.read_text())


if __name__ == "__main__":
    main()
