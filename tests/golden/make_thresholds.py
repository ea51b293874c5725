"""Writes the threshold rows of tests/golden/thresholds.txt with 50-digit decimal arithmetic.

Independent of oracle/ and of the CUDA path: T = floor(scale * exp(-beta*dE)), scale = 2^32 (Philox, rng_mode 0)
or 2^31-1 (MINSTD, rng_mode 1), beta = num/den as an exact rational.  Run: python tests/golden/make_thresholds.py
"""
import os
from decimal import Decimal, getcontext

getcontext().prec = 50
HERE = os.path.dirname(os.path.abspath(__file__))
BETAS = [(10, 11), (10, 7), (0, 1), (1, 2), (3, 10), (1, 10), (2, 1), (50, 1)]


def rows():
    for mode, scale in ((0, Decimal(2) ** 32), (1, Decimal(2) ** 31 - 1)):
        for num, den in BETAS:
            beta = Decimal(num) / Decimal(den)
            T = [int((scale * (-(beta * dE)).exp()).to_integral_value(rounding="ROUND_FLOOR")) for dE in (4, 8, 12)]
            yield f"{mode} {num} {den} {T[0]} {T[1]} {T[2]}"


if __name__ == "__main__":
    path = os.path.join(HERE, "thresholds.txt")
    head = [l for l in open(path).read().splitlines() if l.startswith("#")]
    with open(path, "w") as f:
        f.write("\n".join(head + list(rows())) + "\n")
