"""Writes tests/golden/eigenvalues_d.txt: d_k = 4 (n+1)^2 sin^2(pi k / (2 (n+1))) for a few
(n, k), evaluated with Python's `decimal` at 60 digits from the Taylor series of sin -- no numpy,
no oracle code.  Source of the formula: PAPER.md:198-200 (lambda_k = 2(1 - cos(pi k/(n+1))),
h = 1/(n+1)) in the cancellation-free form 4 sin^2(theta/2) (reading Q1).

Run:  python tests/golden/make_eigenvalues_golden.py
"""
from decimal import Decimal, getcontext
import os

getcontext().prec = 60
PI = Decimal("3.14159265358979323846264338327950288419716939937510582097494")


def dsin(x: Decimal) -> Decimal:
    term = x
    total = x
    i = 1
    while abs(term) > Decimal(10) ** -58:
        term = -term * x * x / ((2 * i) * (2 * i + 1))
        total += term
        i += 1
    return total


def main():
    rows = []
    for p in (8, 12, 16, 20, 22):
        N = 1 << p
        n = N - 1
        for k in (1, 2, 3, 17, N // 4, N // 2, n - 1, n):
            theta_half = PI * k / (2 * N)
            s = dsin(theta_half)
            d = 4 * Decimal(N) * Decimal(N) * s * s
            rows.append(f"{n} {k} {d:.30E}")
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "eigenvalues_d.txt")
    with open(path, "w") as f:
        f.write("# n k d_k=4(n+1)^2 sin^2(pi k/(2(n+1)))  [PAPER.md:198-200, 213; 60-digit decimal Taylor series]\n")
        f.write("\n".join(rows) + "\n")


if __name__ == "__main__":
    main()
