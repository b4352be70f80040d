"""Writes the rows of moving_charge.txt from the closed form in its header, using python's
`decimal` at 50 digits (independent of oracle/ and of the CUDA path).  Run:
    python tests/golden/make_moving_charge.py >> tests/golden/moving_charge.txt
"""
from decimal import Decimal as D, getcontext

getcontext().prec = 50
PI = D("3.14159265358979323846264338327950288419716939937510")
Q = D("-1.602176634e-19")
EPS0 = D("8.8541878128e-12")
C0 = D("299792458")

CASES = [("10", "1e-3", "-2e-3", "3e-4"), ("50", "2e-4", "1e-4", "-1e-5"),
         ("1.5", "0.3", "0.1", "0.2"), ("100", "1e-3", "0", "1e-6"), ("30", "0", "5e-4", "2e-4")]

for g, rx, ry, rz in CASES:
    g, rx, ry, rz = D(g), D(rx), D(ry), D(rz)
    den = (rx * rx + ry * ry + g * g * rz * rz)
    den = den * den.sqrt()
    k = Q / (4 * PI * EPS0) * g / den
    ex, ey, ez = k * rx, k * ry, k * rz
    beta = (1 - 1 / (g * g)).sqrt()
    bx, by, bz = -beta * ey / C0, beta * ex / C0, D(0)
    print(" ".join(f"{float(v):.17e}" for v in (g, rx, ry, rz, ex, ey, ez, bx, by, bz)))
