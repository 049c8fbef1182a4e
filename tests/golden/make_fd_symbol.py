"""Writes fd_symbol.txt: lambda_n(theta) = c_0 + 2 sum_{k=1..n} c_k cos(k theta) with the c_k taken as
exact rationals from fd_coeffs.txt (reading S10).  Uses only the Python standard library."""
import math
import os
from fractions import Fraction

here = os.path.dirname(os.path.abspath(__file__))
rows = {}
for line in open(os.path.join(here, "fd_coeffs.txt")):
    if line.startswith("#") or not line.strip():
        continue
    n, rest = line.split(":")
    rows[int(n)] = [Fraction(t) for t in rest.split()]
with open(os.path.join(here, "fd_symbol.txt"), "w") as f:
    f.write("# n theta_name value ; written by make_fd_symbol.py\n")
    for n, c in rows.items():
        for name, th in (("pi/8", math.pi / 8), ("pi/2", math.pi / 2), ("pi", math.pi)):
            val = math.fsum([float(c[0])] + [2.0 * float(c[k]) * math.cos(k * th) for k in range(1, n + 1)])
            f.write(f"{n} {name} {val!r}\n")
