"""Writes chirp_constants.txt: phase pi*(dx^2+dy^2)*pitch^2/(lambda z) for a few integer offsets,
reduced mod 2 pi, with 50-digit decimal arithmetic (standard library only)."""
from decimal import Decimal, getcontext
import os

getcontext().prec = 60
PI = Decimal("3.14159265358979323846264338327950288419716939937510582097494")
lam, pitch, z = Decimal("785e-9"), Decimal("20e-6"), Decimal("0.2")
rows = ["# dx dy phase_mod_2pi   (q = exp(+i*phase); Eq.1 PAPER.md:33-37, sign per BASELINE.json north_star)"]
for dx, dy in [(0, 0), (1, 0), (0, 1), (-1, 0), (3, -4), (-128, 127), (511, -512), (-1024, 1023)]:
    ph = PI * (Decimal(dx * dx + dy * dy)) * pitch * pitch / (lam * z)
    ph = ph - (ph / (2 * PI)).to_integral_value(rounding="ROUND_FLOOR") * 2 * PI
    rows.append(f"{dx} {dy} {ph:.30f}")
with open(os.path.join(os.path.dirname(__file__), "chirp_constants.txt"), "w") as fh:
    fh.write("\n".join(rows) + "\n")
