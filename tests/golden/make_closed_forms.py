"""Writes tests/golden/closed_forms.txt from closed forms only (no oracle, no CUDA).

tree / decoupled chains:  Z = 2^N prod_b cosh(beta J_b)        (any forest of bonds)
single 2x2 plaquette:     Z = 16 cosh^4(beta) (1 + prod_b J_b tanh^4(beta))   (|J_b| = 1)
"""
import math
import os

lines = ["# name beta logZ   (closed forms; see make_closed_forms.py)"]
# 4x4, all Jd = 0, every Jr = +-1: 12 bonds on 4 decoupled chains
for beta in (0.5, 1.0, 2.0):
    lines.append(f"rows4x4 {beta} {16 * math.log(2) + 12 * math.log(math.cosh(beta))!r}")
for beta in (0.5, 1.0, 2.0):
    for name, prod in (("plaq_ferro", 1.0), ("plaq_frustrated", -1.0)):
        z = 16 * math.cosh(beta) ** 4 * (1 + prod * math.tanh(beta) ** 4)
        lines.append(f"{name} {beta} {math.log(z)!r}")
with open(os.path.join(os.path.dirname(__file__), "closed_forms.txt"), "w") as f:
    f.write("\n".join(lines) + "\n")
