"""Writes tests/golden/tfim_ring_ground_energy.json from the closed form only (no oracle,
no CUDA path): ground energy of the periodic transverse-field Ising ring
H = -sum Z_l Z_{l+1} - h sum X_l (Eq. 41), solved by fermionisation
(PAPER.md:588, ref. [66] Pfeuty 1970, :851).  In the even-parity sector
  E0 = -sum_{m=0}^{N-1} sqrt(1 + h^2 - 2 h cos((2m+1) pi / N)),
which at h = 1 collapses to  E0 = -2 / sin(pi / (2N))  (sum of 2 sin((2m+1) pi / 2N)).
Run:  python tests/golden/make_tfim_golden.py
"""
import json
import math
import os

cases = []
for N, h in [(8, 1.0), (10, 0.75), (6, 3.0), (12, 1.0)]:
    e0 = -sum(math.sqrt(1 + h * h - 2 * h * math.cos((2 * m + 1) * math.pi / N)) for m in range(N))
    if h == 1.0:
        assert abs(e0 + 2 / math.sin(math.pi / (2 * N))) < 1e-12
    cases.append({"N": N, "h": h, "E0": round(e0, 12)})
out = {"source": "closed form, PAPER.md:588 ref [66]; written by tests/golden/make_tfim_golden.py", "cases": cases}
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "tfim_ring_ground_energy.json"), "w") as f:
    json.dump(out, f, indent=1)
print(out)
