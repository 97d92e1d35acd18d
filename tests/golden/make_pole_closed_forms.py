"""Writes the data rows of pole_closed_forms.txt from the closed forms stated in its header
(SURVEY.md 8(c) pin P5), in 30-digit arithmetic (mpmath).  Calls nothing of oracle/ or of the
CUDA path:  python tests/golden/make_pole_closed_forms.py"""
from pathlib import Path

import mpmath as mp

mp.mp.dps = 40
path = Path(__file__).with_name("pole_closed_forms.txt")
header = [ln for ln in path.read_text().splitlines() if ln.startswith("#")]
rows = ["# data: sigma ; l ; Y_l^0 ; d/dx Y_l^{+1} = d/dy Y_l^{-1} ; d/dz Y_l^0 (solid, r = 1)"]
for sigma in (1, -1):
    for l in range(0, 13):
        base = mp.sqrt(mp.mpf(2 * l + 1) / (4 * mp.pi))
        y0 = mp.mpf(sigma) ** l * base
        tang = mp.mpf(sigma) ** (l - 1) * mp.sqrt(mp.mpf((2 * l + 1) * l * (l + 1)) / (8 * mp.pi)) if l else mp.mpf(0)
        dz = l * mp.mpf(sigma) ** (l - 1) * base if l else mp.mpf(0)
        rows.append(f"{sigma:+d} ; {l} ; {mp.nstr(y0, 25)} ; {mp.nstr(tang, 25)} ; {mp.nstr(dz, 25)}")
path.write_text("\n".join([h for h in header if not h.startswith("# data:")] + rows) + "\n")
