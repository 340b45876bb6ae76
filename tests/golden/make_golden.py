"""Writes tests/golden/oracle_n8.txt.  Calls only oracle/ (never the CUDA path).

Run from the repo root:  python tests/golden/make_golden.py
The stored case is form D (the definition) on an 8x8 ramp; test_oracle_pins.py reloads it as
a regression guard on the oracle's arithmetic."""
import pathlib
import sys

import numpy as np

sys.path.insert(0, str(pathlib.Path(__file__).resolve().parents[2]))
from oracle import shifted_fresnel as O  # noqa: E402

u0 = np.arange(64, dtype=np.float64).reshape(8, 8) / 63.0
u1 = O.direct_sum(u0, 632.8e-9, 0.002, 4.65e-6, 2.0e-6, O1=(3e-6, -2e-6))
out = pathlib.Path(__file__).with_name("oracle_n8.txt")
np.savetxt(out, np.stack([u1.real.ravel(), u1.imag.ravel()], axis=1), fmt="%.17e",
           header="form D, N=8, u0=ramp/63, lambda=632.8e-9, z=2e-3, p0=4.65e-6, p1=2e-6, "
                  "O1=(3e-6,-2e-6); columns: re im, row-major [n1][m1]")
print("wrote", out)
