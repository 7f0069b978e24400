"""Writes tests/golden/hyperbolic_closed_forms.txt from closed forms only (no oracle, no CUDA path).

Field B = (k x, -k y, 1), k = 2, box [-1,1]^2 x [0,1], seed (x0, y0, 0)  (BASELINE.json configs[0]; north_star:
"the hyperbolic field B = (k x, -k y, 1) maps z=0 -> z=h with Q = e^{2kh} + e^{-2kh} and L known in closed form").
Field line: x = x0 e^{kz}, y = y0 e^{-kz}.  Columns: x0 y0 endx endy endz L q_bnd q_perp.
  top exit (|x0| <= e^-k):  end = (x0 e^k, y0 e^-k, 1),  q_bnd = e^{2k} + e^{-2k}
  side exit:                z* = ln(1/|x0|)/k, end = (sgn x0, y0 |x0|, z*), q_bnd = k (x0^2 + y0^2) + 1/(k x0^2)
  L = int_0^{z*} sqrt(1 + k^2 x0^2 e^{2kz} + k^2 y0^2 e^{-2kz}) dz   (scipy.integrate.quad, 1e-13)
  q_perp = (m_F/m_0)(|P D a|^2 + |P D b|^2), eq. (11) of the paper with a zero-length backward
  end, D = d(end)/d(seed) of the analytic line, P = I - u_F u_F^T, (a, b) the basis of DESIGN.md reading A7.
Run: python tests/golden/make_golden.py
"""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))
from tests.test_oracle_pins import P2_SEEDS, _closed_forms  # noqa: E402

if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "hyperbolic_closed_forms.txt")
    with open(out, "w") as f:
        f.write("# closed forms for B=(2x,-2y,1) on [-1,1]^2x[0,1], seeds on z=0; see make_golden.py for the formulas\n")
        f.write("# x0 y0 endx endy endz L q_bnd q_perp\n")
        for x0, y0 in P2_SEEDS:
            end, L, qb, qp = _closed_forms(x0, y0)
            f.write(" ".join(repr(float(v)) for v in (x0, y0, *end, L, qb, qp)) + "\n")
    print("wrote", out)
