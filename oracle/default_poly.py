"""Re-derivation of the default grid-force-fit coefficients (reading R4).

ORACLE-SIDE test infrastructure.  PAPER.md:65 only says that spectral filtering sets a
"hand-over" between the PM and the short-range solver; it prints no filter and no fit.
Reading R4: the subtracted grid force is a degree-5 polynomial in s = r^2 whose six fp32
coefficients are a RUNTIME INPUT; the DEFAULT set is the constrained least-squares fit, on
s in [0, rc^2] = [0, 9], to the force of a Gaussian-filtered point mass

    g(s) = [erf(r/sg) - (2 r / (sg sqrt(pi))) exp(-r^2/sg^2)] / r^3,   sg = 1.2,

with P(rc^2) = rc^-3 imposed, following Appendix A step by step:
  nodes    s_k = (9/2)(1 - cos(pi (k + 1/2) / 4096)),  k = 0..4095
  basis    phi_j(s) = (s - 9) T_j(t),  t = 2 s / 9 - 1,  j = 0..4   (Chebyshev T_j)
  solve    sum_j q_j phi_j(s_k) ~= g(s_k) - 1/27         (least squares)
  expand   P(s) = 1/27 + (s - 9) sum_j q_j T_j(t)  to monomials in s, in fp64
  round    each c_k to fp32

Run as a script to print the table; tests/test_oracle_pins.py::test_p10 compares the
rounded bit patterns with Appendix A's.
"""
from __future__ import annotations

import math

import numpy as np
from numpy.polynomial import chebyshev as cheb
from numpy.polynomial import polynomial as npoly

RC2 = 9.0
SIGMA_G = 1.2
NODES = 4096


def gauss_filtered_force(s: np.ndarray, sigma: float = SIGMA_G) -> np.ndarray:
    """g(s): radial force factor of a Gaussian-smoothed unit point mass (force = g * d)."""
    s = np.asarray(s, dtype=np.float64)
    x2 = s / (sigma * sigma)
    out = np.empty_like(s)
    small = x2 < 0.25
    # series: h(x)/x^3 = (4/sqrt(pi)) sum_n (-1)^n x^(2n) / (n! (2n+3)),  h = erf(x) - 2x/sqrt(pi) e^{-x^2}
    acc = np.zeros_like(s[small])
    term = np.ones_like(acc)
    for n in range(0, 30):
        acc += term / (2 * n + 3)
        term = term * (-x2[small]) / (n + 1)
    out[small] = 4.0 / math.sqrt(math.pi) * acc / sigma ** 3
    r = np.sqrt(s[~small])
    x = r / sigma
    erf = np.array([math.erf(v) for v in x])
    out[~small] = (erf - 2.0 * x / math.sqrt(math.pi) * np.exp(-x * x)) / r ** 3
    return out


def derive(sigma: float = SIGMA_G, rc2: float = RC2, nodes: int = NODES):
    """Returns (c64[6], c32[6], q[5]) following Appendix A."""
    k = np.arange(nodes, dtype=np.float64)
    s = 0.5 * rc2 * (1.0 - np.cos(math.pi * (k + 0.5) / nodes))
    t = 2.0 * s / rc2 - 1.0
    A = np.stack([(s - rc2) * cheb.chebval(t, [0] * j + [1]) for j in range(5)], axis=1)
    rhs = gauss_filtered_force(s, sigma) - rc2 ** -1.5
    q, *_ = np.linalg.lstsq(A, rhs, rcond=None)
    # sum_j q_j T_j(t) as a power series in t, then in s (t = 2 s / rc2 - 1)
    pt = cheb.cheb2poly(q)                      # coefficients in t
    ps = np.zeros(1)
    lin = np.array([-1.0, 2.0 / rc2])           # t as a polynomial in s
    for c in pt[::-1]:                          # Horner in the polynomial ring
        ps = npoly.polyadd(npoly.polymul(ps, lin), [c])
    full = npoly.polymul(ps, [-rc2, 1.0])       # times (s - rc2)
    full = npoly.polyadd(full, [rc2 ** -1.5])
    c64 = np.zeros(6)
    c64[: full.size] = full
    return c64, c64.astype(np.float32), q


if __name__ == "__main__":
    c64, c32, q = derive()
    print("q =", ", ".join("%.15f" % v for v in q))
    for i in range(6):
        print("c%d  %.12e  %.9e  0x%08X" % (i, c64[i], c32[i], int(c32[i : i + 1].view(np.uint32)[0])))
    sgrid = np.linspace(0.0, RC2, 20001)
    P = npoly.polyval(sgrid, c32.astype(np.float64))
    print("max |P - g| on [0,9] = %.3e" % np.max(np.abs(P - gauss_filtered_force(sgrid))))
    print("P(9) - 1/27 = %.3e" % (npoly.polyval(9.0, c32.astype(np.float64)) - 1.0 / 27.0))
