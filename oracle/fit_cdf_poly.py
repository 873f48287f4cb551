"""Derivation of the frozen CDF-contract coefficients (reading R-6).

TEST INFRASTRUCTURE ONLY.  The paper's GPU flavour approximates "the cumulative density of the Gaussian
distribution" by a polynomial but gives no coefficients.  The contract used by the oracle
(pv_oracle.c, PVO_G) is: support +-U sigma with U = 3, F(u) = 1/2 + s G(s^2), s = u / U, G of degree 6
(an odd degree-13 polynomial in s), least-squares fitted on 4000 Chebyshev nodes to the truncated,
renormalised Gaussian CDF  (Phi(u) - Phi(-U)) / (1 - 2 Phi(-U)) - 1/2,  converted to monomials and rounded
to fp32.  This script recomputes the seven numbers; tests/test_oracle_fill.py checks that they equal the
literals frozen in pv_oracle.c.  Run: python -m oracle.fit_cdf_poly
"""
import numpy as np
from numpy.polynomial import chebyshev as Ch
from scipy.special import ndtr

U = 3.0
N_NODES = 4000
N_COEF = 7


def fit() -> np.ndarray:
    k = np.arange(N_NODES)
    s = np.cos(np.pi * (k + 0.5) / N_NODES)
    tail = ndtr(-U)
    target = (ndtr(U * s) - tail) / (1.0 - 2.0 * tail) - 0.5
    basis = np.stack([Ch.chebval(s, [0.0] * (2 * j + 1) + [1.0]) for j in range(N_COEF)], axis=1)
    c, *_ = np.linalg.lstsq(basis, target, rcond=None)
    cheb = np.zeros(2 * N_COEF)
    cheb[1::2] = c
    return Ch.cheb2poly(cheb)[1::2].astype(np.float32)


if __name__ == "__main__":
    for v in fit():
        print(float(v).hex(), float(v))
