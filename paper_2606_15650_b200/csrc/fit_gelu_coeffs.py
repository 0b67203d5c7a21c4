"""Derives the coefficients of gelu2_bf16() in gemm_tcgen05.cu (product-side constant generator; not used at run time,
shares nothing with oracle/).

erf-GELU is gelu(z) = z * Phi(z).  The kernel evaluates Phi(z) as sigma(z * P(z^2)) with P of degree 4 in z^2
(odd argument, so Phi(-z) = 1 - Phi(z) holds exactly).  This script fits P by iteratively re-weighted least squares
towards the minimax of |z| * |sigma(z P(z^2)) - Phi(z)| on [0, 6] and then checks the error on [-12, 12]; the leading
coefficient comes out positive, so the form saturates to 0 / 1 outside the fitted range without a clamp.

    python paper_2606_15650_b200/csrc/fit_gelu_coeffs.py
"""
import numpy as np
from scipy.optimize import least_squares
from scipy.special import ndtr

NTERMS = 5


def model(c, z):
    z2, p = z * z, np.zeros_like(z)
    for k in reversed(range(len(c))):
        p = p * z2 + c[k]
    with np.errstate(over="ignore"):
        return 1.0 / (1.0 + np.exp(-z * p))


def fit():
    z = np.linspace(0.0, 6.0, 6001)
    target = ndtr(z)
    resid = lambda c: (model(c, z) - target) * np.maximum(z, 0.3)
    c = np.zeros(NTERMS)
    c[0], c[1] = 1.5976, 0.07056
    kw = dict(xtol=1e-15, ftol=1e-15, gtol=1e-15)
    c = least_squares(resid, c, **kw).x
    w = np.ones_like(z)
    for _ in range(60):
        e = np.abs(resid(c))
        w = w * (1 + 2 * e / e.max())
        w /= w.mean()
        c = least_squares(lambda cc: resid(cc) * w, c, **kw).x
    return c


if __name__ == "__main__":
    c = fit()
    zz = np.linspace(-12, 12, 400001)
    err = model(c, zz) - ndtr(zz)
    print("coefficients c1, c3, c5, c7, c9 =", [repr(float(x)) for x in c])
    print("max |dPhi| = %.3e   max |z dPhi| = %.3e on [-12, 12]" % (np.abs(err).max(), np.abs(zz * err).max()))
