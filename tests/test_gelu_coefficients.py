"""The BF16 FFN1 epilogue evaluates the erf-GELU (reading D3) as z * sigma(z * P(z^2)) with a fitted degree-4 P
(csrc/gemm_tcgen05.cu, gelu2_f32; provenance: csrc/fit_gelu_coeffs.py).  This test reads the five coefficients out of the
kernel source and checks, in float64 against scipy's erf, the bound DESIGN.md states: |gelu_fit(z) - gelu(z)| <= 3.1e-6 for
every z, on a dense grid over [-12, 12] (beyond that both sides are 0 or z to double precision)."""
import os
import re

import numpy as np
from scipy.special import erf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_gelu_polynomial_matches_erf_form():
    src = open(os.path.join(ROOT, "paper_2606_15650_b200", "csrc", "gemm_tcgen05.cu")).read()
    body = src[src.index("gelu2_f32(uint64_t z)"):]
    body = body[:body.index("const uint64_t z2")]
    coef = [float(m) for m in re.findall(r"pk2\(kL \* (-?[0-9.e+-]+)f,", body)]
    assert len(coef) == 5 and coef[0] > 1.5 and coef[4] > 0          # c1 .. c9; a positive leading term saturates correctly
    z = np.linspace(-12.0, 12.0, 2_400_001)
    z2 = z * z
    p = (((coef[4] * z2 + coef[3]) * z2 + coef[2]) * z2 + coef[1]) * z2 + coef[0]
    fit = z / (1.0 + np.exp(-z * p))
    want = 0.5 * z * (1.0 + erf(z / np.sqrt(2.0)))
    assert np.abs(fit - want).max() <= 3.1e-6
    for big in (-40.0, -15.0, 15.0, 40.0):                            # saturation: no overflow to NaN, exact limits
        pb = (((coef[4] * big**2 + coef[3]) * big**2 + coef[2]) * big**2 + coef[1]) * big**2 + coef[0]
        with np.errstate(over="ignore"):
            v = big / (1.0 + np.exp(-big * pb))
        assert v == (big if big > 0 else 0.0) or abs(v - max(big, 0.0)) < 1e-12
