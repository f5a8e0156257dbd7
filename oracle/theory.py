"""Closed forms of the paper's analysis (test infrastructure; used as oracle pins and in reports).

    delta_k(k)      Eq. 3  E[max of k standard normals], by quadrature
    F(Delta, S)     Eq. 7  leading-order underflow fraction
    F_star(...)     the same averaged over the max-of-k distribution instead of its mean
                    (the "per-row spread of m_global" the proof of Cor. 2 names)
    Delta_c(S)      collapse threshold
"""
import math

import numpy as np
from scipy import integrate
from scipy.stats import norm

LN2_10 = 10.0 * math.log(2.0)        # 6.9315


def delta_k(k: int) -> float:
    f = lambda m: m * k * norm.pdf(m) * norm.cdf(m) ** (k - 1)
    val, _ = integrate.quad(f, -12.0, 12.0, epsabs=1e-12, epsrel=1e-12)
    return float(val)


def F(delta: float, S: float, k_sink: int = 4) -> float:
    return float(norm.cdf(delta + delta_k(k_sink) - LN2_10 - math.log(S)))


def F_star(delta: float, S: float, k_sink: int = 4, sigma: float = 1.0, mean_shift: float = 0.0) -> float:
    """Underflow fraction with the sink maximum integrated over its distribution.

    Non-sink scores ~ N(0, sigma^2); sink scores = delta + N(0, sigma^2).
    A non-sink score s underflows iff s < delta + M - 10 ln 2 - ln S, M = max of k noise terms.
    """
    c = delta + mean_shift - LN2_10 - math.log(S)
    f = lambda m: norm.cdf((c + sigma * m) / sigma) * k_sink * norm.pdf(m) * norm.cdf(m) ** (k_sink - 1)
    val, _ = integrate.quad(f, -12.0, 12.0, epsabs=1e-12, epsrel=1e-12)
    return float(val)


def Delta_c(S: float, k_sink: int = 4) -> float:
    return LN2_10 + math.log(S) - delta_k(k_sink)
