"""ORACLE (test infrastructure, not product code): BIAWGN capacity and the sigma at capacity for a code rate.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.

BASELINE.json states the channel point of every config as "x dB above BIAWGN capacity for rate R, computed by the
oracle via numerical integration".  The paper uses s = 1/sigma_Z^2 as the SNR and the unconstrained capacity
(1/2) log2(1+s) in its efficiency beta (Eq. 3); at R = 0.02 the two capacities agree to 7 digits, which
tests/test_capacity.py uses as a closed-form check (reading S15).

Definition used (textbook BIAWGN with BPSK +-1, noise N(0, sigma^2)): the channel LLR given x = 0 is
L ~ N(2/sigma^2, 4/sigma^2) and   C(sigma) = 1 - E[ log2(1 + exp(-L)) ].
The expectation is a plain composite trapezoid rule in the standard-normal variable z on [-12, 12]
(the integrand times the Gaussian weight is < 1e-30 outside) -- no library quadrature, so that the test can compare
it with scipy.integrate.quad as an independent routine.
"""
from __future__ import annotations

import math

import numpy as np

_Z = np.linspace(-12.0, 12.0, 480001)
_W = np.exp(-0.5 * _Z * _Z) / math.sqrt(2.0 * math.pi)


def biawgn_capacity(sigma: float) -> float:
    """C(sigma) in bits per channel use."""
    mu = 2.0 / (sigma * sigma)
    L = mu + math.sqrt(2.0 * mu) * _Z          # std-dev of L is 2/sigma = sqrt(2 mu)
    f = np.logaddexp(0.0, -L) / math.log(2.0) * _W
    h = _Z[1] - _Z[0]
    integral = h * (f.sum() - 0.5 * (f[0] + f[-1]))
    return 1.0 - float(integral)


def sigma_star(rate: float) -> float:
    """sigma with C(sigma) = rate, by bisection (C is decreasing in sigma)."""
    lo, hi = 0.05, 50.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if biawgn_capacity(mid) > rate:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def sigma_for_gap(rate: float, gap_db: float) -> float:
    """sigma^2 = sigma*^2 * 10^(-gap/10): the channel is `gap_db` dB better than the capacity threshold."""
    return sigma_star(rate) * 10.0 ** (-gap_db / 20.0)


def shannon_sigma_star(rate: float) -> float:
    """Unconstrained AWGN: (1/2) log2(1 + 1/sigma^2) = rate."""
    return 1.0 / math.sqrt(2.0 ** (2.0 * rate) - 1.0)
