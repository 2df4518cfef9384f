"""Pins of the BIAWGN capacity integrator (oracle/capacity.py) and of the sigma table stored in workloads.py."""
import math

import numpy as np
import pytest
from scipy import integrate, optimize

from oracle import capacity
from paper_1702_07740_b200 import workloads as W


def _capacity_quad(sigma):
    """Independent routine: scipy adaptive quadrature of the same expectation."""
    mu = 2.0 / sigma ** 2
    sd = 2.0 / sigma

    def f(L):
        return np.logaddexp(0.0, -L) / math.log(2.0) * math.exp(-0.5 * ((L - mu) / sd) ** 2) / (sd * math.sqrt(2 * math.pi))
    val, _ = integrate.quad(f, mu - 12 * sd, mu + 12 * sd, epsabs=1e-13, epsrel=1e-12, limit=400)
    return 1.0 - val


@pytest.mark.parametrize("sigma", [0.5, 1.0, 2.5, 6.0])
def test_capacity_matches_scipy_quad(sigma):
    assert capacity.biawgn_capacity(sigma) == pytest.approx(_capacity_quad(sigma), abs=1e-10)


def test_capacity_limits_and_monotonicity():
    assert capacity.biawgn_capacity(0.05) == pytest.approx(1.0, abs=1e-9)
    assert capacity.biawgn_capacity(40.0) < 1e-3
    cs = [capacity.biawgn_capacity(s) for s in (0.5, 1, 2, 4, 8)]
    assert all(a > b for a, b in zip(cs, cs[1:]))
    # low-SNR closed form: C ~ snr / (2 ln 2) to first order
    s = 20.0
    assert capacity.biawgn_capacity(s) == pytest.approx(1 / (2 * math.log(2) * s * s), rel=2e-3)


def test_sigma_star_table_and_shannon_agreement():
    for rate, stored in W.SIGMA_STAR.items():
        fresh = capacity.sigma_star(rate)
        assert stored == pytest.approx(fresh, abs=5e-10)
        root = optimize.brentq(lambda s: _capacity_quad(s) - rate, 0.5, 20.0, xtol=1e-12)
        assert fresh == pytest.approx(root, abs=1e-7)
    # at R = 0.02 the BIAWGN and the unconstrained thresholds agree to ~7 digits in SNR
    snr_bi = 1.0 / capacity.sigma_star(0.02) ** 2
    snr_sh = 1.0 / capacity.shannon_sigma_star(0.02) ** 2
    assert snr_bi == pytest.approx(0.0281139, abs=2e-7)
    assert snr_bi == pytest.approx(snr_sh, rel=2e-5) and snr_bi > snr_sh
    # paper P:620: SNR 0.161 at R = 0.1 is beta = 0.93 with the unconstrained capacity (Eq. 3)
    assert 0.1 / (0.5 * math.log2(1.161)) == pytest.approx(0.93, abs=2e-3)


def test_config_sigmas_match_survey_digits():
    # SURVEY.md S15 (scipy quad + brentq at survey time)
    want = {(0.1, 1.5): 2.18154369, (0.1, 0.5): 2.44773228, (0.02, 0.3): 5.76154922,
            (0.05, 0.1): 3.68983549, (0.05, 1.1): 3.28856934}
    for (rate, gap), sig in want.items():
        assert W.sigma_for_gap(rate, gap) == pytest.approx(sig, abs=2e-8)
        assert capacity.sigma_for_gap(rate, gap) == pytest.approx(sig, abs=2e-8)
