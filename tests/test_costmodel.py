"""CPU: the Eq. (9) fit recovers known coefficients and predicts with them."""
import numpy as np
import pytest

from paper_2607_01701_b200 import costmodel


def test_fit_recovers_alpha_and_predicts():
    a1, a2 = 3.0e-5, 4.0e-8
    S = np.array([3600, 10800, 32400, 61200, 118800], dtype=np.float64)
    t = a1 * S + a2 * S * S
    f1, f2 = costmodel.fit_alpha(S, t)
    assert abs(f1 - a1) / a1 < 1e-9 and abs(f2 - a2) / a2 < 1e-9
    # Eq. 9: compute scales 1/k, communication term added
    assert costmodel.predict(a1, a2, 2, 1000, k=4, v_comm=8.0, bw_eff=2.0) == pytest.approx((a1 * 2000 + a2 * 2e6) / 4 + 4.0)
    # noisy points: relative-error weighting keeps the short sequences honest
    rng = np.random.default_rng(0)
    g1, g2 = costmodel.fit_alpha(S, t * (1 + 0.01 * rng.standard_normal(S.size)))
    assert abs(g2 - a2) / a2 < 0.05
    with pytest.raises(ValueError):
        costmodel.fit_alpha([1.0], [1.0])
