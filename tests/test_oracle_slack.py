"""Pins for the oracle's force slack (App. H): F_(eps) = F + clip(-eps_F; F~ - F; eps_F)."""
import math

import numpy as np
import pytest
from scipy import special

import lsd_inputs as L
from helpers import custom


def test_clip_componentwise_hand_values(orc):
    Ft = np.array([[1.0, -2.0, 0.5], [0.0, 3.0, -0.25]])
    F = np.array([[0.0, 0.0, 0.0], [0.0, 2.9, 0.0]])
    got = orc.force_slack(Ft, F, 0.3)
    # differences (1, -2, 0.5 | 0, 0.1, -0.25) clipped to +-0.3 and added to F
    assert np.abs(got - np.array([[0.3, -0.3, 0.3], [0.0, 3.0, -0.25]])).max() < 1e-15
    assert np.array_equal(orc.force_slack(Ft, F, 0.0), F)                       # no slack: the true target force
    assert np.array_equal(orc.force_slack(Ft, F, 10.0), Ft)                     # slack beyond every difference: the draft force


def test_slack_shrinks_delta_by_the_ball_radius_and_lowers_eq9(orc):
    """One atom, one non-zero component: delta = (b/sigma)(F~ - F) becomes (b/sigma)(|F~ - F| - eps_F)_+, so the rejection
    probability of Eq. 9 drops from erf(|delta|/sqrt 8) to erf(|delta_eps|/sqrt 8); eps_F >= |F~ - F| gives S2 = 0 (always accepted)."""
    w = custom([[0.0, 0.0, 0.0]], mass=[12.0], T=300.0, gamma=0.01, dt=0.5)
    par = orc.params(w)
    c1 = math.exp(-w.friction_per_fs * w.dt_fs)
    b = (1 + c1) * w.dt_fs / 2
    sigma = math.sqrt(12.0 * L.AMU * L.K_B * w.temperature_K * (1 - c1 * c1))
    Ft, F = np.array([[0.8, 0.0, 0.0]]), np.array([[0.2, 0.0, 0.0]])
    xi, p_prev, qh = np.array([[0.3, -1.0, 0.5]]), np.zeros((1, 3)), np.zeros((1, 3))
    for eps, gap in ((0.0, 0.6), (0.25, 0.35), (0.6, 0.0), (5.0, 0.0)):
        t = orc.transport_step(w, Ft, orc.force_slack(Ft, F, eps), xi, 0.5, p_prev, qh, par)
        assert t["S2"] == pytest.approx((b / sigma * gap) ** 2, rel=1e-12, abs=1e-300)
        assert orc.rejection_probability(math.sqrt(t["S2"])) == pytest.approx(special.erf(b / sigma * gap / math.sqrt(8)), rel=1e-12, abs=1e-300)
        if gap == 0.0:
            assert t["reject"] == 0
