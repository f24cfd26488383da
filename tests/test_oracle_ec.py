"""Pins for the oracle's speculative error correction (EC; App. E :626-630, Alg. 3 :663-717; oracle O-5)."""
import math

import numpy as np
import pytest

import lsd_inputs as L
from test_oracle_lsd import _osc


def test_ec_with_zero_cache_is_the_plain_window(orc):
    """dF = 0 (Alg. 3 line "dF <- 0", :669): the first EC window IS the Alg. 1 window, bit for bit; the cache it leaves is
    F - F~ (bare) of the LAST COMMITTED step, taken from the window's own debug rows (:694, :710-713)."""
    w = L.make_workload("cfg2")
    p0 = orc.initial_momenta(w)
    a = orc.lsd_window(w, w.q0, p0, 0, K=16)
    b = orc.lsd_window(w, w.q0, p0, 0, K=16, dF=np.zeros_like(w.q0))
    for key in ("q", "p", "traj_q", "traj_p", "S1", "S2", "ell", "reject", "Ft", "F"):
        assert np.array_equal(a[key], b[key]), key
    assert (a["first_reject"], a["n_commit"]) == (b["first_reject"], b["n_commit"])
    c = b["n_commit"]
    assert 1 <= c < 16                                           # a rejection inside the window: c = l, the overridden step
    assert np.array_equal(b["dF"], b["F"][c - 1] - b["Ft"][c - 1])
    # draft == target: the cache stays exactly zero and nothing is ever rejected
    d = orc.lsd_window(w, w.q0, p0, 0, K=16, draft=w.target, dF=np.zeros_like(w.q0))
    assert d["first_reject"] == 0 and d["n_commit"] == 16 and not d["dF"].any() and not d["S2"].any()


def test_ec_with_the_exact_error_reproduces_the_target_step(orc):
    """Special case: if the cache equals the true error at the window's first q_half (which depends on the base state
    only), F~ + dF = F there, so delta = 0: S2 vanishes, the step is accepted whatever u is, and the drafted state equals
    the plain TARGET Langevin step under the same noise (a wrong sign of dF in either the draft or the verify half doubles
    delta instead)."""
    w = L.make_workload("cfg2")
    p0 = orc.initial_momenta(w)
    m = (w.mass_amu * L.AMU)[:, None]
    q_half = w.q0 + 0.5 * w.dt_fs * p0 / m
    Fd = orc.energy_forces(w, w.draft, q_half)[1]
    Ft = orc.energy_forces(w, w.target, q_half)[1]
    out = orc.lsd_window(w, w.q0, p0, 0, K=1, dF=Ft - Fd)
    plain = orc.lsd_window(w, w.q0, p0, 0, K=1)
    assert plain["S2"][0] > 1e-3                                 # without the cache the two models do differ
    assert out["S2"][0] < 1e-24 * max(1.0, plain["S2"][0]) and out["first_reject"] == 0
    ref = orc.run_aboba(w, w.target, w.q0, p0, 1)
    assert np.allclose(out["q"], ref["q"], rtol=0, atol=1e-12) and np.allclose(out["p"], ref["p"], rtol=0, atol=1e-12)
    assert np.allclose(out["dF"], Ft - Fd, rtol=0, atol=1e-12)   # cache after the window: same step, same error


def test_ec_first_draft_momentum_is_shifted_by_b_times_the_cache(orc):
    """Eq. 7 with F~ + dF (:681): under the same noise the first draft momentum moves by exactly b dF, b = (1 + c1) dt / 2."""
    w = L.make_workload("cfg2")
    p0 = orc.initial_momenta(w)
    rng = np.random.default_rng(3)
    dF = rng.normal(0, 0.05, w.q0.shape)
    a = orc.lsd_window(w, w.q0, p0, 7, K=1, draft=w.target)                      # nothing rejected: p = draft momentum
    b = orc.lsd_window(w, w.q0, p0, 7, K=1, draft=w.target, dF=dF)
    c1 = math.exp(-w.friction_per_fs * w.dt_fs)
    bb = (1 + c1) * w.dt_fs / 2
    S2 = ((bb * dF) ** 2 / (w.mass_amu[:, None] * L.AMU * L.K_B * w.temperature_K * (1 - c1 * c1))).sum()
    assert b["S2"][0] == pytest.approx(S2, rel=1e-12)            # draft == target, so delta is the cache alone (exact prefactor)
    if b["first_reject"] == 0:
        assert np.allclose(b["p"] - a["p"], bb * dF, rtol=0, atol=1e-13)


def test_ec_keeps_the_target_law_and_lowers_the_rejection_rate(orc):
    """Thm. 3.1 holds for any draft law (:630): with a wrong draft (k_draft = 1.3 k) AND error correction the oscillator
    keeps the TARGET's <q^2> = kT/k; rejections follow Eq. 9 with the corrected delta; and because the error
    (k_draft - k) q changes slowly from step to step, EC rejects less often than plain LSD (:196)."""
    k, mass, T, gamma, dt = 20.0, 1.008, 300.0, 0.2, 0.5
    w = _osc(2, k, mass, T, gamma, dt, seed=9, k_draft=1.3 * k)
    q, p = w.q0, orc.initial_momenta(w)
    sq = cnt = 0.0
    rej = {True: 0, False: 0}
    beta_sum = steps = 0.0
    for chunk in range(40):
        par = orc.params(w, seed=900 + chunk)
        out = orc.run_lsd(w, q, p, 5000, K=8, par=par, ec=True)
        plain = orc.run_lsd(w, q, p, 5000, K=8, par=par, ec=False)
        q, p = out["q"], out["p"]
        sq += (out["traj_q"][::2] ** 2).sum(); cnt += out["traj_q"][::2].size
        rej[True] += out["rejections"]; rej[False] += plain["rejections"]
        beta_sum += out["beta_sum"]; steps += out["examined"]
    kT = L.K_B * T
    assert (sq / cnt) / (kT / k) == pytest.approx(1.0, abs=0.02)
    assert abs(rej[True] - beta_sum) < 4.5 * math.sqrt(beta_sum)
    assert rej[True] < 0.85 * rej[False]                         # measured: 25 % fewer with a cache refreshed once per window of 8
