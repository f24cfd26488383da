"""Pins for the oracle's (OBABO) output recovery by time staggering (App. F :632-753, Eq. 24-30; oracle O-6)."""
import math

import numpy as np
import pytest
from scipy import linalg

import lsd_inputs as L
from test_oracle_lsd import _osc


def _obabo_stationary_cov(k, m, kT, gamma, dt):
    """Stationary covariance of (q, p) at the OUTPUT of one (OBABO) step, Eq. 24 composed as a linear map in numpy and the
    discrete Lyapunov equation solved with scipy -- independent of the oracle."""
    ch = math.exp(-gamma * dt / 2)
    s2 = m * kT * (1 - math.exp(-gamma * dt))                  # Sigma_half
    O = np.array([[1, 0], [0, ch]]); B = np.array([[1, 0], [-k * dt / 2, 1]]); A = np.array([[1, dt / m], [0, 1]])
    M = O @ B @ A @ B @ O
    e = np.array([[0.0], [1.0]])
    first = (O @ B @ A @ B) @ e                                # how the first O's noise reaches the output
    N = s2 * (first @ first.T) + s2 * (e @ e.T)
    return linalg.solve_discrete_lyapunov(M, N)


def test_obabo_outputs_have_the_obabo_stationary_covariance(orc):
    """LSD runs in the staggered (ABOBA) frame with a deliberately wrong draft; the recovered (q_half_n, p_mid_n) must be
    distributed like (OBABO) outputs of the TARGET: <q^2>, <p^2>, <qp> against the Lyapunov solution (they differ from the
    ABOBA values: ABOBA has <q^2> = kT/k exactly, OBABO has <p^2> = m kT exactly)."""
    k, mass, T, gamma, dt = 20.0, 1.008, 300.0, 0.2, 0.5
    w = _osc(2, k, mass, T, gamma, dt, seed=9, k_draft=1.3 * k)
    m, kT = mass * L.AMU, L.K_B * T
    cov = _obabo_stationary_cov(k, m, kT, gamma, dt)
    assert cov[1, 1] == pytest.approx(m * kT, rel=1e-9)          # textbook property of OBABO: exact momentum marginal
    assert cov[0, 0] == pytest.approx(kT / k / (1 - dt * dt * k / (4 * m)), rel=1e-9)
    q, p, n = w.q0, orc.initial_momenta(w), 0
    acc = np.zeros(3); cnt = 0; z1 = []; z2 = []
    c1, ch = math.exp(-gamma * dt), math.exp(-gamma * dt / 2)
    sh = math.sqrt(m * kT * (1 - c1))
    while n < 120000:
        r = orc.lsd_window(w, q, p, n, K=8)
        nc = r["n_commit"]
        for j in range(nc):
            p_prev = p if j == 0 else r["traj_p"][j - 1]
            p_new, F, qh = r["traj_p"][j], r["F"][j], r["q_half"][j]
            pm = orc.obabo_momentum(w, n + j + 1, p_prev, p_new, F)
            acc += [(qh * qh).sum(), (pm * pm).sum(), (qh * pm).sum()]; cnt += qh.size
            if len(z1) < 4000:                                   # the two half-step noises implied by (p_in, p_mid, p_out), Eq. 27
                p_in, p_out = p_prev + dt / 2 * F, p_new - dt / 2 * F
                z1.append(((pm - ch * p_in) / sh).ravel()); z2.append(((p_out - ch * pm) / sh).ravel())
        q, p, n = r["q"], r["p"], n + nc
    qq, pp, qp = acc / cnt
    assert qq == pytest.approx(cov[0, 0], rel=0.02)
    assert pp == pytest.approx(cov[1, 1], rel=0.02)
    assert abs(qp - cov[0, 1]) < 0.02 * math.sqrt(cov[0, 0] * cov[1, 1])
    z1, z2 = np.concatenate(z1), np.concatenate(z2)
    for z in (z1, z2):
        assert abs(z.mean()) < 0.02 and z.var() == pytest.approx(1.0, abs=0.03)
    assert abs(np.corrcoef(z1, z2)[0, 1]) < 0.03                 # xi1* and xi2 are independent


def test_obabo_recovery_is_consistent_with_the_merged_step(orc):
    """Exact identity behind Eq. 28: whatever extra normal is drawn, the two half-steps compose to the staggered result:
    e^{-gamma dt/2} xi1* + xi2 = w, i.e. p_out - e^{-gamma dt} p_in = Sigma_half^{1/2} (e^{-gamma dt/2} xi1* + xi2)."""
    w = L.make_workload("cfg2")
    p0 = orc.initial_momenta(w)
    r = orc.lsd_window(w, w.q0, p0, 0, K=4)
    p_new, F = r["traj_p"][0], r["F"][0]
    pm = orc.obabo_momentum(w, 1, p0, p_new, F)
    dt, g = w.dt_fs, w.friction_per_fs
    c1, ch = math.exp(-g * dt), math.exp(-g * dt / 2)
    sh = np.sqrt(w.mass_amu * L.AMU * L.K_B * w.temperature_K * (1 - c1))[:, None]
    p_in, p_out = p0 + dt / 2 * F, p_new - dt / 2 * F
    xi1, xi2 = (pm - ch * p_in) / sh, (p_out - ch * pm) / sh
    assert np.allclose(ch * xi1 + xi2, (p_out - c1 * p_in) / sh, rtol=0, atol=1e-10)
    pm2 = orc.obabo_momentum(w, 2, p0, p_new, F)                 # another step index: another draw, same conditional mean
    assert not np.allclose(pm, pm2)
