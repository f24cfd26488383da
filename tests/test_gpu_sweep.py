"""SURVEY.md 8(f) rank 4 on the GPU: force slack (App. H) stage-wise against the oracle, and the rejection
statistics behind the Fig. 4-form sweep of bench.py --sweep (Eq. 9 :115, Eq. 11 :185).  -m gpu."""
import math

import numpy as np
import pytest
from scipy.special import erf, erfinv

import lsd_inputs as L

pytestmark = pytest.mark.gpu
BAND = 1e-6


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_02455_b200 as P
    P.load_library()
    return P


def test_force_slack_stagewise_against_oracle(P, orc):
    """The transport kernel with slack eps_F must equal the oracle's transport step fed with orc_force_slack(F~, F, eps_F):
    S1, S2 to 1e-10, decisions bit for bit outside the band, the overridden state to 1e-9; a huge slack accepts everything."""
    w = L.make_workload("cfg2")
    K = w.K
    p0 = orc.initial_momenta(w)
    par = orc.params(w)
    for eps_F, expect_all in ((0.05, False), (1e6, True)):
        ctx = P.context_from_workload(w, precision=P.LSD_FP32, p0=p0)
        P.lsd_set_force_slack(ctx.h, eps_F)
        q_base, p_base, n0 = ctx.state()
        P.lsd_draft_rollout(ctx.h, K); P.lsd_verify_window(ctx.h, K)
        l, nc = P.lsd_transport_accept(ctx.h, K)
        qh, Ft, Fg, yp = ctx.debug("q_half", K), ctx.debug("F_draft", K), ctx.debug("F_target", K), ctx.debug("yp", K)
        S1, S2, rej = ctx.debug("S1", K), ctx.debug("S2", K), ctx.debug("reject", K)
        first = 0
        for j in range(K):
            p_prev = p_base.T if j == 0 else yp[j - 1].T
            Fe = orc.force_slack(Ft[j].T, Fg[j].T, eps_F)
            u = orc.uniform(w.seed, n0 + j + 1)
            t = orc.transport_step(w, Ft[j].T, Fe, orc.normals(w.seed, n0 + j + 1, w.n_atoms), u, p_prev, qh[j].T, par)
            # (F + (F~ - F) is F~ only up to one rounding: with a slack beyond every difference the oracle keeps S2 ~ 1e-38, the kernel exactly 0)
            assert S2[j] == pytest.approx(t["S2"], rel=1e-10, abs=1e-25) and S1[j] == pytest.approx(t["S1"], rel=1e-9, abs=1e-12)
            if abs(t["ell"] - math.log(u)) >= BAND and not expect_all:
                assert rej[j] == t["reject"], j
            if t["reject"] and not first and not expect_all:
                first, xq, xp = j + 1, t["q"], t["p"]
                break                                            # yp rows behind the override are not the draft's any more
        if expect_all:
            assert l == 0 and nc == K and np.all(S2 == 0.0)
        else:
            assert l == first
            P.lsd_rollback(ctx.h, l)
            qg, pg, _ = ctx.state()
            if first:
                assert np.abs(qg.T - xq).max() <= 1e-9 and np.abs(pg.T - xp).max() <= 1e-9 * max(np.abs(xp).max(), 1.0)
        ctx.close()


def test_rejection_rate_matches_eq9_and_the_form_of_eq11(P):
    """fcc Cu, T = 1500 K, dt = 1 fs (the Fig. 4 conditions) with the draft / target gap of bench.py --sweep.  (i) the number of
    rejections over a segment sits within 4 sigma of sum_j erf(|delta_j| / sqrt 8) (Eq. 9), (ii) going from N = 500 to N = 256 and
    from tau = 1 ps to 0.1 ps moves the mean rate as erf(sqrt(N tau) ...) says (Eq. 11), within the sampling error."""
    import bench
    import torch
    stream = torch.cuda.Stream()
    K, nsteps = 8, 600
    eps = 1e-2
    ctx = P.context_from_workload(bench.sweep_workload(L, 5, 1000.0, eps), k_max=K, precision=P.LSD_BF16_TC)
    ctx.window(K, stream)
    eps *= float(erfinv(0.3)) * math.sqrt(8.0) / float(np.mean(np.sqrt(ctx.debug("S2", K))))
    ctx.close()
    rate = {}
    for cells, tau in ((5, 1000.0), (4, 1000.0), (5, 100.0)):
        ctx = P.context_from_workload(bench.sweep_workload(L, cells, tau, eps), k_max=K, precision=P.LSD_BF16_TC)
        P.lsd_run(ctx.h, 2 * K, K, overlap=False, stream=stream)
        s0 = P.lsd_get_stats(ctx.h)
        P.lsd_run(ctx.h, nsteps, K, overlap=False, stream=stream)
        s1 = P.lsd_get_stats(ctx.h)
        nc, R, bsum = s1["committed_steps"] - s0["committed_steps"], s1["rejections"] - s0["rejections"], s1["beta_sum"] - s0["beta_sum"]
        mean_beta = bsum / nc
        sigma = math.sqrt(max(bsum * (1.0 - mean_beta), 1.0))
        assert abs(R - bsum) <= 4.0 * sigma, (cells, tau, R, bsum)
        rate[(cells, tau)] = (mean_beta, sigma / nc)
        ctx.close()
    b0 = rate[(5, 1000.0)][0]
    assert 0.2 < b0 < 0.4                                         # the probe window put the fit point near 0.3
    for (cells, tau) in ((4, 1000.0), (5, 100.0)):
        n_at = 4 * cells**3
        pred = float(erf(math.sqrt(n_at * tau / (500 * 1000.0)) * erfinv(b0)))
        got, err = rate[(cells, tau)]
        assert abs(got - pred) <= 0.15 * pred + 4 * err, (cells, tau, got, pred)


def test_sweep_counts_against_the_oracle_at_n256(P, orc):
    """The counters the sweep reads (lsd_get_stats: rejections, beta_sum, windows) against the oracle's run of the same
    256-atom system (fp32 network path, so that the decisions agree): 24 committed steps in windows of 8."""
    import bench
    K, nsteps = 8, 24
    w = bench.sweep_workload(L, 4, 1000.0, 0.3)
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, k_max=K, precision=P.LSD_FP32, p0=p0)
    P.lsd_run(ctx.h, nsteps, K, overlap=False)
    st = P.lsd_get_stats(ctx.h)
    qg, pg, step = ctx.state()
    ro = orc.run_lsd(w, w.q0, p0, nsteps, K=K, keep_traj=False)
    assert step == nsteps and st["committed_steps"] == nsteps
    assert st["windows"] == ro["windows"] and st["rejections"] == ro["rejections"]
    assert st["beta_sum"] == pytest.approx(ro["beta_sum"], rel=2e-3)
    assert np.abs(qg.T - ro["q"]).max() < 1e-4                   # same decisions => same trajectory up to the fp32 force error
    ctx.close()
