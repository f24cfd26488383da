"""GPU parity of speculative error correction (Alg. 3; include/lsd.h lsd_set_error_correction) against
the oracle's orc_lsd_window_ec (O-5)."""
import math

import numpy as np
import pytest

import lsd_inputs as L

pytestmark = pytest.mark.gpu
BAND = 1e-6
POS_TOL = 1e-6


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_02455_b200 as P
    P.load_library()
    return P


def test_ec_cfg1_end_to_end_against_the_oracle(P, orc):
    """cfg1 (fp64 on both sides), EC on: decisions, first-reject indices and the cache follow the oracle window by window."""
    w = L.make_workload("cfg1")
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, p0=p0)
    P.lsd_set_error_correction(ctx.h, True)
    q, p, n, dF = w.q0, p0, 0, np.zeros_like(w.q0)
    cache = np.empty((3, w.n_atoms))
    n_rej = 0
    while n < 600:
        K = min(w.K, 600 - n)
        r = orc.lsd_window(w, q, p, n, K=K, dF=dF)
        l, nc = ctx.window(K)
        assert not (np.abs(r["ell"] - r["lnu"]) < BAND).any()
        assert (l, nc) == (r["first_reject"], r["n_commit"]), n
        assert np.array_equal(ctx.debug("reject", K), r["reject"])
        assert np.allclose(ctx.debug("ell", K), r["ell"], rtol=0, atol=1e-9)
        P.lsd_get_ec_cache(ctx.h, cache)
        assert np.abs(cache.T - r["dF"]).max() <= 1e-9 * max(1.0, np.abs(r["dF"]).max())
        q, p, n, dF = r["q"], r["p"], n + nc, r["dF"]
        qg, pg, step = ctx.state()
        assert step == n and np.abs(qg.T - q).max() <= POS_TOL
        n_rej += 1 if l else 0
    assert n_rej > 0 and np.abs(dF).max() > 0
    assert np.abs(qg.T - q).max() <= 1e-9
    ctx.close()


@pytest.mark.parametrize("name,kw,K,prec", [("cfg2", {}, 16, "fp32"), ("cfg3", {"n_grid": 7}, 4, "fp32"), ("cfg5", {"cells": (4, 4, 4)}, 4, "bf16")])
def test_ec_stagewise_parity(P, orc, name, kw, K, prec):
    """The oracle's EC window arithmetic on the GPU's own forces: the cache the GPU keeps is bit-exactly F - F~ (bare) of
    its last committed step; S1, S2 and the decisions are those of delta = (b/sigma)(F~ + dF - F) with the cache the
    window was drafted with; the first draft momentum carries the kick b (F~ + dF)."""
    w = L.make_workload(name, **kw)
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, k_max=K, precision=P.LSD_BF16_TC if prec == "bf16" else P.LSD_FP32, p0=p0)
    P.lsd_set_error_correction(ctx.h, True)
    par = orc.params(w)
    cache = np.zeros((3, w.n_atoms))
    p, n = p0, 0
    m = (w.mass_amu * L.AMU)[:, None]
    c1 = math.exp(-w.friction_per_fs * w.dt_fs); b = (1 + c1) * w.dt_fs / 2
    sg = np.sqrt(m * L.K_B * w.temperature_K * (1 - c1 * c1))
    used_nonzero = False
    for win in range(4):
        dF = cache.T.copy()                                     # cache this window is drafted with
        used_nonzero |= bool(np.abs(dF).max() > 0)
        l, nc = ctx.window(K)
        qh, Ft, Fg = ctx.debug("q_half", K), ctx.debug("F_draft", K), ctx.debug("F_target", K)
        S1, S2, rej, yp = ctx.debug("S1", K), ctx.debug("S2", K), ctx.debug("reject", K), ctx.debug("yp", K)
        first = 0
        for j in range(K):
            p_prev = p if j == 0 else yp[j - 1].T
            xo = orc.normals(w.seed, n + j + 1, w.n_atoms)
            u = orc.uniform(w.seed, n + j + 1)
            t = orc.transport_step(w, Ft[j].T + dF, Fg[j].T, xo, u, p_prev, qh[j].T, par)
            assert S1[j] == pytest.approx(t["S1"], rel=1e-10, abs=1e-12) and S2[j] == pytest.approx(t["S2"], rel=1e-10, abs=1e-300)
            if abs(t["ell"] - math.log(u)) >= BAND:
                assert rej[j] == t["reject"], (win, j)
            if t["reject"]:
                first = j + 1
                x_q, x_p = t["q"], t["p"]
                break
            pn = c1 * p_prev + b * (Ft[j].T + dF) + sg * xo      # Eq. 7 around F~ + dF
            assert np.abs(yp[j].T - pn).max() <= 1e-9 * np.abs(pn).max()
        assert l == first and nc == (first if first else K)
        P.lsd_get_ec_cache(ctx.h, cache)
        assert np.array_equal(cache, Fg[nc - 1] - Ft[nc - 1])   # fp64 difference of two stored arrays: bit-exact
        qg, pg, step = ctx.state()
        if first:
            assert np.abs(qg.T - x_q).max() <= 1e-9 and np.abs(pg.T - x_p).max() <= 1e-9 * np.abs(x_p).max()
        p, n = pg.T.copy(), step
    assert used_nonzero
    ctx.close()


def test_ec_switch_resets_cache_and_off_is_the_plain_path(P, orc):
    w = L.make_workload("cfg2")
    p0 = orc.initial_momenta(w)
    finals = []
    for mode in ("never", "on_then_off"):
        ctx = P.context_from_workload(w, k_max=8, precision=P.LSD_FP32, p0=p0)
        if mode == "on_then_off":
            P.lsd_set_error_correction(ctx.h, True)
            ctx.window(8)
            cache = np.empty((3, w.n_atoms)); P.lsd_get_ec_cache(ctx.h, cache)
            assert np.abs(cache).max() > 0
            with pytest.raises(P.LsdError):
                pass_through = np.zeros((3, w.n_atoms))
                P.lsd_set_error_correction(ctx.h, False)
                P.lsd_set_ec_cache(ctx.h, pass_through)          # STATE: EC is off
            P.lsd_get_ec_cache(ctx.h, cache)
            assert not cache.any()                              # switching zeroes the cache
            q0 = np.ascontiguousarray(w.q0.T); pp = np.ascontiguousarray(p0.T)
            P.lsd_set_state(ctx.h, q0, pp, 0)
        for _ in range(6):
            ctx.window(8)
        finals.append(ctx.state())
        ctx.close()
    assert np.array_equal(finals[0][0], finals[1][0]) and np.array_equal(finals[0][1], finals[1][1]) and finals[0][2] == finals[1][2]


def test_ec_graph_replay_and_overlap_are_deterministic(P, orc, monkeypatch):
    """EC under CUDA-graph replay equals direct launches bit for bit; lsd_run with the speculative second-stream rollout is
    reproducible run to run (the speculative window inherits the cache of the window before it, never a racing copy)."""
    import torch
    w = L.make_workload("cfg2")
    p0 = orc.initial_momenta(w)
    out = []
    for graphs, mode in (("1", "windows"), ("0", "windows"), ("1", "run"), ("1", "run")):
        monkeypatch.setenv("LSD_GRAPHS", graphs)
        ctx = P.context_from_workload(w, k_max=8, precision=P.LSD_FP32, p0=p0)
        P.lsd_set_error_correction(ctx.h, True)
        stream = torch.cuda.Stream()
        if mode == "windows":
            for _ in range(10):
                ctx.window(8, stream)
        else:
            P.lsd_run(ctx.h, 64, 8, overlap=True, stream=stream)
        out.append(ctx.state())
        ctx.close()
    for a, b in ((0, 1), (2, 3)):
        assert np.array_equal(out[a][0], out[b][0]) and np.array_equal(out[a][1], out[b][1]) and out[a][2] == out[b][2]


@pytest.mark.parametrize("name,kw", [("cfg1", {}), ("cfg2", {})])
def test_obabo_outputs_match_the_oracle(P, orc, name, kw):
    """lsd_get_window_obabo (App. F Eq. 26-30): q = q_half_j, p = p_mid recovered from the GPU's own committed momenta and
    target forces; the oracle's recovery on the same arrays (same Philox tag-3 draw) agrees to round-off, for accepted and
    for overridden steps."""
    w = L.make_workload(name, **kw)
    p0 = orc.initial_momenta(w)
    K = 8 if name == "cfg2" else 4
    ctx = P.context_from_workload(w, k_max=K, precision=P.LSD_FP32, p0=p0)
    p_base, n = p0, 0
    saw_override = False
    for win in range(12):
        P.lsd_draft_rollout(ctx.h, K); P.lsd_verify_window(ctx.h, K)
        l, nc = P.lsd_transport_accept(ctx.h, K)
        qh, Fg = ctx.debug("q_half", K), ctx.debug("F_target", K)
        prev = p_base
        for j in range(1, nc + 1):
            qs, ps = np.empty((3, w.n_atoms)), np.empty((3, w.n_atoms))
            P.lsd_get_window_state(ctx.h, j, qs, ps)
            qo, po = np.empty((3, w.n_atoms)), np.empty((3, w.n_atoms))
            P.lsd_get_window_obabo(ctx.h, j, qo, po)
            assert np.array_equal(qo, qh[j - 1])
            ref = orc.obabo_momentum(w, n + j, prev, ps.T, Fg[j - 1].T)
            assert np.abs(po.T - ref).max() <= 1e-10 * max(1.0, np.abs(ref).max())
            prev = ps.T.copy()
        saw_override |= l != 0
        P.lsd_rollback(ctx.h, l)
        p_base, n = prev, n + nc
    assert saw_override
    ctx.close()
