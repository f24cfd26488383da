"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (cfg5: 65,536 atoms, K = 8, bf16 tcgen05
path; cfg4: 4,096 atoms, K = 32; cfg3: 1,536 atoms, K = 16).  Forces are compared with the oracle element-wise per atom
(test_full_size_forces_match_oracle: cfg3 / cfg4 two window states each in fp32 and bf16, cfg5 one state, plus the draft forces of
one state each -- one oracle evaluation
of the 6-block network on 65,536 atoms takes about a minute on the box's host cores); everything else the oracle can do at
full size is compared directly too: neighbour lists (cell-list oracle, bit-exact), the transport map / decisions on the GPU's
own forces, the noise; plus properties that hold at any size (sum of forces, batch invariance, reproducibility)."""
import math
import os

import numpy as np
import pytest

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


@pytest.mark.parametrize("name", ["cfg5", "cfg4"])
def test_full_size_window(P, orc, name):
    import torch
    w = L.make_workload(name)
    K, N = w.K, w.n_atoms
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, precision=P.LSD_BF16_TC, p0=p0)
    assert P.lsd_tc_enabled(ctx.h)
    stream = torch.cuda.Stream()
    par = orc.params(w)
    m = (w.mass_amu * L.AMU)[:, None]
    for win in range(2):                                        # the second window replays the captured graphs
        q_base, p_base, n = ctx.state()
        P.lsd_draft_rollout(ctx.h, K, stream); P.lsd_verify_window(ctx.h, K, stream)
        l, nc = P.lsd_transport_accept(ctx.h, K, stream)
        qh, Ft, Fg = ctx.debug("q_half", K), ctx.debug("F_draft", K), ctx.debug("F_target", K)
        S1, S2, rej, yp = ctx.debug("S1", K), ctx.debug("S2", K), ctx.debug("reject", K), ctx.debug("yp", K)
        assert np.isfinite(Fg).all() and np.isfinite(Ft).all()
        # --- properties of the batched target forces at full size
        for j in range(K):
            tot = np.abs(Fg[j]).sum()
            assert np.abs(Fg[j].sum(axis=1)).max() <= 1e-4 * tot / 3          # sum_i F_i = 0 (every term is a pair term)
        # --- neighbour lists of two window states against the oracle's cell list, bit-exact (T1)
        if win == 0:
            for b in (0, K - 1):
                got = P.lsd_get_neighbors(ctx.h, P.LSD_TARGET, 0, b, N)
                want = orc.neighbors(w, np.ascontiguousarray(qh[b].T), w.target.mlip.cutoff, "cell")
                assert np.array_equal(got[0], want[0]) and np.array_equal(got[1], want[1]) and np.array_equal(got[2], want[2])
        # --- first A half-step from the committed base state (T4) and the transport map on the GPU's own forces (T3)
        assert np.abs(qh[0] - (q_base + w.dt_fs / 2 * p_base / m.T)).max() <= 1e-12
        first = 0
        for j in range(K):
            p_prev = p_base.T if j == 0 else yp_before[j - 1].T
            if j == 0:
                yp_before = yp.copy()
            xo = orc.normals(w.seed, n + j + 1, N)
            u = orc.uniform(w.seed, n + j + 1)
            t = orc.transport_step(w, Ft[j].T, Fg[j].T, xo, u, p_prev, qh[j].T, par)
            assert S1[j] == pytest.approx(t["S1"], rel=1e-9, abs=1e-9) and S2[j] == pytest.approx(t["S2"], rel=1e-10)
            if abs(t["ell"] - math.log(u)) >= BAND:
                assert rej[j] == t["reject"], (win, j)
            if t["reject"] and not first:
                first, x_q, x_p = j + 1, t["q"], t["p"]
        assert l == first and nc == (first if first else K)
        P.lsd_rollback(ctx.h, l)
        qg, pg, step = ctx.state()
        assert step == n + nc
        if first:
            assert np.abs(qg.T - x_q).max() <= 1e-9 and np.abs(pg.T - x_p).max() <= 1e-9 * np.abs(x_p).max()
    # --- batch invariance at full size: one state alone == the same state inside the batch of K
    Q = np.ascontiguousarray(qh[:2])
    F2, _ = ctx.forces(P.LSD_TARGET, Q)
    F1, _ = ctx.forces(P.LSD_TARGET, Q[1:2])
    assert np.array_equal(F1[0], F2[1])
    assert np.array_equal(F2[0], Fg[0])                         # and equal to what the (graph-replayed) verification produced
    ctx.close()


@pytest.mark.parametrize("name,kw", [("cfg4", {"n_atoms": 700}), ("cfg5", {"cells": (5, 5, 4)}), ("cfg3", {"n_grid": 7})])
def test_bf16_runs_are_reproducible_bit_for_bit(P, orc, name, kw):
    """Two independent contexts, 40 windows each on their own streams (graph replay, tcgen05 kernels with dynamic tile
    scheduling, asynchronous copies, mbarrier hand-offs): a race or an order-dependent sum would show up as a difference."""
    import torch
    w = L.make_workload(name, **kw)
    p0 = orc.initial_momenta(w)
    finals = []
    for rep in range(2):
        ctx = P.context_from_workload(w, k_max=4, precision=P.LSD_BF16_TC, p0=p0)
        stream = torch.cuda.Stream()
        hist = [ctx.window(4, stream) for _ in range(40)]
        finals.append((hist, *ctx.state()))
        ctx.close()
    assert finals[0][0] == finals[1][0]
    assert np.array_equal(finals[0][1], finals[1][1]) and np.array_equal(finals[0][2], finals[1][2]) and finals[0][3] == finals[1][3]
    assert np.isfinite(finals[0][1]).all()


def _t2_error(Fg, Fo):
    """T2: max_i |dF_i| / max(|F_i|, F_rms); Fg, Fo: [N, 3]."""
    nrm = np.linalg.norm(Fo, axis=1)
    rms = math.sqrt((Fo**2).sum(1).mean())
    return float((np.linalg.norm(Fg - Fo, axis=1) / np.maximum(nrm, rms)).max())


# (workload, precision, window states compared with the oracle).  One oracle evaluation costs about 0.2 s (cfg3), 1 s (cfg4) and one
# minute (cfg5: 65,536 atoms, 6 blocks of width 128 in fp64 on the box's host cores), so cfg5 compares one state.
FULL_FORCE_CASES = [("cfg3", "fp32", (0, 15)), ("cfg3", "bf16", (0, 15)), ("cfg4", "fp32", (0, 31)), ("cfg4", "bf16", (0, 31)),
                    ("cfg5", "bf16", (7,))]


@pytest.mark.parametrize("name,prec,states", FULL_FORCE_CASES)
def test_full_size_forces_match_oracle(P, orc, name, prec, states):
    """north_star: in-tolerance forces against the oracle on the configurations at the sizes BASELINE.json states, in the launch
    configuration bench.py times: the batched target forces of a whole window of K states (second window of the context, i.e.
    the graph-replayed launch sequence), element-wise per atom against the fp64 oracle at the same q_half (T2: 1e-5 fp32,
    2e-2 bf16).  The test also asserts which edge kernel instantiation produced them."""
    import torch
    w = L.make_workload(name)
    K, N = w.K, w.n_atoms
    bf16 = prec == "bf16"
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, precision=P.LSD_BF16_TC if bf16 else P.LSD_FP32, p0=p0)
    assert bool(P.lsd_tc_enabled(ctx.h)) == bf16
    stream = torch.cuda.Stream()
    ctx.window(K, stream)                                       # first window: plain launches, captures the graphs
    P.lsd_draft_rollout(ctx.h, K, stream); P.lsd_verify_window(ctx.h, K, stream)
    l, nc = P.lsd_transport_accept(ctx.h, K, stream)
    qh, Fg, Ft = ctx.debug("q_half", K), ctx.debug("F_target", K), ctx.debug("F_draft", K)
    if bf16:
        fwd, bwd = P.lsd_get_edge_launch_info(False), P.lsd_get_edge_launch_info(True)
        assert fwd["width"] == w.target.mlip.width and bwd["width"] == w.target.mlip.width     # the target's launches were the last ones
        if w.target.mlip.width == 128:
            # the kernels the cfg5 / cfg4 bench lines time, with a grid that fills the device
            tma = os.environ.get("LSD_EDGE_TMA", "0") not in ("", "0")          # tests/test_gpu_variants.py: the switch reached the kernel
            assert bwd["kernel"] == ("k_edge_rows_tma" if tma else "k_edge_rows")
            assert fwd["kernel"] == ("k_edge_rows" if os.environ.get("LSD_EDGE_FWD4") == "0" else "k_edge_fwd4")
            assert bwd["grid"] >= 148 and fwd["grid"] >= 148
        else:
            assert bwd["kernel"] == fwd["kernel"] == "k_edge_rows_narrow"
    tol = 2e-2 if bf16 else 1e-5
    for j in states:
        Eo, Fo = orc.energy_forces(w, w.target, np.ascontiguousarray(qh[j].T))
        err = _t2_error(Fg[j].T, Fo)
        assert err <= tol, (name, prec, j, err)
    # the draft forces of the same rollout (cfg4 / cfg5: the width-32 one-block network, whose four-team tcgen05 kernels run here
    # in the full-size launch configuration; cfg3: the classical prior alone), one state
    j = states[-1]
    Fo = orc.energy_forces(w, w.draft, np.ascontiguousarray(qh[j].T))[1]
    err = _t2_error(Ft[j].T, Fo)
    assert err <= tol, (name, prec, "draft", j, err)
    P.lsd_rollback(ctx.h, l)
    ctx.close()
