"""The one-kernel draft rollout of tiny systems (tiny_rollout.cu; a0, PAPER.md:584-593 DRAFT_STEP) against the CPU oracle and against
the general launch-per-stage rollout.  -m gpu."""
import dataclasses
import math

import numpy as np
import pytest

import lsd_inputs as L
from lsd_inputs.workloads import Potential, make_mlip

pytestmark = pytest.mark.gpu

FP32_TOL = 1e-5        # north_star: max relative force error <= 1e-5 in fp32 (metric T2)


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_02455_b200 as P
    P.load_library()
    return P


def t2_error(Fg, Fo):
    nrm = np.linalg.norm(Fo, axis=1)
    rms = math.sqrt((Fo**2).sum(1).mean())
    return float((np.linalg.norm(Fg - Fo, axis=1) / np.maximum(nrm, rms)).max())


def _workload(case):
    if case == "cfg1":                       # 64 atoms, periodic, pair prior only
        return L.make_workload("cfg1")
    if case == "cfg2":                       # 22 atoms, vacuum, bonds + angles + (32, 1) network
        return L.make_workload("cfg2")
    if case == "cfg2-9":                     # odd sizes: 9 atoms on 8 CTAs
        return L.make_workload("cfg2", n_chain=9)
    # 64 periodic atoms with a pair prior AND a (32, 1) network in the draft: every atom has ~26 network neighbours, 7 units of 4
    w = L.make_workload("cfg1")
    net = make_mlip(32, 1, 32, 6.5, w.n_species, 77, 0.02)
    return dataclasses.replace(w, draft=Potential(w.draft.pair, w.draft.use_bonded, net), K=6)


@pytest.mark.parametrize("case", ["cfg1", "cfg2", "cfg2-9", "cfg1+net"])
def test_tiny_rollout_matches_oracle_and_general_rollout(P, orc, case, monkeypatch):
    """Draft forces of every step against the oracle at the same q_half (T2, 1e-5), the draft states against Eq. 2 / Eq. 7
    recomputed on the CPU from the oracle's normals, and the whole window against the launch-per-stage rollout (LSD_TINY=0),
    which must agree to fp32 round-off of the forces; decisions of the window must be the same."""
    w = _workload(case)
    K, N = w.K, w.n_atoms
    p0 = orc.initial_momenta(w)
    monkeypatch.delenv("LSD_TINY", raising=False)
    ctx = P.context_from_workload(w, p0=p0, precision=P.LSD_FP32)
    assert P.lsd_tiny_rollout_enabled(ctx.h)
    monkeypatch.setenv("LSD_TINY", "0")
    ref = P.context_from_workload(w, p0=p0, precision=P.LSD_FP32)
    assert not P.lsd_tiny_rollout_enabled(ref.h)
    m = (w.mass_amu * L.AMU)[:, None]
    c1 = math.exp(-w.friction_per_fs * w.dt_fs); b = (1 + c1) * w.dt_fs / 2
    sg = np.sqrt(m * L.K_B * w.temperature_K * (1 - c1 * c1))
    q, p, n = np.array(w.q0, float), np.array(p0, float), 0
    for win in range(3):                                     # the third window replays the captured graph
        n_before = P.lsd_launch_count(ctx.h)
        l, nc = ctx.window(K)
        l2, nc2 = ref.window(K)
        assert (l, nc) == (l2, nc2)
        qh, Ft, yq, yp = (ctx.debug(x, K) for x in ("q_half", "F_draft", "yq", "yp"))
        qh2, Ft2, yq2, yp2 = (ref.debug(x, K) for x in ("q_half", "F_draft", "yq", "yp"))
        for j in range(K):
            Fo = orc.energy_forces(w, w.draft, np.ascontiguousarray(qh[j].T))[1]
            assert t2_error(Ft[j].T, Fo) <= FP32_TOL, (case, win, j)
            if l == 0 or j + 1 < l:                          # (row l of y holds the overridden state x_l after the commit)
                q_prev, p_prev = (q, p) if j == 0 else (yq[j - 1].T, yp[j - 1].T)
                assert np.abs(qh[j].T - (q_prev + w.dt_fs / 2 * p_prev / m)).max() <= 1e-12
                xo = orc.normals(w.seed, n + j + 1, N)
                pn = c1 * p_prev + b * Ft[j].T + sg * xo
                assert np.abs(yp[j].T - pn).max() <= 1e-12 * max(1.0, np.abs(pn).max()), (case, win, j, l)
                assert np.abs(yq[j].T - (qh[j].T + w.dt_fs / 2 * pn / m)).max() <= 1e-12
        assert np.array_equal(qh[0], qh2[0])                 # same base state, same first half-step
        assert t2_error(Ft[0].T, Ft2[0].T) <= 2e-6           # same point, other summation order
        assert np.abs(yq - yq2).max() <= 1e-8                # K steps of fp32 round-off in the forces
        qg, pg, step = ctx.state()
        qr, pr, step_r = ref.state()
        assert step == step_r == n + nc and np.abs(qg - qr).max() <= 1e-8
        P.lsd_set_state(ref.h, qg, pg, step)                       # keep the two trajectories on the same base state
        q, p, n = qg.T.copy(), pg.T.copy(), step
    # one launch for the K draft steps instead of a launch sequence per step
    assert P.lsd_launch_count(ctx.h) < P.lsd_launch_count(ref.h)
    ctx.close(); ref.close()


def test_tiny_rollout_is_not_used_when_draft_equals_target(P):
    """draft == target must reproduce the target bitwise (R8): the rollout then runs the batched kernels."""
    w = L.with_target_as_draft(L.make_workload("cfg2"))
    ctx = P.context_from_workload(w, precision=P.LSD_FP32)
    assert not P.lsd_tiny_rollout_enabled(ctx.h)
    l, nc = ctx.window(w.K)
    assert (l, nc) == (0, w.K)
    ctx.close()


def test_tiny_rollout_with_error_correction_and_skin_flag(P, orc):
    """EC cache in the draft kick (Alg. 3) and the skin check of the window-shared lists, both inside the kernel."""
    w = L.make_workload("cfg2")
    K = w.K
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, p0=p0, precision=P.LSD_FP32)
    assert P.lsd_tiny_rollout_enabled(ctx.h)
    P.lsd_set_error_correction(ctx.h, True)
    dF = 0.05 * np.random.default_rng(3).standard_normal((3, w.n_atoms))
    P.lsd_set_ec_cache(ctx.h, dF)
    ctx.window(K)
    qh, Ft, yp = (ctx.debug(x, K) for x in ("q_half", "F_draft", "yp"))
    m = (w.mass_amu * L.AMU)[:, None]
    c1 = math.exp(-w.friction_per_fs * w.dt_fs); b = (1 + c1) * w.dt_fs / 2
    sg = np.sqrt(m * L.K_B * w.temperature_K * (1 - c1 * c1))
    pn = c1 * p0 + b * (Ft[0].T + dF.T) + sg * orc.normals(w.seed, 1, w.n_atoms)       # the kick uses F~ + dF, the stored F~ is bare
    assert np.abs(yp[0].T - pn).max() <= 1e-12 * max(1.0, np.abs(pn).max())
    Fo = orc.energy_forces(w, w.draft, np.ascontiguousarray(qh[0].T))[1]
    assert t2_error(Ft[0].T, Fo) <= FP32_TOL
    ctx.close()
    tight = P.context_from_workload(w, p0=40.0 * p0, precision=P.LSD_FP32, skin=0.05)   # fast atoms, thin skin
    with pytest.raises(P.LsdError) as ei:
        tight.window(K)
    assert ei.value.status == -7
    tight.close()
