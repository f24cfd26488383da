"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.  -m gpu."""
import dataclasses
import math

import numpy as np
import pytest

import lsd_inputs as L
from helpers import edge_set

pytestmark = pytest.mark.gpu

FP32_TOL = 1e-5        # north_star: max relative force error <= 1e-5 in fp32 (metric T2)
BF16_TOL = 2e-2        # north_star: <= 2e-2 in the bf16 tensor-core variant
BF16_NN_TOL = 5e-2     # the network's own force (a tenth of the total): bf16 operands, fp32 accumulation
POS_TOL = 1e-6         # Angstrom per step
BAND = 1e-6            # decisions compared outside |ell - ln u| < 1e-6


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_02455_b200 as P
    P.load_library()                       # fails loudly if the extension is missing
    return P


def soa(x):
    return np.ascontiguousarray(np.asarray(x, np.float64).T)


def t2_error(Fg, Fo):
    """max_i |dF_i| / max(|F_i|, F_rms)   (Fg, Fo: [N,3])"""
    nrm = np.linalg.norm(Fo, axis=1)
    rms = math.sqrt((Fo**2).sum(1).mean())
    return float((np.linalg.norm(Fg - Fo, axis=1) / np.maximum(nrm, rms)).max())


CASES = [("cfg1", {}), ("cfg2", {}), ("cfg3", {"n_grid": 7}), ("cfg4", {"n_atoms": 500}), ("cfg5", {"cells": (4, 4, 4)})]


def _states(w, B, seed=0, unwrap=True):
    rng = np.random.default_rng(seed)
    qs = np.stack([w.q0 + rng.normal(0, 0.02, w.q0.shape) for _ in range(B)])
    if w.periodic and unwrap:                                  # unwrapped positions: move some atoms by whole box vectors
        sh = rng.integers(-2, 3, (len(w.q0[::5]), 3)) * w.box
        qs[:, ::5] += sh
    return qs


@pytest.mark.parametrize("name,kw", CASES)
def test_neighbour_lists_bit_exact(P, orc, name, kw):
    w = L.make_workload(name, **kw)
    B = 3
    ctx = P.context_from_workload(w, k_max=B, precision=P.LSD_FP32)
    qs = _states(w, B, seed=1)
    ctx.forces(P.LSD_TARGET, np.stack([soa(q) for q in qs]))
    kinds = []
    if w.target.mlip is not None:
        kinds.append((0, w.target.mlip.cutoff))
    if w.n_species == 1 and w.target.pair_cutoff() > 0:
        kinds.append((1, w.target.pair_cutoff()))
    assert kinds or name == "cfg2"
    for kind, rc in kinds:
        for b in range(B):
            got = P.lsd_get_neighbors(ctx.h, P.LSD_TARGET, kind, b, w.n_atoms)
            want = orc.neighbors(w, qs[b], rc, "brute")
            assert np.array_equal(got[0], want[0]), (name, kind, b)
            assert np.array_equal(got[1], want[1]) and np.array_equal(got[2], want[2])
    ctx.close()


@pytest.mark.parametrize("name,kw", CASES)
def test_forces_match_oracle_fp32(P, orc, name, kw):
    w = L.make_workload(name, **kw)
    B = 2
    ctx = P.context_from_workload(w, k_max=B, precision=P.LSD_FP32)
    qs = _states(w, B, seed=2)
    for which, pot in ((P.LSD_TARGET, w.target), (P.LSD_DRAFT, w.draft)):
        F, e = ctx.forces(which, np.stack([soa(q) for q in qs]))
        for b in range(B):
            Eo, Fo = orc.energy_forces(w, pot, qs[b])
            err = t2_error(F[b].T, Fo)
            assert err <= (1e-12 if pot.mlip is None else FP32_TOL), (name, which, b, err)
            if pot.mlip is not None:
                Enn = orc.mlip_energy_forces(w, pot.mlip, qs[b], want_forces=False)[0]
                assert e[b].sum() == pytest.approx(Enn, rel=2e-5, abs=1e-6 * w.n_atoms)
    ctx.close()


@pytest.mark.parametrize("name,kw", [("cfg2", {}), ("cfg3", {"n_grid": 7}), ("cfg4", {"n_atoms": 500}), ("cfg5", {"cells": (4, 4, 4)}),
                                     ("cfg5", {"cells": (5, 4, 4)})])
def test_forces_match_oracle_bf16_tensor_core(P, orc, name, kw):
    """LSD_BF16_TC: filter contractions on tcgen05 (bf16 operands, fp32 accumulation) for every network width (128: one
    edge set per tile, 64: two, 32: four); several tiles per chunk, ragged last group, chunks that end inside a state."""
    w = L.make_workload(name, **kw)
    B = 3
    ctx = P.context_from_workload(w, k_max=B, precision=P.LSD_BF16_TC)
    assert P.lsd_tc_enabled(ctx.h)                             # the tcgen05 kernels are the ones that run
    qs = _states(w, B, seed=3)
    Q = np.stack([soa(q) for q in qs])
    for which, pot in ((P.LSD_TARGET, w.target), (P.LSD_DRAFT, w.draft)):
        if pot.mlip is None:
            continue
        F, e = ctx.forces(which, Q)
        F2, _ = ctx.forces(which, Q)
        assert np.array_equal(F, F2)                           # deterministic (no float atomics, fixed summation order)
        F1, _ = ctx.forces(which, Q[1:2])
        assert np.array_equal(F1[0], F[1])                     # batch-invariant: same state alone == inside the batch
        for b in range(B):
            Eo, Fo = orc.energy_forces(w, pot, qs[b])
            Enn, Fnn = orc.mlip_energy_forces(w, pot.mlip, qs[b])
            assert t2_error(F[b].T, Fo) <= BF16_TOL, (name, which, b)
            assert t2_error(F[b].T - (Fo - Fnn), Fnn) <= BF16_NN_TOL, (name, which, b)
            assert e[b].sum() == pytest.approx(Enn, rel=2e-2, abs=2e-3 * w.n_atoms * abs(pot.mlip.alpha))
    ctx.close()


def test_bf16_tensor_core_empty_and_tiny_rows(P, orc):
    """tcgen05 path edge cases: an atom without neighbours inside a chunk, a system much smaller than one tile (vacuum)."""
    w = L.make_workload("cfg2", n_chain=9)
    net = L.make_mlip(128, 2, 32, 5.0, w.n_species, seed=11, alpha=w.target.mlip.alpha)
    w = dataclasses.replace(w, target=dataclasses.replace(w.target, mlip=net))
    q = w.q0.copy()
    q[8] += np.array([40.0, 0, 0])                              # beyond every cutoff: empty MLIP row (still bonded)
    ctx = P.context_from_workload(w, k_max=2, precision=P.LSD_BF16_TC)
    assert P.lsd_tc_enabled(ctx.h)
    for qq in (q, w.q0):                                       # separate calls: the two states are > skin/2 apart
        F, _ = ctx.forces(P.LSD_TARGET, np.stack([soa(qq), soa(qq)]))
        assert np.array_equal(F[0], F[1])
        Fo = orc.energy_forces(w, w.target, qq)[1]
        Fnn = orc.mlip_energy_forces(w, w.target.mlip, qq)[1]
        assert t2_error(F[0].T, Fo) <= BF16_TOL
        assert t2_error(F[0].T - (Fo - Fnn), Fnn) <= BF16_NN_TOL
    ctx.close()


def test_forces_ragged_and_empty_neighbourhoods(P, orc):
    """Edge cases: an isolated atom (no neighbours), rows that are not a multiple of the warp tile, 2-atom system."""
    w = L.make_workload("cfg2", n_chain=5)
    q = w.q0.copy()
    q[4] += np.array([40.0, 0, 0])                              # beyond every cutoff: empty MLIP row (still bonded)
    ctx = P.context_from_workload(w, k_max=1, precision=P.LSD_FP32)
    F, _ = ctx.forces(P.LSD_TARGET, soa(q)[None])
    Fo = orc.energy_forces(w, w.target, q)[1]
    assert t2_error(F[0].T, Fo) <= FP32_TOL
    ctx.close()


def test_lsd_cfg1_end_to_end_decisions_and_positions(P, orc):
    """cfg1 (fp64 both sides): 2,000 committed steps, K = 4.  Accept / first-reject indices bit-exact, positions <= 1e-6 A."""
    w = L.make_workload("cfg1")
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, p0=p0)
    q, p, n = w.q0, p0, 0
    n_rej = 0
    while n < 2000:
        K = min(w.K, 2000 - n)
        r = orc.lsd_window(w, q, p, n, K=K)
        l, nc = ctx.window(K)
        ell, lnu = ctx.debug("ell", K), ctx.debug("lnu", K)
        in_band = np.abs(r["ell"] - r["lnu"]) < BAND
        assert not in_band.any()
        assert (l, nc) == (r["first_reject"], r["n_commit"]), n
        assert np.array_equal(ctx.debug("reject", K), r["reject"])
        assert np.allclose(ell, r["ell"], rtol=0, atol=1e-9) and np.allclose(lnu, r["lnu"], rtol=1e-14)
        q, p, n = r["q"], r["p"], n + nc
        qg, pg, step = ctx.state()
        assert step == n
        assert np.abs(qg.T - q).max() <= POS_TOL
        n_rej += 1 if l else 0
    assert n_rej > 0                                           # the run exercised the override path
    assert np.abs(qg.T - q).max() <= 1e-9 and np.abs(pg.T - p).max() <= 1e-9 * np.abs(p).max() + 1e-12
    st = P.lsd_get_stats(ctx.h)
    assert st["committed_steps"] == 2000 and st["rejections"] == n_rej
    ctx.close()


@pytest.mark.parametrize("name,kw,K", [("cfg2", {}, 16), ("cfg3", {"n_grid": 7}, 4), ("cfg4", {"n_atoms": 500}, 4), ("cfg5", {"cells": (4, 4, 4)}, 4)])
def test_stagewise_transport_parity(P, orc, name, kw, K):
    """T3: the oracle's transport map is fed the GPU's own F~, F, q_half: S1, S2, ell, decisions, l, n_commit and the
    overridden state must match (decisions bit-for-bit outside the band); one integrator step from a common state
    agrees to <= 1e-6 A (T4)."""
    w = L.make_workload(name, **kw)
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, k_max=K, precision=P.LSD_FP32, p0=p0)
    par = orc.params(w)
    q, p, n = w.q0, p0, 0
    for win in range(3):
        l, nc = ctx.window(K)
        qh, Ft, Fg = ctx.debug("q_half", K), ctx.debug("F_draft", K), ctx.debug("F_target", K)
        S1, S2, ell, lnu, rej = (ctx.debug(x, K) for x in ("S1", "S2", "ell", "lnu", "reject"))
        yq, yp, xi = ctx.debug("yq", K), ctx.debug("yp", K), ctx.debug("xi", K)
        first = 0
        for j in range(K):
            p_prev = p if j == 0 else yp_d[j - 1].T
            if j == 0:
                yp_d = yp.copy()
            xo = orc.normals(w.seed, n + j + 1, w.n_atoms)
            assert np.abs(xi[j].T - xo).max() < 1e-12
            # T4: the oracle's integrator from the same state and the GPU's draft force
            qh_o = (q if j == 0 else yq_prev) + w.dt_fs / 2 * p_prev / (w.mass_amu * L.AMU)[:, None]
            assert np.abs(qh[j].T - qh_o).max() <= 1e-12
            u = orc.uniform(w.seed, n + j + 1)
            t = orc.transport_step(w, Ft[j].T, Fg[j].T, xo, u, p_prev, qh[j].T, par)
            assert S1[j] == pytest.approx(t["S1"], rel=1e-10, abs=1e-12) and S2[j] == pytest.approx(t["S2"], rel=1e-10, abs=1e-300)
            assert lnu[j] == pytest.approx(math.log(u), rel=1e-14)
            if abs(t["ell"] - math.log(u)) >= BAND:
                assert rej[j] == t["reject"], (win, j)
            if t["reject"] and not first:
                first = j + 1
                x_q, x_p = t["q"], t["p"]
            if not (first and first == j + 1):
                yq_prev = yq[j].T
                if l == 0 or j + 1 < l:
                    # committed draft state: p' = c1 p + b F~ + sigma xi, q' = q_half + dt/2 p'/m recomputed on the CPU
                    c1 = math.exp(-w.friction_per_fs * w.dt_fs); b = (1 + c1) * w.dt_fs / 2
                    sg = np.sqrt((w.mass_amu * L.AMU) * L.K_B * w.temperature_K * (1 - c1 * c1))[:, None]
                    pn = c1 * p_prev + b * Ft[j].T + sg * xo
                    assert np.abs(yp[j].T - pn).max() <= 1e-9 * np.abs(pn).max()
                    assert np.abs(yq[j].T - (qh[j].T + w.dt_fs / 2 * pn / (w.mass_amu * L.AMU)[:, None])).max() <= POS_TOL * 1e-3
            else:
                break
        assert l == first and nc == (first if first else K)
        qg, pg, step = ctx.state()
        if first:
            assert np.abs(qg.T - x_q).max() <= 1e-9 and np.abs(pg.T - x_p).max() <= 1e-9 * np.abs(x_p).max()
        else:
            assert np.array_equal(qg, yq[K - 1]) and np.array_equal(pg, yp[K - 1])
        q, p, n = qg.T.copy(), pg.T.copy(), step
        assert step == n
    ctx.close()


@pytest.mark.parametrize("name,kw", [("cfg1", {}), ("cfg2", {}), ("cfg3", {"n_grid": 7}), ("cfg5", {"cells": (4, 4, 4)})])
def test_draft_equals_target_accepts_everything(P, orc, name, kw):
    """draft = target: F~ and F are bit-identical (batch-invariant kernels), S2 == 0, acceptance exactly 1."""
    w = L.with_target_as_draft(L.make_workload(name, **kw))
    K = 4
    ctx = P.context_from_workload(w, k_max=K, precision=P.LSD_FP32)
    for _ in range(5):
        l, nc = ctx.window(K)
        assert (l, nc) == (0, K)
        assert np.array_equal(ctx.debug("F_draft", K), ctx.debug("F_target", K))
        assert (ctx.debug("S2", K) == 0).all()
    ctx.close()


def test_committed_trajectory_independent_of_K_and_overlap(P, orc):
    """K-invariance on the device, and lsd_run with the speculative second-stream rollout gives the same trajectory."""
    w = L.make_workload("cfg2")
    p0 = orc.initial_momenta(w)
    finals = []
    for K, mode in ((1, "manual"), (4, "manual"), (16, "manual"), (16, "run_overlap"), (8, "run_serial")):
        ctx = P.context_from_workload(w, k_max=16, precision=P.LSD_FP32, p0=p0)
        if mode == "manual":
            n = 0
            while n < 48:
                _, nc = ctx.window(min(K, 48 - n))
                n += nc
        else:
            P.lsd_run(ctx.h, 48, K, overlap=(mode == "run_overlap"))
        q, p, step = ctx.state()
        assert step == 48
        finals.append((q, p, P.lsd_get_stats(ctx.h)["rejections"]))
        ctx.close()
    assert finals[0][2] > 0
    for q, p, _ in finals[1:]:
        assert np.array_equal(q, finals[0][0]) and np.array_equal(p, finals[0][1])


@pytest.mark.gpu
@pytest.mark.parametrize("name,prec", [("cfg1", "fp64"), ("cfg2", "fp32"), ("cfg2", "bf16")])
def test_cuda_graph_replay_is_bit_identical_to_direct_launches(P, orc, name, prec, monkeypatch):
    """On a non-default stream the rollout / verification / transport launch sequences are captured into CUDA graphs and
    replayed (lsd_api.cu run_graphed); decisions, committed trajectory and the launch count must not depend on it."""
    import torch
    w = L.make_workload(name)
    p0 = orc.initial_momenta(w)
    precision = {"fp64": None, "fp32": P.LSD_FP32, "bf16": P.LSD_BF16_TC}[prec]
    out = []
    for graphs in ("1", "0"):
        monkeypatch.setenv("LSD_GRAPHS", graphs)
        ctx = P.context_from_workload(w, k_max=8, precision=precision, p0=p0)
        stream = torch.cuda.Stream()
        decisions = []
        for i in range(14):                                     # two window lengths: two graphs per stage and slot
            decisions.append(ctx.window(8 if i % 3 else 5, stream))
        P.lsd_run(ctx.h, 40, 8, overlap=True, stream=stream)    # speculative rollouts on the side stream
        q, p, step = ctx.state()
        out.append((decisions, q, p, step, P.lsd_launch_count(ctx.h)))
        ctx.close()
    assert out[0][0] == out[1][0] and out[0][3] == out[1][3]
    assert np.array_equal(out[0][1], out[1][1]) and np.array_equal(out[0][2], out[1][2])
    assert out[0][4] == out[1][4]                               # replayed kernel nodes are counted like direct launches


def test_skin_violation_is_detected(P, orc):
    w = L.make_workload("cfg1")
    ctx = P.context_from_workload(w, k_max=2, skin=0.05)
    qs = np.stack([soa(w.q0), soa(w.q0 + 0.2)])
    with pytest.raises(P.LsdError) as ei:
        ctx.forces(P.LSD_TARGET, qs)
    assert ei.value.status == -7
    ctx.close()


def test_call_order_is_enforced(P):
    w = L.make_workload("cfg1")
    ctx = P.context_from_workload(w)
    with pytest.raises(P.LsdError):
        P.lsd_verify_window(ctx.h, 4)
    P.lsd_draft_rollout(ctx.h, 4)
    with pytest.raises(P.LsdError):
        P.lsd_transport_accept(ctx.h, 4)
    with pytest.raises(P.LsdError):
        P.lsd_draft_rollout(ctx.h, 99)
    ctx.close()


def test_plain_langevin_is_lsd_with_draft_equal_target_and_matches_the_oracle(P, orc):
    """lsd_plain_langevin(LSD_TARGET): the serial baseline.  Same kernels and noise keying as the rollout, so it equals LSD
    with draft = target bit for bit (north_star: "the trajectory equals plain target Langevin under the same noise"), and
    the oracle's plain ABOBA (cfg1, fp64) to round-off."""
    w = L.make_workload("cfg1")
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, p0=p0)
    P.lsd_plain_langevin(ctx.h, P.LSD_TARGET, 50)
    qa, pa, step = ctx.state()
    assert step == 50
    ref = orc.run_aboba(w, w.target, w.q0, p0, 50)
    assert np.abs(qa.T - ref["q"]).max() <= 1e-9 and np.abs(pa.T - ref["p"]).max() <= 1e-9 * np.abs(ref["p"]).max()
    ctx.close()
    wt = L.with_target_as_draft(w)
    ctx = P.context_from_workload(wt, p0=p0)
    n = 0
    while n < 50:
        l, nc = ctx.window(min(4, 50 - n))
        assert l == 0
        n += nc
    qb, pb, _ = ctx.state()
    assert np.array_equal(qa, qb) and np.array_equal(pa, pb)
    with pytest.raises(P.LsdError):
        P.lsd_draft_rollout(ctx.h, 4)
        P.lsd_plain_langevin(ctx.h, P.LSD_TARGET, 4)             # STATE: a drafted window is pending
    ctx.close()


def test_adaptive_lookahead_does_not_change_the_trajectory(P, orc):
    """lsd_run with K = 0 chooses the window length by measurement; with noise keyed by the step index (R5) the committed
    trajectory is the same as with any fixed K, with and without the speculative second-stream rollout."""
    import torch
    w = L.make_workload("cfg2")
    p0 = orc.initial_momenta(w)
    finals = []
    for K, overlap in ((16, False), (0, False), (0, True)):
        ctx = P.context_from_workload(w, k_max=16, precision=P.LSD_FP32, p0=p0)
        stream = torch.cuda.Stream()
        P.lsd_run(ctx.h, 300, K, overlap=overlap, stream=stream)
        q, p, step = ctx.state()
        assert step == 300
        if K == 0:
            assert P.lsd_get_adaptive_k(ctx.h) in (1, 2, 4, 8, 16)
        finals.append((q, p))
        ctx.close()
    for q, p in finals[1:]:
        assert np.array_equal(q, finals[0][0]) and np.array_equal(p, finals[0][1])


@pytest.mark.parametrize("K", [1, 64])
def test_window_length_extremes_match_the_oracle(P, orc, K):
    """K = 1 (every window is one step) and K = LSD_MAX_K = 64 (the largest batch the transport kernels accept), cfg1 in fp64
    on both sides: decisions, first-reject index and committed state follow the oracle."""
    w = L.make_workload("cfg1")
    if K == 64:
        w = dataclasses.replace(w, dt_fs=0.5)                   # 64 steps of 2 fs would leave the Verlet skin (the box allows 0.6 A at most)
    p0 = orc.initial_momenta(w)
    ctx = P.context_from_workload(w, p0=p0, k_max=K)
    q, p, n = w.q0, p0, 0
    for _ in range(6 if K == 64 else 40):
        r = orc.lsd_window(w, q, p, n, K=K)
        l, nc = ctx.window(K)
        assert not (np.abs(r["ell"] - r["lnu"]) < BAND).any()
        assert (l, nc) == (r["first_reject"], r["n_commit"])
        assert np.array_equal(ctx.debug("reject", K), r["reject"])
        q, p, n = r["q"], r["p"], n + nc
        qg, pg, step = ctx.state()
        assert step == n and np.abs(qg.T - q).max() <= POS_TOL
    with pytest.raises(P.LsdError):
        P.lsd_draft_rollout(ctx.h, K + 1)                       # beyond k_max
    ctx.close()
    with pytest.raises(P.LsdError):
        P.context_from_workload(w, p0=p0, k_max=65)            # beyond LSD_MAX_K


def test_nonfinite_forces_are_reported_and_nothing_is_committed(P, orc):
    """Two atoms on top of each other: the pair prior returns inf - inf = NaN for both the draft and the target.  Comparisons
    with NaN are false, so without a check every step of the window would read as accepted and the NaN draft state would be
    committed as target-exact.  The transport kernel raises the non-finite flag instead: LSD_ERR_NONFINITE, base state untouched."""
    w = L.make_workload("cfg1")
    ctx = P.context_from_workload(w, precision=P.LSD_FP32, p0=np.zeros_like(w.q0))
    q, p, step = ctx.state()
    q_bad = q.copy()
    q_bad[:, 1] = q_bad[:, 0]
    P.lsd_set_state(ctx.h, q_bad, np.zeros_like(q_bad), 0)
    with pytest.raises(P.LsdError) as ei:
        ctx.window(w.K)
    assert ei.value.status == -8
    q2, p2, step2 = ctx.state()
    assert step2 == 0 and np.array_equal(q2, q_bad) and np.array_equal(p2, np.zeros_like(q_bad))
    ctx.close()
