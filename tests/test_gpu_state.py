"""State hand-over at the C ABI (include/lsd.h lsd_get_state / lsd_set_state / lsd_get_ec_cache): ordering against the caller's
own device work, exact resume of a trajectory in a new context (checkpoint / resume), and the small
call-order guards (OBABO outputs under force slack, draft lists of a tiny context, caller streams).  -m gpu."""
import numpy as np
import pytest

import lsd_inputs as L

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_02455_b200 as P
    P.load_library()
    return P


def test_device_state_copies_are_ordered_after_the_callers_kernels(P, orc):
    """where = LSD_DEVICE: q, p are torch tensors whose producer still runs on torch's stream when lsd_set_state is called,
    and lsd_get_state writes into tensors an earlier torch kernel still reads.  Both must see the final values."""
    import torch
    w = L.make_workload("cfg3", n_grid=7)
    n = w.n_atoms
    ctx = P.context_from_workload(w, k_max=4, precision=P.LSD_FP32, p0=orc.initial_momenta(w))
    rng = np.random.default_rng(5)
    q_new = np.ascontiguousarray((w.q0 + rng.normal(0, 0.01, w.q0.shape)).T)
    p_new = np.ascontiguousarray(rng.normal(0, 1.0, (3, n)))
    dev = torch.device("cuda:0")
    src_q, src_p = torch.tensor(q_new, device=dev), torch.tensor(p_new, device=dev)
    for trial in range(3):
        qd, pd = torch.zeros((3, n), dtype=torch.float64, device=dev), torch.zeros((3, n), dtype=torch.float64, device=dev)
        torch.cuda.synchronize()
        torch.cuda._sleep(200_000_000)                 # ~0.1 s of busy waiting on torch's current stream ...
        qd.copy_(src_q); pd.copy_(src_p)               # ... then the producers of q, p (not finished when the next line is reached)
        P.lsd_set_state(ctx.h, qd, pd, 7 + trial)
        qh, ph = np.empty((3, n)), np.empty((3, n))
        assert P.lsd_get_state(ctx.h, qh, ph) == 7 + trial
        assert np.array_equal(qh, q_new) and np.array_equal(ph, p_new), trial
        # the other direction: the tensors are still being read (after the sleep) by a torch kernel when get_state overwrites them
        out_q = torch.full((3, n), -1.0, dtype=torch.float64, device=dev)
        torch.cuda._sleep(200_000_000)
        snapshot = out_q.clone()                        # reads out_q after the sleep
        P.lsd_get_state(ctx.h, out_q, None)
        torch.cuda.synchronize()
        assert (snapshot.cpu().numpy() == -1.0).all() and np.array_equal(out_q.cpu().numpy(), q_new)
    ctx.close()


@pytest.mark.parametrize("name,kw,prec,ec", [("cfg2", {}, "fp32", True), ("cfg3", {"n_grid": 7}, "fp32", False),
                                             ("cfg5", {"cells": (4, 4, 4)}, "bf16", True)])
def test_resume_is_exact(P, orc, name, kw, prec, ec):
    """2 W windows in one context == W windows, (q, p, step, EC cache) read out, a NEW context set to them, W more windows: bit
    for bit.  (Whole windows, not step counts: with error correction the trajectory depends on where the windows end, since the
    cache is refreshed once per window, include/lsd.h.)"""
    w = L.make_workload(name, **kw)
    K = min(w.K, 8)
    W = 6
    p0 = orc.initial_momenta(w)
    precision = P.LSD_BF16_TC if prec == "bf16" else P.LSD_FP32

    def fresh():
        c = P.context_from_workload(w, k_max=K, precision=precision, p0=p0)
        if ec:
            P.lsd_set_error_correction(c.h, True)
        return c

    a = fresh()
    verdicts_a = [a.window(K) for _ in range(2 * W)]
    qa, pa, sa = a.state()
    a.close()

    b = fresh()
    verdicts_b = [b.window(K) for _ in range(W)]
    qb, pb, sb = b.state()
    cache = np.zeros((3, w.n_atoms))
    if ec:
        P.lsd_get_ec_cache(b.h, cache)
        assert np.abs(cache).max() > 0
    b.close()
    assert sb == sum(nc for _, nc in verdicts_b) and verdicts_b == verdicts_a[:W]

    c = fresh()
    P.lsd_set_state(c.h, qb, pb, sb)                  # (zeroes the cache: it is restored next)
    if ec:
        P.lsd_set_ec_cache(c.h, cache)
    verdicts_c = [c.window(K) for _ in range(W)]
    qc, pc, sc = c.state()
    c.close()
    assert verdicts_c == verdicts_a[W:] and sc == sa
    assert np.array_equal(qa, qc) and np.array_equal(pa, pc)


def test_obabo_outputs_are_refused_while_force_slack_is_on(P, orc):
    w = L.make_workload("cfg3", n_grid=7)
    ctx = P.context_from_workload(w, k_max=4, precision=P.LSD_FP32, p0=orc.initial_momenta(w))
    P.lsd_set_force_slack(ctx.h, 0.05)
    l, nc = ctx.window(4)
    q, p = np.empty((3, w.n_atoms)), np.empty((3, w.n_atoms))
    with pytest.raises(P.LsdError) as ei:
        P.lsd_get_window_obabo(ctx.h, 1, q, p)
    assert ei.value.status == -4 and "slack" in str(ei.value)
    P.lsd_set_force_slack(ctx.h, 0.0)
    ctx.window(4)
    P.lsd_get_window_obabo(ctx.h, 1, q, p)            # exact method: available again
    assert np.isfinite(p).all()
    ctx.close()


def test_draft_lists_of_a_tiny_context_after_an_explicit_evaluation(P, orc):
    """The one-kernel rollout keeps its neighbour rows on chip, so lsd_get_neighbors(LSD_DRAFT) is refused after it; after an
    lsd_eval_forces(LSD_DRAFT) the list of THAT evaluation is served (and equals the oracle's)."""
    w = L.make_workload("cfg2")
    if w.draft.mlip is None:
        pytest.skip("cfg2's draft has no network list")
    ctx = P.context_from_workload(w, precision=P.LSD_FP32, p0=orc.initial_momenta(w))
    assert P.lsd_tiny_rollout_enabled(ctx.h)
    ctx.window(w.K)
    with pytest.raises(P.LsdError) as ei:
        P.lsd_get_neighbors(ctx.h, P.LSD_DRAFT, 0, 0, w.n_atoms)
    assert ei.value.status == -4
    q = np.ascontiguousarray(w.q0.T)[None]
    ctx.forces(P.LSD_DRAFT, q)
    got = P.lsd_get_neighbors(ctx.h, P.LSD_DRAFT, 0, 0, w.n_atoms)
    want = orc.neighbors(w, w.q0, w.draft.mlip.cutoff, "brute")
    assert all(np.array_equal(g, r) for g, r in zip(got, want))
    ctx.window(w.K)                                    # the next tiny rollout makes the draft lists stale again
    with pytest.raises(P.LsdError):
        P.lsd_get_neighbors(ctx.h, P.LSD_DRAFT, 0, 0, w.n_atoms)
    ctx.close()


def test_plain_langevin_forgets_the_callers_stream(P, orc):
    """lsd_plain_langevin has synchronised `stream` when it returns and keeps no handle of it: the caller destroys the stream,
    and the next state read-back must not touch it."""
    import torch
    w = L.make_workload("cfg3", n_grid=7)
    p0 = orc.initial_momenta(w)
    ref = P.context_from_workload(w, k_max=4, precision=P.LSD_FP32, p0=p0)
    P.lsd_plain_langevin(ref.h, P.LSD_TARGET, 12)
    q_ref, p_ref, _ = ref.state()
    ref.close()
    ctx = P.context_from_workload(w, k_max=4, precision=P.LSD_FP32, p0=p0)
    s = torch.cuda.Stream()
    P.lsd_plain_langevin(ctx.h, P.LSD_TARGET, 12, stream=s)
    del s
    import gc; gc.collect()
    torch.cuda.synchronize()
    q, p, step = ctx.state()
    assert step == 12 and np.array_equal(q, q_ref) and np.array_equal(p, p_ref)
    ctx.close()
