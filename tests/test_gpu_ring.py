"""Ring of window slots (Alg. 2 semantics on one device): lsd_set_window_slots, lsd_run with a
pipeline depth.  -m gpu."""
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


def test_window_ring_depth_does_not_change_the_committed_trajectory(P, orc):
    """SURVEY 8(f) rank 3 / Alg. 2 on one device: with W window slots lsd_run keeps up to W - 1 speculative
    windows drafted ahead on the second stream and flushes them all on a rejection (:611-612).  The committed trajectory is a
    function of (x0, seed) only (R5): depth 0, 1, 3 and 7 give the same bits, on a workload with rejections (cfg2) and on one
    that accepts nearly everything (cfg1), and the oracle's own LSD run agrees on cfg1 (fp64 both sides)."""
    for name, K, steps in (("cfg2", 4, 60), ("cfg1", 4, 120)):
        w = L.make_workload(name)
        p0 = orc.initial_momenta(w)
        finals = []
        for slots, depth in ((2, 0), (2, 1), (4, 3), (8, 7)):
            ctx = P.context_from_workload(w, k_max=K, precision=P.LSD_FP32, p0=p0)
            if slots != 2:
                P.lsd_set_window_slots(ctx.h, slots)
            P.lsd_run(ctx.h, steps, K, overlap=depth)
            q, p, step = ctx.state()
            st = P.lsd_get_stats(ctx.h)
            assert step == steps and st["committed_steps"] == steps
            finals.append((q, p, st["rejections"], st["windows"]))
            ctx.close()
        assert finals[0][2] > 0
        for q, p, rej, _ in finals[1:]:
            assert np.array_equal(q, finals[0][0]) and np.array_equal(p, finals[0][1]) and rej == finals[0][2]
        if name == "cfg1":
            ref = orc.run_lsd(w, w.q0, p0, steps, K)
            assert np.abs(finals[0][0].T - ref["q"]).max() <= 1e-9


def test_window_ring_call_order(P):
    """W slots hold W drafted, unverified windows; one more is refused (LSD_ERR_STATE); a rejection flushes all of them."""
    w = L.make_workload("cfg2")
    ctx = P.context_from_workload(w, k_max=4, precision=P.LSD_FP32)
    P.lsd_draft_rollout(ctx.h, 4); P.lsd_draft_rollout(ctx.h, 4)
    with pytest.raises(P.LsdError) as ei:
        P.lsd_draft_rollout(ctx.h, 4)
    assert ei.value.status == -4
    P.lsd_set_window_slots(ctx.h, 3)                         # (drops the drafted windows)
    for _ in range(3):
        P.lsd_draft_rollout(ctx.h, 4)
    with pytest.raises(P.LsdError) as ei:
        P.lsd_draft_rollout(ctx.h, 4)
    assert ei.value.status == -4
    flushed = False
    for _ in range(40):                                      # verify windows until one rejects: every speculative window goes
        P.lsd_verify_window(ctx.h, 4)
        l, nc = P.lsd_transport_accept(ctx.h, 4)
        P.lsd_rollback(ctx.h, l)
        if l:
            with pytest.raises(P.LsdError):
                P.lsd_verify_window(ctx.h, 4)                # nothing drafted any more
            flushed = True
            break
        P.lsd_draft_rollout(ctx.h, 4)                        # refill the ring
    assert flushed
    with pytest.raises(P.LsdError):
        P.lsd_set_window_slots(ctx.h, 9)
    ctx.close()
