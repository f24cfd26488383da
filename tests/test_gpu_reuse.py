"""Work the verification shares with the draft rollout (a1 / a2): the prior forces of the K draft states when draft and target
have the same classical prior, one per-state list for prior and network when their cutoffs coincide.  Both must leave every
bit of the window unchanged.  -m gpu."""
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


@pytest.mark.parametrize("name,kw,prec", [("cfg3", {"n_grid": 7}, "fp32"), ("cfg4", {"n_atoms": 500}, "bf16"), ("cfg5", {"cells": (4, 4, 4)}, "bf16")])
def test_prior_reuse_leaves_the_window_bit_identical(P, orc, name, kw, prec, monkeypatch):
    """LSD_PRIOR_REUSE=0 evaluates the target's prior on the K states again; the default copies the rollout's prior forces
    (same positions, same prior, same batch-invariant kernel).  Target forces, decisions and the committed state must be
    equal bit for bit, over windows that are graph-replayed."""
    w = L.make_workload(name, **kw)
    K = min(w.K, 8)
    p0 = orc.initial_momenta(w)
    out = []
    for reuse in ("1", "0"):
        monkeypatch.setenv("LSD_PRIOR_REUSE", reuse)
        ctx = P.context_from_workload(w, k_max=K, precision=P.LSD_BF16_TC if prec == "bf16" else P.LSD_FP32, p0=p0)
        rec = []
        for _ in range(3):
            l, nc = ctx.window(K)
            rec.append((l, nc, ctx.debug("F_target", K).copy(), ctx.debug("F_draft", K).copy()))
        q, p, step = ctx.state()
        out.append((rec, q, p, step, P.lsd_launch_count(ctx.h)))
        ctx.close()
    (ra, qa, pa, sa, la), (rb, qb, pb, sb, lb) = out
    assert sa == sb and np.array_equal(qa, qb) and np.array_equal(pa, pb)
    for (l1, n1, Fg1, Ft1), (l2, n2, Fg2, Ft2) in zip(ra, rb):
        assert (l1, n1) == (l2, n2) and np.array_equal(Fg1, Fg2) and np.array_equal(Ft1, Ft2)
    assert la < lb                                           # the shared work is really skipped
