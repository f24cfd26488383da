"""Long run of the default bf16 tcgen05 kernels: thousands of graph-replayed windows in two contexts whose kernels overlap on
the GPU, bit-identical trajectories.  A missing fence or barrier between the generic and the async proxy (the edge kernels write
TMEM / shared-memory operands that tcgen05.mma reads) would show up as a rare wrong sum: the short parity tests would not see
it, this one compares every verdict and the final state of two racing copies of the same trajectory, and a third, serial one.
(compute-sanitizer is closed on the GPU pool this was developed on, so this is the long-run check.)  -m gpu."""
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


@pytest.mark.parametrize("name,kw,K,windows", [("cfg4", {"n_atoms": 1500}, 4, 2000),          # width 128 + width-32 draft, random order
                                               ("cfg3", {"n_grid": 8}, 4, 1000)])              # width 64
def test_soak_two_concurrent_contexts_are_bit_identical(P, orc, name, kw, K, windows):
    import torch
    w = L.make_workload(name, **kw)
    p0 = orc.initial_momenta(w)
    ctxs = [P.context_from_workload(w, k_max=K, precision=P.LSD_BF16_TC, p0=p0) for _ in range(2)]
    assert all(P.lsd_tc_enabled(c.h) for c in ctxs)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    verdicts = [[], []]
    for _ in range(windows):
        for c, s in zip(ctxs, streams):                       # both contexts' rollout + verification are enqueued before either is waited for
            P.lsd_draft_rollout(c.h, K, s)
            P.lsd_verify_window(c.h, K, s)
        for i, (c, s) in enumerate(zip(ctxs, streams)):
            l, nc = P.lsd_transport_accept(c.h, K, s)
            P.lsd_rollback(c.h, l)
            verdicts[i].append((l, nc))
    states = [c.state() for c in ctxs]
    assert verdicts[0] == verdicts[1]
    assert np.array_equal(states[0][0], states[1][0]) and np.array_equal(states[0][1], states[1][1]) and states[0][2] == states[1][2]
    assert np.isfinite(states[0][0]).all() and np.isfinite(states[0][1]).all()
    assert P.lsd_get_stats(ctxs[0].h)["windows"] == windows
    for c in ctxs:
        c.close()
    # the same trajectory alone on the default stream (no overlap with another context)
    solo = P.context_from_workload(w, k_max=K, precision=P.LSD_BF16_TC, p0=p0)
    v = [solo.window(K) for _ in range(windows)]
    q, p, step = solo.state()
    solo.close()
    assert v == verdicts[0] and step == states[0][2]
    assert np.array_equal(q, states[0][0]) and np.array_equal(p, states[0][1])
