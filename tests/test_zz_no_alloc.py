"""lsd_transport_window_noalloc against the context path (lsd_transport_accept).  -m gpu.

Some users of the library cannot let it allocate GPU memory: their own memory pool already owns the device (a cudaMalloc from
the library would fail or fragment it), or they call from inside another program's step loop where cudaMalloc's device-wide
synchronisation is not acceptable.  For them the library has one entry point that works on caller-owned device arrays plus a
fixed scratch array compiled into the library.  That array is shared by all calls and keeps the previous call's contents, so
the check that matters is: call it twice in a row, with different windows, and both results must equal what the ordinary
(allocating) context path computed from the same forces.

This file is named test_zz_* so that pytest collects it after every other test file: with `pytest -x` a failure here cannot
hide a failure of the older tests.  It must pass alone in a fresh process and after the rest of the suite."""
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
    P.load_library()                       # fails loudly if the extension is missing
    return P


def _windows_from_context(P, orc, name, kw, Ks):
    """Runs one window per entry of Ks through the ordinary path; returns what it computed for each of them."""
    w = L.make_workload(name, **kw)
    ctx = P.context_from_workload(w, k_max=max(Ks), precision=P.LSD_FP32, p0=orc.initial_momenta(w))
    out = []
    for K in Ks:
        n0 = ctx.state()[2]
        l, nc = ctx.window(K)
        out.append(dict(K=K, n0=n0, l=l, nc=nc, Ft=ctx.debug("F_draft", K), Fg=ctx.debug("F_target", K),
                        **{x: ctx.debug(x, K) for x in ("S1", "S2", "ell", "lnu", "reject")}))
    ctx.close()
    return w, out


@pytest.mark.parametrize("name,kw,Ks", [("cfg2", {}, (16, 5)),                 # 22 atoms: one block per step; second call shorter than the first
                                        ("cfg3", {"n_grid": 7}, (3, 8))])      # 1,029 atoms: two blocks per step with a ragged second block; second call longer
def test_noalloc_transport_equals_the_context_path_on_two_calls_in_a_row(P, orc, name, kw, Ks):
    import torch
    w, wins = _windows_from_context(P, orc, name, kw, Ks)
    dev = torch.device("cuda:0")
    n = w.n_atoms
    mass = torch.tensor(np.asarray(w.mass_amu, np.float64), device=dev)
    # every buffer of both calls exists before the first call: the two calls run back to back with nothing in between
    bufs = []
    for d in wins:
        K = d["K"]
        bufs.append(dict(Ft=torch.tensor(d["Ft"], device=dev), Fg=torch.tensor(d["Fg"], device=dev),
                         stats=torch.full((4, K), float("nan"), dtype=torch.float64, device=dev),
                         reject=torch.full((K,), -1, dtype=torch.int32, device=dev),
                         verdict=torch.full((3,), -1, dtype=torch.int32, device=dev)))
    torch.cuda.synchronize()
    for d, b in zip(wins, bufs):
        P.lsd_transport_window_noalloc(n, d["K"], int(w.seed), int(d["n0"]), w.temperature_K, w.friction_per_fs, w.dt_fs,
                                       mass, b["Ft"], b["Fg"], b["stats"], b["reject"], b["verdict"])
    torch.cuda.synchronize()
    for d, b in zip(wins, bufs):
        S1, S2, ell, lnu = b["stats"].cpu().numpy()
        # the tolerances of test_stagewise_transport_parity (same arithmetic in the same order: in practice the bits agree)
        np.testing.assert_allclose(S1, d["S1"], rtol=1e-10, atol=1e-12)
        np.testing.assert_allclose(S2, d["S2"], rtol=1e-10, atol=1e-300)
        np.testing.assert_allclose(ell, d["ell"], rtol=1e-10, atol=1e-12)
        np.testing.assert_allclose(lnu, d["lnu"], rtol=1e-14, atol=0)
        assert np.array_equal(b["reject"].cpu().numpy(), d["reject"])
        assert b["verdict"].cpu().tolist() == [d["l"], d["nc"], 0]
        assert (d["S2"] > 0).all()                              # the comparison is not one of zeros


def test_noalloc_transport_refuses_sizes_beyond_its_scratch(P):
    import torch
    dev = torch.device("cuda:0")
    K = P.LSD_NOALLOC_MAX_K + 1
    z = torch.zeros((K, 3, 4), dtype=torch.float64, device=dev)
    args = (torch.ones(4, dtype=torch.float64, device=dev), z, z, torch.zeros((4, K), dtype=torch.float64, device=dev),
            torch.zeros(K, dtype=torch.int32, device=dev), torch.zeros(3, dtype=torch.int32, device=dev))
    with pytest.raises(P.LsdError) as ei:
        P.lsd_transport_window_noalloc(4, K, 1, 0, 300.0, 0.01, 0.5, *args)
    assert ei.value.status == -1 and "LSD_NOALLOC_MAX_K" in str(ei.value)
    with pytest.raises(P.LsdError) as ei:
        P.lsd_transport_window_noalloc(P.LSD_NOALLOC_MAX_ATOMS + 1, 2, 1, 0, 300.0, 0.01, 0.5, *args)
    assert ei.value.status == -1 and "LSD_NOALLOC_MAX_ATOMS" in str(ei.value)
    torch.cuda.synchronize()                                    # nothing was launched, nothing faulted
