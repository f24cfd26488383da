"""ctypes binding with the same names as include/lsd.h.  Argument marshalling only.

Bulk arguments may be numpy arrays (host) or torch tensors (host or CUDA); the `where` flag of the C call is
derived from them.  Vectors over atoms are component-major [3][N] float64 (see include/lsd.h)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblsd_b200.so")

LSD_HOST, LSD_DEVICE = 0, 1
LSD_FP32, LSD_BF16_TC = 1, 2
LSD_DRAFT, LSD_TARGET = 0, 1
DBG = dict(q_half=0, F_draft=1, F_target=2, S1=3, S2=4, ell=5, lnu=6, reject=7, xi=8, yp=9, yq=10)
_STATUS = {0: "LSD_OK", -1: "LSD_ERR_INVALID_ARG", -2: "LSD_ERR_CUDA", -3: "LSD_ERR_OOM", -4: "LSD_ERR_STATE",
           -5: "LSD_ERR_UNSUPPORTED", -6: "LSD_ERR_NBR_OVERFLOW", -7: "LSD_ERR_SKIN_VIOLATED", -8: "LSD_ERR_NONFINITE"}

EXPORTED_SYMBOLS = ["lsd_init", "lsd_destroy", "lsd_last_error", "lsd_draft_rollout", "lsd_verify_window", "lsd_transport_accept",
                    "lsd_rollback", "lsd_run", "lsd_get_state", "lsd_set_state", "lsd_get_stats", "lsd_get_window_state",
                    "lsd_get_window_debug", "lsd_eval_forces", "lsd_get_neighbors", "lsd_set_skin", "lsd_launch_count", "lsd_version", "lsd_profile", "lsd_get_profile", "lsd_get_edge_count", "lsd_tc_enabled",
                    "lsd_set_error_correction", "lsd_get_ec_cache", "lsd_set_ec_cache", "lsd_plain_langevin", "lsd_get_adaptive_k",
                    "lsd_get_window_obabo", "lsd_get_edge_launch_info", "lsd_measure_fma_peak", "lsd_set_force_slack", "lsd_tiny_rollout_enabled", "lsd_set_window_slots",
                    "lsd_transport_window_noalloc", "lsd_noalloc_last_error"]


class LsdError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _System(C.Structure):
    _fields_ = [("n_atoms", C.c_int32), ("n_species", C.c_int32), ("periodic", C.c_int32), ("box", C.c_double * 3),
                ("species", C.c_void_p), ("mass_amu", C.c_void_p),
                ("n_bonds", C.c_int32), ("bonds", C.c_void_p), ("bond_k", C.c_void_p), ("bond_r0", C.c_void_p),
                ("n_angles", C.c_int32), ("angles", C.c_void_p), ("angle_k", C.c_void_p), ("angle_theta0", C.c_void_p)]


class _Mlip(C.Structure):
    _fields_ = [("width", C.c_int32), ("n_blocks", C.c_int32), ("n_rbf", C.c_int32), ("n_species", C.c_int32),
                ("cutoff", C.c_double), ("energy_scale", C.c_double), ("weights", C.c_void_p)]


class _Potential(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("use_bonded", C.c_int32), ("pair", C.c_void_p), ("mlip", _Mlip)]


class _Config(C.Structure):
    _fields_ = [("temperature_K", C.c_double), ("friction_per_fs", C.c_double), ("dt_fs", C.c_double), ("seed", C.c_uint64),
                ("scheme", C.c_int32), ("precision", C.c_int32), ("k_max", C.c_int32), ("skin", C.c_double)]


class _Stats(C.Structure):
    _fields_ = [("windows", C.c_int64), ("committed_steps", C.c_int64), ("rejections", C.c_int64), ("beta_sum", C.c_double), ("step", C.c_int64)]


_lib = None


def library_path() -> str:
    return _SO


def load_library():
    """dlopen liblsd_b200.so (fails loudly if it has not been built: no fallback path exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} is missing: build it with `python -m paper_2606_02455_b200.build` (there is no CPU fallback)")
        L = C.CDLL(_SO)
        L.lsd_last_error.restype = C.c_char_p
        L.lsd_last_error.argtypes = [C.c_void_p]
        L.lsd_version.restype = C.c_char_p
        L.lsd_launch_count.restype = C.c_int64
        L.lsd_launch_count.argtypes = [C.c_void_p]
        L.lsd_destroy.restype = None
        L.lsd_destroy.argtypes = [C.c_void_p]
        L.lsd_noalloc_last_error.restype = C.c_char_p
        L.lsd_noalloc_last_error.argtypes = []
        _lib = L
    return _lib


def _ptr(a):
    """(address, where) of a numpy array or torch tensor; None -> (None, LSD_HOST)."""
    if a is None:
        return None, LSD_HOST
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data), LSD_HOST
    assert a.is_contiguous()                      # torch tensor
    return C.c_void_p(a.data_ptr()), (LSD_DEVICE if a.is_cuda else LSD_HOST)


def _stream(s):
    if s is None:
        return C.c_void_p(0)
    return C.c_void_p(int(getattr(s, "cuda_stream", s)))


def _check(h, status):
    if status != 0:
        msg = load_library().lsd_last_error(h)
        raise LsdError(status, msg.decode() if msg else "")


# ------------------------------------------------------------------------------------------- C-ABI wrappers
def lsd_version() -> str:
    return load_library().lsd_version().decode()


def lsd_init(cfg: dict, system: dict, draft: dict, target: dict, q0: np.ndarray, p0=None):
    """Returns an opaque handle.  Dict fields follow lsd_config / lsd_system / lsd_potential; arrays are host numpy."""
    L = load_library()
    keep = []

    def arr(x, dt):
        if x is None:
            return None
        a = np.ascontiguousarray(x, dtype=dt)
        keep.append(a)
        return a.ctypes.data

    def pot(p):
        m = p.get("mlip")
        ml = _Mlip(0, 0, 0, 0, 0.0, 0.0, None) if m is None else _Mlip(m["width"], m["n_blocks"], m["n_rbf"], m["n_species"], m["cutoff"],
                                                                       m["energy_scale"], arr(m["weights"], np.float64))
        return _Potential(system["n_species"], int(bool(p["use_bonded"])), arr(p["pair"], np.float64), ml)

    bonds, angles = system.get("bonds"), system.get("angles")
    nb = 0 if bonds is None else len(bonds)
    na = 0 if angles is None else len(angles)
    s = _System(system["n_atoms"], system["n_species"], int(bool(system["periodic"])), (C.c_double * 3)(*[float(v) for v in system["box"]]),
                arr(system["species"], np.int32), arr(system["mass_amu"], np.float64),
                nb, arr(bonds, np.int32) if nb else None, arr(system.get("bond_k"), np.float64) if nb else None, arr(system.get("bond_r0"), np.float64) if nb else None,
                na, arr(angles, np.int32) if na else None, arr(system.get("angle_k"), np.float64) if na else None, arr(system.get("angle_theta0"), np.float64) if na else None)
    c = _Config(cfg["temperature_K"], cfg["friction_per_fs"], cfg["dt_fs"], cfg["seed"], cfg.get("scheme", 0), cfg.get("precision", LSD_FP32),
                cfg["k_max"], cfg.get("skin", 0.5))
    d, t = pot(draft), pot(target)
    h = C.c_void_p()
    q0 = np.ascontiguousarray(q0, np.float64)
    p0 = None if p0 is None else np.ascontiguousarray(p0, np.float64)
    st = L.lsd_init(C.byref(c), C.byref(s), C.byref(d), C.byref(t), C.c_void_p(q0.ctypes.data), C.c_void_p(p0.ctypes.data) if p0 is not None else None, C.byref(h))
    _check(None, st)
    return h


def lsd_destroy(h):
    load_library().lsd_destroy(h)


def lsd_draft_rollout(h, K, stream=None):
    _check(h, load_library().lsd_draft_rollout(h, C.c_int32(K), _stream(stream)))


def lsd_verify_window(h, K, stream=None):
    _check(h, load_library().lsd_verify_window(h, C.c_int32(K), _stream(stream)))


def lsd_transport_accept(h, K, stream=None):
    fr, nc = C.c_int32(), C.c_int32()
    _check(h, load_library().lsd_transport_accept(h, C.c_int32(K), _stream(stream), C.byref(fr), C.byref(nc)))
    return fr.value, nc.value


def lsd_rollback(h, first_reject):
    _check(h, load_library().lsd_rollback(h, C.c_int32(first_reject)))


def lsd_run(h, n_steps, K, overlap=True, stream=None):
    _check(h, load_library().lsd_run(h, C.c_int64(n_steps), C.c_int32(K), C.c_int32(int(overlap)), _stream(stream)))


def lsd_get_adaptive_k(h) -> int:
    return int(load_library().lsd_get_adaptive_k(h))


def lsd_plain_langevin(h, which, n_steps, stream=None):
    _check(h, load_library().lsd_plain_langevin(h, C.c_int32(which), C.c_int64(n_steps), _stream(stream)))


def lsd_get_state(h, q=None, p=None):
    """Fills q, p ([3][N]; numpy or torch) and returns the committed step index."""
    step = C.c_int64()
    (qp, wq), (pp, wp) = _ptr(q), _ptr(p)
    assert q is None or p is None or wq == wp
    _check(h, load_library().lsd_get_state(h, qp, pp, C.byref(step), C.c_int32(wq if q is not None else wp)))
    return step.value


def lsd_set_state(h, q, p, step):
    (qp, wq), (pp, wp) = _ptr(q), _ptr(p)
    assert wq == wp
    _check(h, load_library().lsd_set_state(h, qp, pp, C.c_int64(step), C.c_int32(wq)))


def lsd_set_error_correction(h, enable: bool):
    _check(h, load_library().lsd_set_error_correction(h, C.c_int32(int(bool(enable)))))


def lsd_set_force_slack(h, eps_F: float):
    _check(h, load_library().lsd_set_force_slack(h, C.c_double(eps_F)))


def lsd_get_ec_cache(h, dF):
    ptr, where = _ptr(dF)
    _check(h, load_library().lsd_get_ec_cache(h, ptr, C.c_int32(where)))


def lsd_set_ec_cache(h, dF):
    ptr, where = _ptr(dF)
    _check(h, load_library().lsd_set_ec_cache(h, ptr, C.c_int32(where)))


def lsd_get_stats(h) -> dict:
    s = _Stats()
    _check(h, load_library().lsd_get_stats(h, C.byref(s)))
    return {k: getattr(s, k) for k, _ in _Stats._fields_}


def lsd_get_window_state(h, j, q=None, p=None):
    (qp, wq), (pp, wp) = _ptr(q), _ptr(p)
    _check(h, load_library().lsd_get_window_state(h, C.c_int32(j), qp, pp, C.c_int32(wq if q is not None else wp)))


def lsd_get_window_obabo(h, j, q=None, p=None):
    (qp, wq), (pp, wp) = _ptr(q), _ptr(p)
    _check(h, load_library().lsd_get_window_obabo(h, C.c_int32(j), qp, pp, C.c_int32(wq if q is not None else wp)))


def lsd_get_window_debug(h, what, out):
    ptr, where = _ptr(out)
    _check(h, load_library().lsd_get_window_debug(h, C.c_int32(DBG[what] if isinstance(what, str) else what), ptr, C.c_int32(where)))


def lsd_eval_forces(h, which, q, F, energy_nn=None, stream=None):
    """q, F: [B][3][N] float64 (numpy or torch, same residence)."""
    (qp, wq), (fp, wf), (ep, we) = _ptr(q), _ptr(F), _ptr(energy_nn)
    assert wq == wf and (energy_nn is None or we == wq)
    _check(h, load_library().lsd_eval_forces(h, C.c_int32(which), C.c_int32(q.shape[0]), qp, fp, ep, C.c_int32(wq), _stream(stream)))


def lsd_get_neighbors(h, which, kind, b, n_atoms):
    L = load_library()
    start = np.zeros(n_atoms + 1, np.int64)
    ne = C.c_int64()
    cap = 0
    idx, sh = np.zeros(1, np.int32), np.zeros((1, 3), np.int8)
    for _ in range(2):
        _check(h, L.lsd_get_neighbors(h, C.c_int32(which), C.c_int32(kind), C.c_int32(b), C.c_int64(cap), C.c_void_p(start.ctypes.data),
                                      C.c_void_p(idx.ctypes.data), C.c_void_p(sh.ctypes.data), C.byref(ne)))
        if ne.value <= cap:
            break
        cap = int(ne.value)
        idx, sh = np.zeros(max(cap, 1), np.int32), np.zeros((max(cap, 1), 3), np.int8)
    return start, idx[: ne.value].copy(), sh[: ne.value].copy()


def lsd_get_edge_count(h, which, kind, n_states) -> int:
    t = C.c_int64()
    _check(h, load_library().lsd_get_edge_count(h, C.c_int32(which), C.c_int32(kind), C.c_int32(n_states), C.byref(t)))
    return int(t.value)


def lsd_set_skin(h, skin):
    _check(h, load_library().lsd_set_skin(h, C.c_double(skin)))


PROFILE_CLASSES = ["neighbor", "prior", "mlip_dense", "mlip_edge_fwd", "mlip_edge_bwd", "integrator", "transport", "draft_mlip"]


def lsd_profile(h, enable=True):
    _check(h, load_library().lsd_profile(h, C.c_int32(int(enable))))


def lsd_get_profile(h) -> dict:
    ms, cnt = (C.c_double * 8)(), (C.c_int64 * 8)()
    _check(h, load_library().lsd_get_profile(h, ms, cnt))
    return {name: dict(ms=ms[i], launches=cnt[i]) for i, name in enumerate(PROFILE_CLASSES)}


EDGE_KERNELS = {0: None, 4: "k_edge_rows", 7: "k_edge_rows_narrow", 8: "k_edge_fwd4", 9: "k_edge_rows_tma"}


def lsd_get_edge_launch_info(backward: bool) -> dict:
    out = (C.c_int32 * 5)()
    _check(None, load_library().lsd_get_edge_launch_info(C.c_int32(int(bool(backward))), out))
    return dict(kernel=EDGE_KERNELS.get(out[0], out[0]), atoms_per_chunk=out[1], threads=out[2], grid=out[3], width=out[4])


def lsd_measure_fma_peak(kind: int, stream=None) -> float:
    """Measured FMA peak of the current device in TFLOP/s (kind 0 = fp32, 1 = fp64)."""
    out = C.c_double()
    _check(None, load_library().lsd_measure_fma_peak(C.c_int32(kind), _stream(stream), C.byref(out)))
    return float(out.value)


LSD_NOALLOC_MAX_K, LSD_NOALLOC_MAX_ATOMS = 64, 1 << 28


def lsd_transport_window_noalloc(n_atoms, K, seed, n0, temperature_K, friction_per_fs, dt_fs, mass_amu, F_draft, F_target,
                                 stats, reject, verdict, stream=None):
    """Accept / reject decisions of one drafted window from forces already on the device, for callers that must not allocate
    GPU memory (a host program whose pool owns the device; a callback that may not trigger cudaMalloc's device-wide
    synchronisation): see include/lsd.h.  Every array is a CUDA tensor the caller owns: mass_amu [n] f64, F_draft / F_target
    [K][3][n] f64 in, stats [4][K] f64 (S1 | S2 | ell | ln u), reject [K] i32, verdict [3] i32 out.  Asynchronous on `stream`;
    calls that may overlap on the GPU race on the library's fixed scratch array.  This wrapper allocates nothing either."""
    ptrs = []
    for a in (mass_amu, F_draft, F_target, stats, reject, verdict):
        ptr, where = _ptr(a)
        if where != LSD_DEVICE:
            raise LsdError(-1, "lsd_transport_window_noalloc takes device (CUDA) tensors only")
        ptrs.append(ptr)
    L = load_library()
    st = L.lsd_transport_window_noalloc(C.c_int32(n_atoms), C.c_int32(K), C.c_uint64(seed), C.c_uint64(n0), C.c_double(temperature_K),
                                        C.c_double(friction_per_fs), C.c_double(dt_fs), *ptrs, _stream(stream))
    if st != 0:
        raise LsdError(st, L.lsd_noalloc_last_error().decode())


def lsd_tc_enabled(h) -> bool:
    return bool(load_library().lsd_tc_enabled(h))


def lsd_set_window_slots(h, n_slots: int):
    _check(h, load_library().lsd_set_window_slots(h, C.c_int32(n_slots)))


def lsd_tiny_rollout_enabled(h) -> bool:
    return bool(load_library().lsd_tiny_rollout_enabled(h))


def lsd_launch_count(h) -> int:
    return int(load_library().lsd_launch_count(h))


# ------------------------------------------------------------------------------------------- convenience
def _pot_dict(p):
    m = None
    if p.mlip is not None:
        m = dict(width=p.mlip.width, n_blocks=p.mlip.n_blocks, n_rbf=p.mlip.n_rbf, n_species=p.mlip.n_species, cutoff=p.mlip.cutoff,
                 energy_scale=p.mlip.alpha, weights=p.mlip.weights)
    return dict(use_bonded=p.use_bonded, pair=p.pair, mlip=m)


def context_from_workload(w, k_max=None, precision=None, p0=None, seed=None, draft=None, target=None, skin=None):
    """Marshal an lsd_inputs.Workload (positions [N,3]) into lsd_init.  p0: [N,3] or None (Maxwell-Boltzmann on the device)."""
    prec = precision if precision is not None else (LSD_BF16_TC if w.precision == "bf16" else LSD_FP32)
    cfg = dict(temperature_K=w.temperature_K, friction_per_fs=w.friction_per_fs, dt_fs=w.dt_fs, seed=int(w.seed if seed is None else seed),
               precision=prec, k_max=int(k_max or w.K), skin=float(w.skin if skin is None else skin))
    system = dict(n_atoms=w.n_atoms, n_species=w.n_species, periodic=w.periodic, box=w.box, species=w.species, mass_amu=w.mass_amu,
                  bonds=w.bonds, bond_k=w.bond_k, bond_r0=w.bond_r0, angles=w.angles, angle_k=w.angle_k, angle_theta0=w.angle_theta0)
    q0 = np.ascontiguousarray(np.asarray(w.q0, np.float64).T)
    p0s = None if p0 is None else np.ascontiguousarray(np.asarray(p0, np.float64).T)
    return Context(lsd_init(cfg, system, _pot_dict(draft or w.draft), _pot_dict(target or w.target), q0, p0s), w.n_atoms)


class Context:
    """Owns a handle; methods forward to the functions above."""

    def __init__(self, handle, n_atoms):
        self.h, self.n = handle, n_atoms

    def close(self):
        if self.h is not None:
            lsd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def window(self, K, stream=None):
        """rollout -> verify -> transport -> rollback; returns (first_reject, n_commit)."""
        lsd_draft_rollout(self.h, K, stream)
        lsd_verify_window(self.h, K, stream)
        l, nc = lsd_transport_accept(self.h, K, stream)
        lsd_rollback(self.h, l)
        return l, nc

    def state(self):
        q, p = np.empty((3, self.n)), np.empty((3, self.n))
        step = lsd_get_state(self.h, q, p)
        return q, p, step

    def debug(self, what, K):
        shape = (K, 3, self.n) if what in ("q_half", "F_draft", "F_target", "xi", "yp", "yq") else (K,)
        out = np.empty(shape, np.int32 if what == "reject" else np.float64)
        lsd_get_window_debug(self.h, what, out)
        return out

    def forces(self, which, q):
        """q: [B][3][N] numpy -> (F [B][3][N], e_nn [B][N])."""
        q = np.ascontiguousarray(q, np.float64)
        F, e = np.empty_like(q), np.empty((q.shape[0], self.n))
        lsd_eval_forces(self.h, which, q, F, e)
        return F, e
