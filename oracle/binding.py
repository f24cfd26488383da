"""ctypes binding of oracle/lsd_oracle.c (fp64, plain C).  Builds the shared object with gcc on
first use (and whenever the source is newer).  Arrays are [N,3] float64 numpy arrays."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lsd_oracle.c")
_SO = os.path.join(_HERE, "liblsd_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """gcc -O3, no FMA contraction (T1: neighbour tests are fma-free), OpenMP over atoms."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O3", "-march=x86-64-v2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
               "-std=c11", "-o", tmp, _SRC, "-lm"]
        subprocess.check_call(cmd)
        os.replace(tmp, _SO)
    return _SO


class _Mlip(C.Structure):
    _fields_ = [("width", C.c_int32), ("n_blocks", C.c_int32), ("n_rbf", C.c_int32), ("n_species", C.c_int32),
                ("cutoff", C.c_double), ("alpha", C.c_double), ("w", C.POINTER(C.c_double))]


class _Potential(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("use_bonded", C.c_int32), ("pair", C.POINTER(C.c_double)), ("mlip", _Mlip)]


class _System(C.Structure):
    _fields_ = [("n", C.c_int32), ("periodic", C.c_int32), ("box", C.c_double * 3),
                ("species", C.POINTER(C.c_int32)), ("mass_amu", C.POINTER(C.c_double)),
                ("n_bonds", C.c_int32), ("bonds", C.POINTER(C.c_int32)), ("bond_k", C.POINTER(C.c_double)), ("bond_r0", C.POINTER(C.c_double)),
                ("n_angles", C.c_int32), ("angles", C.POINTER(C.c_int32)), ("angle_k", C.POINTER(C.c_double)), ("angle_t0", C.POINTER(C.c_double))]


class _Params(C.Structure):
    _fields_ = [("temperature_K", C.c_double), ("friction_per_fs", C.c_double), ("dt_fs", C.c_double), ("seed", C.c_uint64)]


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def lib():
    global _lib
    with _lock:
        if _lib is None:
            build()
            try:
                L = C.CDLL(_SO)
            except OSError:
                build(force=True)
                L = C.CDLL(_SO)
            L.orc_energy_forces.restype = C.c_double
            L.orc_mlip_energy_forces.restype = C.c_double
            L.orc_uniform.restype = C.c_double
            L.orc_uniform.argtypes = [C.c_uint64, C.c_uint64]
            L.orc_neighbors_brute.restype = C.c_int64
            L.orc_neighbors_cell.restype = C.c_int64
            L.orc_lsd_window.restype = C.c_int32
            L.orc_transport_step.restype = C.c_int32
            L.orc_run_lsd.restype = C.c_int64
            L.orc_lsd_window_ec.restype = C.c_int32
            L.orc_run_lsd_ec.restype = C.c_int64
            L.orc_rejection_probability.restype = C.c_double
            L.orc_rejection_probability.argtypes = [C.c_double]
            _lib = L
    return _lib


def set_threads(n: int) -> None:
    os.environ["OMP_NUM_THREADS"] = str(n)


class System:
    """Keeps the numpy arrays alive behind the C struct."""

    def __init__(self, w):
        self.n = int(w.n_atoms)
        self._keep = dict(
            species=np.ascontiguousarray(w.species, np.int32), mass=np.ascontiguousarray(w.mass_amu, np.float64),
            bonds=np.ascontiguousarray(w.bonds, np.int32).reshape(-1), bond_k=np.ascontiguousarray(w.bond_k, np.float64),
            bond_r0=np.ascontiguousarray(w.bond_r0, np.float64), angles=np.ascontiguousarray(w.angles, np.int32).reshape(-1),
            angle_k=np.ascontiguousarray(w.angle_k, np.float64), angle_t0=np.ascontiguousarray(w.angle_theta0, np.float64))
        k = self._keep
        self.c = _System(self.n, int(bool(w.periodic)), (C.c_double * 3)(*[float(x) for x in w.box]),
                         _ip(k["species"]), _dp(k["mass"]),
                         len(w.bonds), _ip(k["bonds"]), _dp(k["bond_k"]), _dp(k["bond_r0"]),
                         len(w.angles), _ip(k["angles"]), _dp(k["angle_k"]), _dp(k["angle_t0"]))


class Pot:
    def __init__(self, pot):
        self._pair = np.ascontiguousarray(pot.pair, np.float64)
        ns = self._pair.shape[0]
        if pot.mlip is not None:
            m = pot.mlip
            self._w = np.ascontiguousarray(m.weights, np.float64)
            ml = _Mlip(m.width, m.n_blocks, m.n_rbf, m.n_species, m.cutoff, m.alpha, _dp(self._w))
        else:
            ml = _Mlip(0, 0, 0, 0, 0.0, 0.0, None)
        self.c = _Potential(ns, int(bool(pot.use_bonded)), _dp(self._pair), ml)


def params(w, seed=None, temperature_K=None, friction_per_fs=None, dt_fs=None):
    return _Params(float(w.temperature_K if temperature_K is None else temperature_K),
                   float(w.friction_per_fs if friction_per_fs is None else friction_per_fs),
                   float(w.dt_fs if dt_fs is None else dt_fs), int(w.seed if seed is None else seed))


# ------------------------------------------------------------------------------------ wrappers
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def normals(seed, step, n, tag=0):
    xi = np.empty((n, 3))
    lib().orc_normals(C.c_uint64(seed), C.c_uint64(step), C.c_int32(n), C.c_uint32(tag), _dp(xi))
    return xi


def uniform(seed, step):
    return float(lib().orc_uniform(int(seed), int(step)))


def rejection_probability(delta_norm):
    return float(lib().orc_rejection_probability(float(delta_norm)))


def initial_momenta(w, seed=None):
    s = System(w)
    p = np.empty((s.n, 3))
    par = params(w, seed)
    lib().orc_initial_momenta(C.byref(s.c), C.byref(par), _dp(p))
    return p


def neighbors(w, q, rc, method="brute"):
    """Directed edge set {(i, j, shift)}: returns (start[N+1] int64, idx int32, shifts int8 [E,3])."""
    s = System(w)
    q = np.ascontiguousarray(q, np.float64)
    fn = lib().orc_neighbors_brute if method == "brute" else lib().orc_neighbors_cell
    start = np.empty(s.n + 1, np.int64)
    cap = max(1024, s.n * 64)
    while True:
        idx = np.empty(cap, np.int32)
        sh = np.empty((cap, 3), np.int8)
        e = fn(C.byref(s.c), _dp(q), C.c_double(rc), C.c_int64(cap), start.ctypes.data_as(C.POINTER(C.c_int64)),
               _ip(idx), sh.ctypes.data_as(C.POINTER(C.c_int8)))
        if e <= cap:
            return start, idx[:e].copy(), sh[:e].copy()
        cap = int(e)


def energy_forces(w, pot, q, want_forces=True):
    s, P = System(w), Pot(pot)
    q = np.ascontiguousarray(q, np.float64)
    F = np.zeros((s.n, 3)) if want_forces else None
    E = lib().orc_energy_forces(C.byref(s.c), C.byref(P.c), _dp(q), _dp(F) if want_forces else None)
    return float(E), F


def mlip_energy_forces(w, mlip, q, want_forces=True):
    from types import SimpleNamespace
    s = System(w)
    P = Pot(SimpleNamespace(pair=np.zeros((w.n_species, w.n_species, 8)), use_bonded=False, mlip=mlip))
    q = np.ascontiguousarray(q, np.float64)
    F = np.zeros((s.n, 3)) if want_forces else None
    E = lib().orc_mlip_energy_forces(C.byref(s.c), C.byref(P.c.mlip), _dp(q), _dp(F) if want_forces else None)
    return float(E), F


def aboba_step(w, pot, step, q, p, par=None):
    """One ABOBA step (Eq. 2).  Returns new (q, p) and (q_half, F(q_half), xi)."""
    s, P = System(w), Pot(pot)
    par = par or params(w)
    q = np.array(q, np.float64, order="C", copy=True)
    p = np.array(p, np.float64, order="C", copy=True)
    qh, Fh, xi = np.empty_like(q), np.empty_like(q), np.empty_like(q)
    lib().orc_aboba_step(C.byref(s.c), C.byref(par), C.byref(P.c), C.c_uint64(step), _dp(q), _dp(p), _dp(qh), _dp(Fh), _dp(xi))
    return q, p, qh, Fh, xi


def transport_step(w, Ft, F, xi, u, p_prev, q_half, par=None):
    """Eq. 8 on one step.  Returns dict(reject, S1, S2, ell, q, p) (q, p only meaningful on reject)."""
    s = System(w)
    par = par or params(w)
    arrs = [np.ascontiguousarray(a, np.float64) for a in (Ft, F, xi, p_prev, q_half)]
    S1, S2, ell = C.c_double(), C.c_double(), C.c_double()
    qo, po = np.zeros((s.n, 3)), np.zeros((s.n, 3))
    rej = lib().orc_transport_step(C.byref(s.c), C.byref(par), _dp(arrs[0]), _dp(arrs[1]), _dp(arrs[2]), C.c_double(u),
                                   _dp(arrs[3]), _dp(arrs[4]), C.byref(S1), C.byref(S2), C.byref(ell), _dp(qo), _dp(po))
    return dict(reject=int(rej), S1=S1.value, S2=S2.value, ell=ell.value, q=qo, p=po)


def force_slack(Ft, F, eps_F):
    """App. H: F + clip(-eps_F; Ft - F; eps_F), arrays [N,3]."""
    a, b = np.ascontiguousarray(Ft, np.float64), np.ascontiguousarray(F, np.float64)
    out = np.empty_like(b)
    lib().orc_force_slack(C.c_int32(len(b)), _dp(a), _dp(b), C.c_double(eps_F), _dp(out))
    return out


def lsd_window(w, q, p, n0, K=None, draft=None, target=None, par=None, debug=True, dF=None):
    """One synchronous window (Alg. 1).  Returns dict with new base state, committed trajectory, debug rows.
    dF ([N,3]) switches speculative error correction on (Alg. 3): the cache used by this window; "dF" in the result is the
    cache after it."""
    s = System(w)
    D, T = Pot(draft or w.draft), Pot(target or w.target)
    par = par or params(w)
    K = int(K or w.K)
    q = np.array(q, np.float64, order="C", copy=True)
    p = np.array(p, np.float64, order="C", copy=True)
    n = s.n
    tq, tp = np.zeros((K, n, 3)), np.zeros((K, n, 3))
    qh, Ft, Fg = np.zeros((K, n, 3)), np.zeros((K, n, 3)), np.zeros((K, n, 3))
    S1, S2, ell, lnu = np.zeros(K), np.zeros(K), np.zeros(K), np.zeros(K)
    rej = np.zeros(K, np.int32)
    l = C.c_int32()
    if dF is not None:
        dF = np.array(dF, np.float64, order="C", copy=True)
        dbg = (_dp(qh), _dp(Ft), _dp(Fg), _dp(S1), _dp(S2), _dp(ell), _dp(lnu), _ip(rej)) if debug else (None,) * 8
        nc = lib().orc_lsd_window_ec(C.byref(s.c), C.byref(par), C.byref(D.c), C.byref(T.c), C.c_uint64(n0), C.c_int32(K), _dp(q), _dp(p),
                                     _dp(dF), C.byref(l), _dp(tq), _dp(tp), *dbg)
    elif debug:
        nc = lib().orc_lsd_window(C.byref(s.c), C.byref(par), C.byref(D.c), C.byref(T.c), C.c_uint64(n0), C.c_int32(K), _dp(q), _dp(p),
                                  C.byref(l), _dp(tq), _dp(tp), _dp(qh), _dp(Ft), _dp(Fg), _dp(S1), _dp(S2), _dp(ell), _dp(lnu), _ip(rej))
    else:
        nc = lib().orc_lsd_window(C.byref(s.c), C.byref(par), C.byref(D.c), C.byref(T.c), C.c_uint64(n0), C.c_int32(K), _dp(q), _dp(p),
                                  C.byref(l), _dp(tq), _dp(tp), None, None, None, None, None, None, None, None)
    return dict(q=q, p=p, n_commit=int(nc), first_reject=int(l.value), traj_q=tq[:nc], traj_p=tp[:nc],
                q_half=qh, Ft=Ft, F=Fg, S1=S1, S2=S2, ell=ell, lnu=lnu, reject=rej, dF=dF)


def obabo_momentum(w, step, p_prev, p_new, F, par=None):
    """(OBABO) output momentum of committed step `step` (App. F Eq. 26-30); arrays [N,3]."""
    s = System(w)
    par = par or params(w)
    out = np.zeros((s.n, 3))
    a, b, c = (np.ascontiguousarray(x, np.float64) for x in (p_prev, p_new, F))
    lib().orc_obabo_momentum(C.byref(s.c), C.byref(par), C.c_uint64(step), _dp(a), _dp(b), _dp(c), _dp(out))
    return out


def run_lsd(w, q, p, n_steps, K=None, draft=None, target=None, par=None, keep_traj=True, ec=False):
    s = System(w)
    D, T = Pot(draft or w.draft), Pot(target or w.target)
    par = par or params(w)
    K = int(K or w.K)
    q = np.array(q, np.float64, order="C", copy=True)
    p = np.array(p, np.float64, order="C", copy=True)
    tq = np.zeros((n_steps, s.n, 3)) if keep_traj else None
    tp = np.zeros((n_steps, s.n, 3)) if keep_traj else None
    stats = np.zeros(4)
    dF = np.zeros((s.n, 3)) if ec else None
    if ec:
        lib().orc_run_lsd_ec(C.byref(s.c), C.byref(par), C.byref(D.c), C.byref(T.c), C.c_int64(n_steps), C.c_int32(K), _dp(q), _dp(p),
                             _dp(dF), _dp(tq) if keep_traj else None, _dp(tp) if keep_traj else None, _dp(stats))
    else:
        lib().orc_run_lsd(C.byref(s.c), C.byref(par), C.byref(D.c), C.byref(T.c), C.c_int64(n_steps), C.c_int32(K), _dp(q), _dp(p),
                          _dp(tq) if keep_traj else None, _dp(tp) if keep_traj else None, _dp(stats))
    return dict(q=q, p=p, traj_q=tq, traj_p=tp, windows=int(stats[0]), rejections=int(stats[1]),
                beta_sum=float(stats[2]), examined=int(stats[3]), dF=dF)


def run_aboba(w, pot, q, p, n_steps, par=None, keep_traj=True):
    s, P = System(w), Pot(pot)
    par = par or params(w)
    q = np.array(q, np.float64, order="C", copy=True)
    p = np.array(p, np.float64, order="C", copy=True)
    tq = np.zeros((n_steps, s.n, 3)) if keep_traj else None
    tp = np.zeros((n_steps, s.n, 3)) if keep_traj else None
    lib().orc_run_aboba(C.byref(s.c), C.byref(par), C.byref(P.c), C.c_int64(n_steps), _dp(q), _dp(p),
                        _dp(tq) if keep_traj else None, _dp(tp) if keep_traj else None)
    return dict(q=q, p=p, traj_q=tq, traj_p=tp)
