"""Small hand-built systems for pins (data only; uses lsd_inputs dataclasses)."""
import numpy as np

import lsd_inputs as L
from lsd_inputs.workloads import Potential, Workload, PAIR_COLS


def custom(q, species=None, mass=None, box=None, pair=None, n_species=1, bonds=None, angles=None,
           bond_k=20.0, bond_r0=1.4, angle_k=2.0, angle_t0=np.radians(110.0), mlip=None, draft=None,
           T=300.0, gamma=0.01, dt=0.5, K=4, seed=11, use_bonded=None):
    q = np.asarray(q, float)
    n = len(q)
    species = np.zeros(n, np.int32) if species is None else np.asarray(species, np.int32)
    mass = np.full(n, 39.948) if mass is None else np.asarray(mass, float)
    pair = np.zeros((n_species, n_species, PAIR_COLS)) if pair is None else pair
    bonds = np.zeros((0, 2), np.int32) if bonds is None else np.asarray(bonds, np.int32)
    angles = np.zeros((0, 3), np.int32) if angles is None else np.asarray(angles, np.int32)
    ub = bool(len(bonds) or len(angles)) if use_bonded is None else use_bonded
    tgt = Potential(pair, ub, mlip)
    drf = draft if draft is not None else tgt
    return Workload("custom", n, n_species, species, mass, np.zeros(3) if box is None else np.asarray(box, float),
                    box is not None, q, bonds, np.full(len(bonds), bond_k), np.full(len(bonds), bond_r0),
                    angles, np.full(len(angles), angle_k), np.full(len(angles), angle_t0),
                    drf, tgt, T, gamma, dt, K, seed, 100, "fp64")


def tether_pair(k, n_species=1):
    p = np.zeros((n_species, n_species, PAIR_COLS))
    for s in range(n_species):
        p[s, s, 7] = k
    return p


def fd_forces(energy_fn, q, h=1e-4, idx=None):
    """Central finite differences of an energy function: -dE/dq for the listed (atom, comp)."""
    q = np.array(q, float)
    out = {}
    for (i, c) in idx:
        qp, qm = q.copy(), q.copy()
        qp[i, c] += h
        qm[i, c] -= h
        out[(i, c)] = -(energy_fn(qp) - energy_fn(qm)) / (2 * h)
    return out


def edge_set(start, idx, shifts):
    n = len(start) - 1
    i = np.repeat(np.arange(n), np.diff(start))
    return set(zip(i.tolist(), idx.tolist(), map(tuple, shifts.tolist())))
