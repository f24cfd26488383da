"""The five BASELINE.json workloads, completed as in SURVEY.md section 8(c) / DESIGN.md.

Everything here is *data*: positions, species, masses, topology, pair-parameter
tables, MLIP weight vectors and integrator settings.  Units: Angstrom, fs, eV, K,
masses in amu.  No force, energy, integrator or RNG-of-the-method code lives here;
the only random numbers drawn are numpy PCG64 draws for the synthetic inputs.

Stand-in statement: the paper measures on FCC copper, bulk water and
alanine peptides with pretrained UMA/Orb models;
those structures and weights are not available, so seeded synthetic systems of
the same shapes and random-weight SchNet-style networks stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

K_B = 8.617333262e-5      # eV / K
AMU = 103.642696          # eV fs^2 / A^2 per amu

# pair-table columns (per ordered species pair)
PAIR_COLS = 8
LJ_EPS, LJ_SIGMA, LJ_RC, MORSE_D, MORSE_A, MORSE_R0, MORSE_RC = range(7)


@dataclass
class Mlip:
    """SchNet-style network M1-M8; weights flat fp64, layout below."""
    width: int            # F
    n_blocks: int         # T
    n_rbf: int            # R
    cutoff: float         # r_c (A)
    alpha: float          # energy scale (M8)
    n_species: int
    weights: np.ndarray   # flat float64, see mlip_weight_offsets
    seed: int = 0


@dataclass
class Potential:
    pair: np.ndarray                  # [ns, ns, PAIR_COLS] float64, zeros = term off
    use_bonded: bool
    mlip: Optional[Mlip] = None

    def pair_cutoff(self) -> float:
        return float(max(self.pair[..., LJ_RC].max(), self.pair[..., MORSE_RC].max()))


@dataclass
class Workload:
    name: str
    n_atoms: int
    n_species: int
    species: np.ndarray               # int32 [N]
    mass_amu: np.ndarray              # float64 [N]
    box: np.ndarray                   # float64 [3] (ignored if not periodic)
    periodic: bool
    q0: np.ndarray                    # float64 [N, 3]
    bonds: np.ndarray                 # int32 [nb, 2]
    bond_k: np.ndarray                # float64 [nb]
    bond_r0: np.ndarray               # float64 [nb]
    angles: np.ndarray                # int32 [na, 3]  (end, apex, end)
    angle_k: np.ndarray               # float64 [na]
    angle_theta0: np.ndarray          # float64 [na] (rad)
    draft: Potential
    target: Potential
    temperature_K: float
    friction_per_fs: float
    dt_fs: float
    K: int
    seed: int
    n_steps: int
    precision: str                    # 'fp64' | 'fp32' | 'bf16'
    skin: float = 0.5
    notes: dict = field(default_factory=dict)


# --------------------------------------------------------------------------- MLIP weights
def mlip_weight_offsets(F: int, T: int, R: int, ns: int) -> dict:
    """Offsets (in elements) into the flat weight vector.

    emb[ns][F]; per block t: W_in[F][F], W_f1[F][R], W_f2[F][F], W_o1[F][F], W_o2[F][F]
    (all row-major [out][in]); readout W_r1[F/2][F], w_r2[F/2].
    """
    off = {"emb": 0}
    o = ns * F
    per_block = 4 * F * F + F * R
    off["block0"] = o
    off["per_block"] = per_block
    off["W_in"] = 0
    off["W_f1"] = F * F
    off["W_f2"] = F * F + F * R
    off["W_o1"] = 2 * F * F + F * R
    off["W_o2"] = 3 * F * F + F * R
    o += T * per_block
    off["W_r1"] = o
    o += (F // 2) * F
    off["w_r2"] = o
    o += F // 2
    off["total"] = o
    return off


def mlip_weight_count(F: int, T: int, R: int, ns: int) -> int:
    return mlip_weight_offsets(F, T, R, ns)["total"]


def make_mlip(F: int, T: int, R: int, cutoff: float, ns: int, seed: int, alpha: float) -> Mlip:
    """Weights N(0, 1/fan_in), embeddings N(0, 1), no biases (M4, M7)."""
    rng = np.random.default_rng(seed)
    off = mlip_weight_offsets(F, T, R, ns)
    w = np.empty(off["total"], dtype=np.float64)
    w[: ns * F] = rng.standard_normal(ns * F)
    for t in range(T):
        b = off["block0"] + t * off["per_block"]
        for name, rows, cols in (("W_in", F, F), ("W_f1", F, R), ("W_f2", F, F),
                                 ("W_o1", F, F), ("W_o2", F, F)):
            n = rows * cols
            w[b + off[name]: b + off[name] + n] = rng.standard_normal(n) / math.sqrt(cols)
    n = (F // 2) * F
    w[off["W_r1"]: off["W_r1"] + n] = rng.standard_normal(n) / math.sqrt(F)
    w[off["w_r2"]: off["w_r2"] + F // 2] = rng.standard_normal(F // 2) / math.sqrt(F // 2)
    return Mlip(width=F, n_blocks=T, n_rbf=R, cutoff=cutoff, alpha=alpha, n_species=ns,
                weights=w, seed=seed)


# Energy scales alpha (M8): "NN force RMS ~ 10 % of the prior's" on a thermalised
# reference configuration.  Written by oracle/calibrate_alpha.py (calls only oracle/);
# stored here as plain data so that the product path never needs the oracle.
ALPHA = {
    ("cfg2", "target"): 1.849763e-01,
    ("cfg2", "draft"): 1.924046e-01,
    ("cfg3", "target"): 1.553548e-01,
    ("cfg4", "target"): 3.928412e-02,
    ("cfg4", "draft"): 6.446018e-02,
    ("cfg5", "target"): 1.926644e-02,
    ("cfg5", "draft"): 4.538489e-01,
}


def _empty_topology():
    z = np.zeros
    return (z((0, 2), np.int32), z(0), z(0), z((0, 3), np.int32), z(0), z(0))


def _pair_table(ns: int) -> np.ndarray:
    return np.zeros((ns, ns, PAIR_COLS), dtype=np.float64)


# --------------------------------------------------------------------------- cfg 1
def _cfg1() -> Workload:
    rng = np.random.default_rng(0)
    g = np.arange(4) * 3.8
    q = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    q = q + rng.uniform(-0.1, 0.1, size=q.shape)
    n = len(q)
    lj = _pair_table(1)
    lj[0, 0, LJ_EPS], lj[0, 0, LJ_SIGMA], lj[0, 0, LJ_RC] = 0.0104, 3.4, 7.0
    tgt = lj.copy()
    tgt[0, 0, MORSE_D], tgt[0, 0, MORSE_A], tgt[0, 0, MORSE_R0], tgt[0, 0, MORSE_RC] = 0.002, 1.5, 3.8, 7.0
    b, bk, br, a, ak, at = _empty_topology()
    return Workload("cfg1", n, 1, np.zeros(n, np.int32), np.full(n, 39.948), np.full(3, 15.2), True, q,
                    b, bk, br, a, ak, at, Potential(lj, False), Potential(tgt, False),
                    120.0, 0.01, 2.0, 4, 0, 2000, "fp64", skin=0.5)


# --------------------------------------------------------------------------- cfg 2
_HCNO_MASS = np.array([1.008, 12.011, 14.007, 15.999])


def _chain_topology(n):
    bonds = np.stack([np.arange(n - 1), np.arange(1, n)], 1).astype(np.int32)
    angles = np.stack([np.arange(n - 2), np.arange(1, n - 1), np.arange(2, n)], 1).astype(np.int32)
    return bonds, angles


def _cfg2(n_chain: int = 22) -> Workload:
    rng = np.random.default_rng(100)          # geometry jitter stream (config seeds 1, 2 are the nets')
    r0, th0 = 1.4, math.radians(110.0)
    half = 0.5 * (math.pi - th0)
    q = np.zeros((n_chain, 3))
    for i in range(1, n_chain):
        sgn = 1.0 if i % 2 else -1.0
        q[i] = q[i - 1] + r0 * np.array([math.cos(half), sgn * math.sin(half), 0.0])
    q += rng.normal(0.0, 0.02, size=q.shape)
    species = (np.arange(n_chain) % 4).astype(np.int32)
    bonds, angles = _chain_topology(n_chain)
    prior = _pair_table(4)
    tgt = Potential(prior, True, make_mlip(64, 3, 32, 5.0, 4, 1, ALPHA[("cfg2", "target")]))
    drf = Potential(prior, True, make_mlip(32, 1, 32, 5.0, 4, 2, ALPHA[("cfg2", "draft")]))
    return Workload("cfg2", n_chain, 4, species, _HCNO_MASS[species], np.zeros(3), False, q,
                    bonds, np.full(len(bonds), 20.0), np.full(len(bonds), r0),
                    angles, np.full(len(angles), 2.0), np.full(len(angles), th0),
                    drf, tgt, 300.0, 0.01, 0.5, 16, 1, 10000, "fp32", skin=2.0)


# --------------------------------------------------------------------------- cfg 3
def _random_rotations(rng, n):
    """Uniform random rotation matrices from normalised Gaussian quaternions."""
    qn = rng.standard_normal((n, 4))
    qn /= np.linalg.norm(qn, axis=1, keepdims=True)
    w, x, y, z = qn.T
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def _cfg3(n_grid: int = 8) -> Workload:
    rng = np.random.default_rng(3)
    spacing = 3.1
    L = n_grid * spacing
    g = (np.arange(n_grid) + 0.5) * spacing
    o = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    nm = len(o)
    roh, th = 0.96, math.radians(104.5)
    h1 = roh * np.array([math.sin(th / 2), 0.0, math.cos(th / 2)])
    h2 = roh * np.array([-math.sin(th / 2), 0.0, math.cos(th / 2)])
    R = _random_rotations(rng, nm)
    q = np.empty((nm, 3, 3))
    q[:, 0] = o
    q[:, 1] = o + R @ h1
    q[:, 2] = o + R @ h2
    q = q.reshape(-1, 3)
    species = np.tile(np.array([0, 1, 1], np.int32), nm)
    mass = np.where(species == 0, 15.999, 1.008)
    oi = 3 * np.arange(nm)
    bonds = np.concatenate([np.stack([oi, oi + 1], 1), np.stack([oi, oi + 2], 1)]).astype(np.int32)
    angles = np.stack([oi + 1, oi, oi + 2], 1).astype(np.int32)
    prior = _pair_table(2)
    prior[0, 0, LJ_EPS], prior[0, 0, LJ_SIGMA], prior[0, 0, LJ_RC] = 0.0067, 3.17, 9.0
    tgt = Potential(prior, True, make_mlip(64, 3, 32, 5.0, 2, 4, ALPHA[("cfg3", "target")]))
    drf = Potential(prior, True, None)
    name = "cfg3" if n_grid == 8 else f"cfg3_g{n_grid}"
    return Workload(name, 3 * nm, 2, species, mass, np.full(3, L), True, q,
                    bonds, np.full(len(bonds), 20.0), np.full(len(bonds), roh),
                    angles, np.full(len(angles), 2.0), np.full(len(angles), th),
                    drf, tgt, 300.0, 0.01, 0.5, 16, 3, 1000, "fp32", skin=1.2)


# --------------------------------------------------------------------------- cfg 4
def _push_apart(q, L, dmin_of_pair, species, iters, rng):
    """Geometric overlap removal ("relaxed 200 steps"): every pair closer than its
    contact distance is moved apart symmetrically by half the overlap.  Pure geometry,
    no force field (stands in for the unspecified relaxation)."""
    from scipy.spatial import cKDTree
    dmax = float(dmin_of_pair.max())
    for _ in range(iters):
        qw = np.mod(q, L)
        tree = cKDTree(qw, boxsize=L)
        pairs = tree.query_pairs(dmax, output_type="ndarray")
        if len(pairs) == 0:
            break
        i, j = pairs[:, 0], pairs[:, 1]
        d = qw[j] - qw[i]
        d -= L * np.rint(d / L)
        r = np.linalg.norm(d, axis=1)
        want = dmin_of_pair[species[i], species[j]]
        m = r < want
        if not m.any():
            break
        i, j, d, r, want = i[m], j[m], d[m], r[m], want[m]
        r = np.maximum(r, 1e-6)
        shift = (0.5 * (want - r) / r)[:, None] * d
        np.add.at(q, j, shift)
        np.add.at(q, i, -shift)
    return q


def _cfg4(n_atoms: int = 4096) -> Workload:
    rng = np.random.default_rng(5)
    sig, eps = 3.4, 0.0104
    L = (n_atoms / 1.2) ** (1.0 / 3.0) * sig
    nB = int(round(0.2 * n_atoms))
    species = np.zeros(n_atoms, np.int32)
    species[rng.permutation(n_atoms)[:nB]] = 1
    sig_ab = np.array([[1.0, 0.8], [0.8, 0.88]]) * sig
    eps_ab = np.array([[1.0, 1.5], [1.5, 0.5]]) * eps
    q = rng.uniform(0.0, L, size=(n_atoms, 3))
    q = _push_apart(q, L, 0.95 * sig_ab, species, 200, rng)
    prior = _pair_table(2)
    prior[..., LJ_EPS], prior[..., LJ_SIGMA], prior[..., LJ_RC] = eps_ab, sig_ab, 2.5 * sig_ab
    tgt = Potential(prior, False, make_mlip(128, 4, 32, 6.0, 2, 6, ALPHA[("cfg4", "target")]))
    drf = Potential(prior, False, make_mlip(32, 1, 32, 6.0, 2, 61, ALPHA[("cfg4", "draft")]))
    name = "cfg4" if n_atoms == 4096 else f"cfg4_n{n_atoms}"
    return Workload(name, n_atoms, 2, species, np.full(n_atoms, 39.948), np.full(3, L), True, q,
                    *_empty_topology(), drf, tgt, 0.8 * eps / K_B, 0.01, 1.0, 32, 5, 1000, "fp32", skin=0.5)


# --------------------------------------------------------------------------- cfg 5
def _cfg5(cells=(32, 32, 16), noise: float = 0.05) -> Workload:
    rng = np.random.default_rng(7)
    a = 3.615
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])
    nx, ny, nz = cells
    cell = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij"), -1).reshape(-1, 1, 3)
    q = ((cell + basis[None]) * a).reshape(-1, 3)
    if noise > 0:
        q = q + rng.normal(0.0, noise, size=q.shape)
    n = len(q)
    prior = _pair_table(1)
    prior[0, 0, MORSE_D], prior[0, 0, MORSE_A], prior[0, 0, MORSE_R0], prior[0, 0, MORSE_RC] = 0.34, 1.36, 2.87, 6.0
    tgt = Potential(prior, False, make_mlip(128, 6, 32, 6.0, 1, 8, ALPHA[("cfg5", "target")]))
    drf = Potential(prior, False, make_mlip(32, 1, 32, 6.0, 1, 81, ALPHA[("cfg5", "draft")]))
    name = "cfg5" if tuple(cells) == (32, 32, 16) and noise == 0.05 else f"cfg5_{nx}x{ny}x{nz}"
    return Workload(name, n, 1, np.zeros(n, np.int32), np.full(n, 63.546), np.array(cells, float) * a, True, q,
                    *_empty_topology(), drf, tgt, 600.0, 0.005, 2.0, 8, 7, 1000, "bf16", skin=0.5)


WORKLOADS = {"cfg1": _cfg1, "cfg2": _cfg2, "cfg3": _cfg3, "cfg4": _cfg4, "cfg5": _cfg5}


def make_workload(name: str, **kw) -> Workload:
    """name in cfg1..cfg5; kw are size overrides for scaled-down parity cases
    (cfg2: n_chain; cfg3: n_grid; cfg4: n_atoms; cfg5: cells, noise)."""
    return WORKLOADS[name](**kw)


def with_target_as_draft(w: Workload) -> Workload:
    """draft == target variant (acceptance must be exactly 1)."""
    return replace(w, draft=w.target)


def tile_periodic(w: Workload, reps) -> Workload:
    """Replicate a periodic workload reps=(rx,ry,rz) times (property tests: forces of the
    replicated system equal the tiled forces of the small one)."""
    assert w.periodic
    rx, ry, rz = reps
    offs = np.stack(np.meshgrid(np.arange(rx), np.arange(ry), np.arange(rz), indexing="ij"), -1).reshape(-1, 3)
    n = w.n_atoms
    q = np.concatenate([w.q0 + o * w.box for o in offs])
    m = len(offs)
    bonds = np.concatenate([w.bonds + k * n for k in range(m)]).astype(np.int32) if len(w.bonds) else w.bonds
    angles = np.concatenate([w.angles + k * n for k in range(m)]).astype(np.int32) if len(w.angles) else w.angles
    return replace(w, name=f"{w.name}_x{rx}{ry}{rz}", n_atoms=n * m, species=np.tile(w.species, m),
                   mass_amu=np.tile(w.mass_amu, m), box=w.box * np.array(reps, float), q0=q,
                   bonds=bonds, bond_k=np.tile(w.bond_k, m), bond_r0=np.tile(w.bond_r0, m),
                   angles=angles, angle_k=np.tile(w.angle_k, m), angle_theta0=np.tile(w.angle_theta0, m))


def to_soa(x: np.ndarray) -> np.ndarray:
    """[N,3] -> contiguous [3,N] (the boundary's component-major layout)."""
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64).T)


def from_soa(x: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(x).T)
