"""Pins for the oracle's priors, neighbour lists and MLIP."""
import numpy as np
import pytest

import lsd_inputs as L
from lsd_inputs.workloads import PAIR_COLS
from helpers import custom, fd_forces, edge_set


# ------------------------------------------------------------------ priors: closed forms
def test_lj_minimum_and_shift(orc):
    eps, sig, rc = 0.0104, 3.4, 7.0
    pair = np.zeros((1, 1, PAIR_COLS)); pair[0, 0, :3] = eps, sig, rc
    rmin = 2 ** (1 / 6) * sig
    w = custom([[0, 0, 0], [rmin, 0, 0]], pair=pair)
    E, F = orc.energy_forces(w, w.target, w.q0)
    u_rc = 4 * eps * ((sig / rc) ** 12 - (sig / rc) ** 6)
    assert abs(E - (-eps - u_rc)) < 1e-15
    assert np.abs(F).max() < 1e-15
    # repulsive inside the minimum, attractive outside, textbook -dU/dr value at r = sigma: 24 eps / sigma
    w = custom([[0, 0, 0], [sig, 0, 0]], pair=pair)
    _, F = orc.energy_forces(w, w.target, w.q0)
    assert F[0, 0] == pytest.approx(-24 * eps / sig, rel=1e-13) and F[1, 0] == pytest.approx(24 * eps / sig, rel=1e-13)
    # beyond the cutoff: nothing
    w = custom([[0, 0, 0], [rc + 1e-9, 0, 0]], pair=pair)
    E, F = orc.energy_forces(w, w.target, w.q0)
    assert E == 0.0 and np.abs(F).max() == 0.0


def test_morse_minimum(orc):
    D, a, r0, rc = 0.34, 1.36, 2.87, 6.0
    pair = np.zeros((1, 1, PAIR_COLS)); pair[0, 0, 3:7] = D, a, r0, rc
    w = custom([[0, 0, 0], [0, r0, 0]], pair=pair)
    E, F = orc.energy_forces(w, w.target, w.q0)
    x = np.exp(-a * (rc - r0))
    assert abs(E - (-D - D * ((1 - x) ** 2 - 1))) < 1e-15 and np.abs(F).max() < 1e-15
    # stiffness at the minimum: U'' = 2 D a^2  => F ~ -2 D a^2 dr
    dr = 1e-6
    w = custom([[0, 0, 0], [0, r0 + dr, 0]], pair=pair)
    _, F = orc.energy_forces(w, w.target, w.q0)
    assert F[1, 1] == pytest.approx(-2 * D * a * a * dr, rel=1e-5)


def test_bond_and_angle_closed_forms(orc):
    w = custom([[0, 0, 0], [1.5, 0, 0]], bonds=[[0, 1]], bond_k=20.0, bond_r0=1.4)
    E, F = orc.energy_forces(w, w.target, w.q0)
    assert E == pytest.approx(0.5 * 20 * 0.01) and F[0, 0] == pytest.approx(2.0) and F[1, 0] == pytest.approx(-2.0)
    # right angle, theta0 = 110 deg: U = k/2 (90-110 deg)^2; forces perpendicular to the arms, magnitude k dtheta / |arm|
    th0 = np.radians(110.0)
    w = custom([[2.0, 0, 0], [0, 0, 0], [0, 1.0, 0]], angles=[[0, 1, 2]], angle_k=2.0, angle_t0=th0)
    E, F = orc.energy_forces(w, w.target, w.q0)
    dth = np.pi / 2 - th0
    assert E == pytest.approx(0.5 * 2.0 * dth**2)
    # theta < theta0 => ends pushed apart (opening the angle): atom a moves -y, atom c moves -x
    assert F[0] == pytest.approx([0, 2.0 * dth / 2.0, 0], abs=1e-14)
    assert F[2] == pytest.approx([2.0 * dth / 1.0, 0, 0], abs=1e-14)
    assert np.abs(F.sum(0)).max() < 1e-14


@pytest.mark.parametrize("name,kw", [("cfg1", {}), ("cfg2", {}), ("cfg3", {"n_grid": 4}), ("cfg4", {"n_atoms": 256}),
                                     ("cfg5", {"cells": (3, 3, 3)})])
def test_forces_equal_finite_differences(orc, name, kw):
    """north_star pin: forces equal finite-difference gradients of the energy (full target potential)."""
    w = L.make_workload(name, **kw)
    rng = np.random.default_rng(0)
    q = w.q0 + rng.normal(0, 0.03, w.q0.shape)
    E, F = orc.energy_forces(w, w.target, q)
    idx = [(int(i), int(c)) for i, c in zip(rng.integers(0, w.n_atoms, 6), rng.integers(0, 3, 6))]
    fd = fd_forces(lambda x: orc.energy_forces(w, w.target, x, want_forces=False)[0], q, h=1e-4, idx=idx)
    scale = np.abs(F).max()
    for (i, c), v in fd.items():
        assert abs(F[i, c] - v) <= 2e-7 * scale + 1e-9, (i, c, F[i, c], v)
    assert np.abs(F.sum(0)).max() < 1e-9 * max(1.0, scale) * w.n_atoms ** 0.5
    if not w.periodic:                      # net torque vanishes in vacuum
        assert np.abs(np.cross(q, F).sum(0)).max() < 1e-10 * scale * w.n_atoms


def test_mlip_forces_fd_isolated_and_draft(orc):
    w = L.make_workload("cfg2")
    rng = np.random.default_rng(1)
    q = w.q0 + rng.normal(0, 0.05, w.q0.shape)
    for pot in (w.target, w.draft):
        E, F = orc.mlip_energy_forces(w, pot.mlip, q)
        idx = [(i, c) for i in (0, 7, 21) for c in range(3)]
        fd = fd_forces(lambda x: orc.mlip_energy_forces(w, pot.mlip, x, want_forces=False)[0], q, h=1e-4, idx=idx)
        for k, v in fd.items():
            assert abs(F[k] - v) <= 1e-7 * np.abs(F).max()


# ------------------------------------------------------------------ MLIP invariances
def _rot(rng):
    A = rng.standard_normal((3, 3)); Q, _ = np.linalg.qr(A)
    return Q * np.sign(np.linalg.det(Q))


def test_mlip_invariances_vacuum(orc):
    w = L.make_workload("cfg2")
    rng = np.random.default_rng(2)
    E0, F0 = orc.mlip_energy_forces(w, w.target.mlip, w.q0)
    Rm = _rot(rng)
    E1, F1 = orc.mlip_energy_forces(w, w.target.mlip, w.q0 @ Rm.T + np.array([3.0, -2.0, 7.0]))
    assert E1 == pytest.approx(E0, rel=1e-12)
    assert np.allclose(F1, F0 @ Rm.T, atol=1e-11 * np.abs(F0).max() + 1e-13)
    # permutation
    perm = rng.permutation(w.n_atoms)
    import dataclasses
    wp = dataclasses.replace(w, species=w.species[perm], mass_amu=w.mass_amu[perm], q0=w.q0[perm])
    E2, F2 = orc.mlip_energy_forces(wp, w.target.mlip, wp.q0)
    assert E2 == pytest.approx(E0, rel=1e-12) and np.allclose(F2, F0[perm], atol=1e-12)
    # extensivity: two copies further apart than T * r_c => 2 E
    import dataclasses as dc
    far = np.array([0.0, 0.0, 200.0])
    w2 = dc.replace(w, n_atoms=2 * w.n_atoms, species=np.tile(w.species, 2), mass_amu=np.tile(w.mass_amu, 2),
                    q0=np.concatenate([w.q0, w.q0 + far]))
    E3, F3 = orc.mlip_energy_forces(w2, w.target.mlip, w2.q0)
    assert E3 == pytest.approx(2 * E0, rel=1e-12) and np.allclose(F3[: w.n_atoms], F0, atol=1e-13)


def test_mlip_periodic_image_shift_invariance(orc):
    w = L.make_workload("cfg5", cells=(3, 3, 3))
    E0, F0 = orc.mlip_energy_forces(w, w.target.mlip, w.q0)
    q = w.q0.copy()
    q[5] += w.box * np.array([1, -2, 0]); q[40] -= w.box * np.array([0, 0, 3])
    E1, F1 = orc.mlip_energy_forces(w, w.target.mlip, q)
    assert E1 == pytest.approx(E0, rel=1e-11) and np.allclose(F1, F0, atol=1e-9 * np.abs(F0).max())


def test_perfect_fcc_has_zero_force(orc):
    """Special case: every site of a perfect single-species fcc crystal is an inversion centre => F = 0."""
    w = L.make_workload("cfg5", cells=(4, 4, 4), noise=0.0)
    E, F = orc.energy_forces(w, w.target, w.q0)
    Fm = orc.mlip_energy_forces(w, w.target.mlip, w.q0)[1]
    assert np.abs(F).max() < 1e-10 and np.abs(Fm).max() < 1e-10
    # and the noisy crystal does feel forces (the pin is not vacuous)
    wn = L.make_workload("cfg5", cells=(4, 4, 4))
    assert np.abs(orc.mlip_energy_forces(wn, wn.target.mlip, wn.q0)[1]).max() > 1e-4


def test_periodic_replica_forces_tile(orc):
    """Forces of a periodically replicated system equal the tiled forces of the small one (property used at full size)."""
    w = L.make_workload("cfg5", cells=(4, 4, 4))
    F0 = orc.energy_forces(w, w.target, w.q0)[1]
    w2 = L.tile_periodic(w, (2, 1, 1))
    F2 = orc.energy_forces(w2, w2.target, w2.q0)[1]
    assert np.allclose(F2, np.tile(F0, (2, 1)), atol=1e-10 * np.abs(F0).max())


# ------------------------------------------------------------------ neighbour lists
def test_shell_counts_sc_and_fcc(orc):
    w = L.make_workload("cfg1")                                     # jittered sc lattice: 6 + 12 + 8 = 26 inside 7.0 A
    start, idx, sh = orc.neighbors(w, w.q0, 7.0)
    assert (np.diff(start) == 26).all()
    w = L.make_workload("cfg5", cells=(4, 4, 4), noise=0.0)         # fcc: 12 + 6 + 24 + 12 + 24 = 78 inside 6.0 A
    start, idx, sh = orc.neighbors(w, w.q0, 6.0)
    assert (np.diff(start) == 78).all()
    start, idx, sh = orc.neighbors(w, w.q0, 3.0)                    # first shell only: a / sqrt 2 = 2.556 A
    assert (np.diff(start) == 12).all()


@pytest.mark.parametrize("name,kw,rc", [("cfg1", {}, 7.0), ("cfg3", {"n_grid": 6}, 5.0), ("cfg4", {"n_atoms": 1000}, 6.0),
                                        ("cfg5", {"cells": (5, 5, 4)}, 6.0), ("cfg2", {}, 5.0)])
def test_cell_list_equals_brute_force_and_is_symmetric(orc, name, kw, rc):
    w = L.make_workload(name, **kw)
    rng = np.random.default_rng(3)
    q = w.q0 + rng.normal(0, 0.05, w.q0.shape)
    if w.periodic:                                                  # unwrapped positions: move some atoms by box vectors
        q[::7] += w.box * rng.integers(-2, 3, (len(q[::7]), 3))
    a = orc.neighbors(w, q, rc, "brute")
    b = orc.neighbors(w, q, rc, "cell")
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    es = edge_set(*a)
    assert all((j, i, (-s[0], -s[1], -s[2])) in es for (i, j, s) in es)
    # brute-force check of membership with numpy (independent of the C loop)
    i = 3
    d = q - q[i]
    if w.periodic:
        d -= w.box * np.rint(d / w.box)
    r = np.linalg.norm(d, axis=1)
    want = set(np.nonzero((r < rc) & (np.arange(w.n_atoms) != i))[0].tolist())
    assert want == set(a[1][a[0][i]:a[0][i + 1]].tolist())
    assert (np.diff(a[1][a[0][i]:a[0][i + 1]]) > 0).all()           # sorted by j


def test_angle_term_near_and_at_collinear_arms(orc):
    """The angle force has the form 0/0 for collinear arms (theta = pi: numerator v - cos(theta) u and sin(theta) both vanish).
    Reading R19: sin(theta) is bounded below by 1e-12, so the force stays finite there; next to the singular
    point the analytic force still equals the finite-difference gradient."""
    th0 = np.radians(110.0)
    for eps in (1e-3, 1e-5):
        q = np.array([[1.3, 0.0, 0.0], [0.0, 0.0, 0.0], [-1.1 * np.cos(eps), 1.1 * np.sin(eps), 0.0]])
        w = custom(q, angles=[[0, 1, 2]], angle_k=2.0, angle_t0=th0)
        E, F = orc.energy_forces(w, w.target, w.q0)
        assert E == pytest.approx(0.5 * 2.0 * (np.pi - eps - th0) ** 2, rel=1e-9)
        fd = fd_forces(lambda x: orc.energy_forces(w, w.target, x, want_forces=False)[0], q, h=1e-7, idx=[(0, 1), (2, 1), (1, 1)])
        for (i, c), v in fd.items():
            assert F[i, c] == pytest.approx(v, rel=1e-4, abs=1e-6)
        # |F_a| = dU/dtheta / |arm|, perpendicular to the arm
        # (sin(theta) = sqrt(1 - cos^2) loses digits next to pi: relative error ~ 1e-16 / eps^2)
        assert np.linalg.norm(F[0]) == pytest.approx(2.0 * (np.pi - eps - th0) / 1.3, rel=1e-5)
    w = custom([[1.3, 0.0, 0.0], [0.0, 0.0, 0.0], [-1.1, 0.0, 0.0]], angles=[[0, 1, 2]], angle_k=2.0, angle_t0=th0)
    E, F = orc.energy_forces(w, w.target, w.q0)
    assert np.isfinite(F).all() and E == pytest.approx(0.5 * 2.0 * (np.pi - th0) ** 2, rel=1e-12)
