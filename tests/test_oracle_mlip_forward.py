"""Pins for the FORWARD definition of the oracle's SchNet-style network.

Finite differences pin the oracle's gradient against its own energy and the invariance tests hold for any smooth
pair-distance network, so neither fixes the definition itself.  Here the weights are set by hand so that the energy has a
closed form at special distances, and the expected numbers are written out from M1-M8 with math.log / math.exp only
(never by calling the oracle):

  * r = k Delta with Delta = r_c / (R - 1):  g_k = 1 exactly (M1: centre spacing);  r = (k + 1) Delta:  g_k = e^{-1/2}
    (M1: width 2 Delta^2 in the exponent);  r = r_c / 2:  f_c = 1/2 (M2);  r >= r_c: no edge;
  * ssp(0) = 0, ssp(ln 3) = ln 2, ssp(ln 2) = ln 1.5 (M3: the shift by ln 2);
  * non-symmetric permutation matrices with different scales for W_in, W_f2, W_o1, W_o2, so that taking one for another,
    or a matrix for its transpose, changes the number (M5 wiring), residual update x <- x + v (M5), readout with F/2 rows
    and the scale alpha (M6).

Each plausible mistake was introduced into oracle/lsd_oracle.c by hand once and made at least one test here fail
(list in the commit message that added this file).
"""
import math

import numpy as np
import pytest

from lsd_inputs.workloads import Mlip, mlip_weight_offsets
from helpers import custom

LN2 = math.log(2.0)


def ssp(x):
    """M3 written out: ln(1 + e^x) - ln 2."""
    return math.log(1.0 + math.exp(x)) - LN2


def shift_matrix(F, s, scale):
    """out[f] = scale * in[(f + s) % F]: a non-symmetric permutation (its transpose shifts the other way)."""
    W = np.zeros((F, F))
    for f in range(F):
        W[f, (f + s) % F] = scale
    return W


def build(F, T, R, rc, alpha, emb, blocks, Wr1, wr2):
    """Flat weight vector in the generator's documented order (lsd_inputs.mlip_weight_offsets)."""
    ns = emb.shape[0]
    off = mlip_weight_offsets(F, T, R, ns)
    w = np.zeros(off["total"])
    w[: ns * F] = emb.reshape(-1)
    for t, blk in enumerate(blocks):
        b = off["block0"] + t * off["per_block"]
        for name in ("W_in", "W_f1", "W_f2", "W_o1", "W_o2"):
            m = np.asarray(blk[name], float)
            w[b + off[name]: b + off[name] + m.size] = m.reshape(-1)
    w[off["W_r1"]: off["W_r1"] + Wr1.size] = Wr1.reshape(-1)
    w[off["w_r2"]: off["w_r2"] + wr2.size] = wr2
    w = np.concatenate([w, np.full(4 * F * F, 0.77)])     # anything read past the documented layout changes the result
    return Mlip(width=F, n_blocks=T, n_rbf=R, cutoff=rc, alpha=alpha, n_species=ns, weights=w)


# hand-set network: F = 6, R = 9 (Delta = r_c / 8, so that k = 4 sits at r_c / 2), one block.  The four square matrices
# are scaled cyclic shifts by 1, 2, 4, 5 channels: none is symmetric (mod 6 only the shift by 3 is) and all differ.
F, R, RC, ALPHA = 6, 9, 4.0, 0.37
DELTA = RC / (R - 1)
EMB = np.array([[2.0, -1.0, 0.5, 3.0, -0.4, 1.1], [1.0, 4.0, -2.0, 0.25, 0.6, -1.3]])     # two species
C_F = np.array([math.log(3.0), -0.7, 1.3, 0.0, 0.45, -1.9])               # W_f1[f][k*] = C_F[f], every other column zero
S_IN, S_F2, S_O1, S_O2 = 0.5, 2.0, 3.0, -1.5
H_IN, H_F2, H_O1, H_O2 = 1, 2, 4, 5
WR1 = np.array([[1.0, 0.0, -1.0, 0.5, 0.0, 0.3], [0.0, 2.0, 0.0, -0.25, 1.0, 0.0], [0.4, 0.0, 0.0, 0.0, -0.6, 0.9]])   # [F/2][F]
WR2 = np.array([0.8, -1.7, 0.55])


def block(kstar, zero_in=False):
    Wf1 = np.zeros((F, R))
    Wf1[:, kstar] = C_F
    return dict(W_in=shift_matrix(F, H_IN, 0.0 if zero_in else S_IN), W_f1=Wf1, W_f2=shift_matrix(F, H_F2, S_F2),
                W_o1=shift_matrix(F, H_O1, S_O1), W_o2=shift_matrix(F, H_O2, S_O2))


def expected_pair_energy(gk, fc, s0, s1):
    """E of two atoms (species s0, s1) that see each other through one RBF value gk and cutoff value fc, from M4-M6
    with the hand-set matrices above, channel by channel."""
    a = [ssp(C_F[f] * gk) for f in range(F)]                              # ssp(W_f1 g)
    w = [S_F2 * a[(f + H_F2) % F] * fc for f in range(F)]                     # (W_f2 a) f_c
    E = 0.0
    for si, sj in ((s0, s1), (s1, s0)):
        y = [S_IN * EMB[sj][(f + H_IN) % F] for f in range(F)]               # y_j = W_in x_j
        m = [y[f] * w[f] for f in range(F)]                               # one neighbour
        h = [S_O1 * m[(f + H_O1) % F] for f in range(F)]                     # W_o1 m
        sh = [ssp(v) for v in h]
        x = [EMB[si][f] + S_O2 * sh[(f + H_O2) % F] for f in range(F)]       # residual update
        z = [sum(WR1[k][f] * x[f] for f in range(F)) for k in range(F // 2)]
        E += sum(WR2[k] * ssp(z[k]) for k in range(F // 2))
    return ALPHA * E


def isolated_energy(species):
    E = 0.0
    for s in species:
        z = [sum(WR1[k][f] * EMB[s][f] for f in range(F)) for k in range(F // 2)]
        E += sum(WR2[k] * ssp(z[k]) for k in range(F // 2))
    return ALPHA * E


def two_atoms(r, net, species=(0, 1)):
    return custom([[0.0, 0.0, 0.0], [0.0, r, 0.0]], species=list(species), n_species=2, mlip=net)


def test_ssp_special_values_used_below():
    assert ssp(0.0) == 0.0
    assert ssp(math.log(3.0)) == pytest.approx(LN2, abs=1e-15) and ssp(LN2) == pytest.approx(math.log(1.5), abs=1e-15)


def test_zero_filter_gives_position_independent_readout_energy(orc):
    """W_f1 = 0 => ssp(0) = 0 => every filter vanishes => E = alpha sum_i w_r2 . ssp(W_r1 Emb[s_i]), F = 0.
    A missing -ln 2 in ssp, a readout with the wrong number of rows or a missing alpha changes E or makes F non-zero."""
    blk = block(4)
    blk["W_f1"] = np.zeros((F, R))
    net = build(F, 1, R, RC, ALPHA, EMB, [blk], WR1, WR2)
    rng = np.random.default_rng(5)
    q = rng.uniform(0, 3.0, (7, 3))
    sp = [0, 1, 1, 0, 1, 0, 0]
    w = custom(q, species=sp, n_species=2, mlip=net)
    E, Fo = orc.mlip_energy_forces(w, net, w.q0)
    assert E == pytest.approx(isolated_energy(sp), rel=1e-14)
    assert np.abs(Fo).max() == 0.0
    # one explicit number: species 0, z = (2 - 0.5 + 1.5 + 0.33, -2 - 0.75 - 0.4, 0.8 + 0.24 + 0.99) = (3.33, -3.15, 2.03)
    e0 = ALPHA * (0.8 * (math.log(1 + math.exp(3.33)) - LN2) - 1.7 * (math.log(1 + math.exp(-3.15)) - LN2)
                  + 0.55 * (math.log(1 + math.exp(2.03)) - LN2))
    assert isolated_energy([0]) == pytest.approx(e0, rel=1e-15)


@pytest.mark.parametrize("kstar", [4, 2, 6])
def test_pair_energy_on_an_rbf_centre(orc, kstar):
    """r = k* Delta: g_k* = 1 (fails for a centre spacing r_c / R or centres shifted by one); k* = 4 is r_c / 2 where
    f_c = 1/2 exactly; the other two use f_c = (cos(pi k*/8) + 1) / 2."""
    net = build(F, 1, R, RC, ALPHA, EMB, [block(kstar)], WR1, WR2)
    r = kstar * DELTA
    fc = 0.5 if kstar == 4 else 0.5 * (math.cos(math.pi * kstar / 8.0) + 1.0)
    w = two_atoms(r, net)
    E, _ = orc.mlip_energy_forces(w, net, w.q0)
    assert E == pytest.approx(expected_pair_energy(1.0, fc, 0, 1), rel=1e-13)
    assert abs(E - isolated_energy([0, 1])) > 1e-3          # the pair term is not negligible in this check


def test_pair_energy_one_spacing_off_centre(orc):
    """r = (k* + 1) Delta: g_k* = exp(-1/2) (a width Delta^2 instead of 2 Delta^2 would give exp(-1))."""
    kstar = 3
    net = build(F, 1, R, RC, ALPHA, EMB, [block(kstar)], WR1, WR2)
    r = (kstar + 1) * DELTA                                  # = r_c / 2 again: f_c = 1/2
    w = two_atoms(r, net, species=(1, 1))
    E, _ = orc.mlip_energy_forces(w, net, w.q0)
    assert E == pytest.approx(expected_pair_energy(math.exp(-0.5), 0.5, 1, 1), rel=1e-13)
    assert abs(E - expected_pair_energy(math.exp(-1.0), 0.5, 1, 1)) > 1e-4


def test_cutoff_limit_and_beyond(orc):
    """r -> r_c: E -> isolated atoms continuously (f_c -> 0 with zero slope); r >= r_c: exactly isolated, no force."""
    net = build(F, 1, R, RC, ALPHA, EMB, [block(8)], WR1, WR2)      # k* = 8 sits at r_c: g = 1 there, only f_c kills it
    iso = isolated_energy([0, 1])
    for eps, tol in ((1e-3, 1e-6), (1e-5, 1e-10)):
        w = two_atoms(RC - eps, net)
        E, _ = orc.mlip_energy_forces(w, net, w.q0)
        assert abs(E - iso) < tol and E != iso                   # f_c ~ (pi eps / 2 r_c)^2
    for r in (RC, RC + 0.5):
        w = two_atoms(r, net)
        E, Fo = orc.mlip_energy_forces(w, net, w.q0)
        assert E == pytest.approx(iso, rel=1e-15) and np.abs(Fo).max() == 0.0


def test_neighbour_sum_and_self_exclusion(orc):
    """m_i is a SUM over neighbours j != i: a centre atom with two identical neighbours at r_c / 2 (the outer two are
    r_c apart, so they do not see each other) gets twice the message."""
    net = build(F, 1, R, RC, ALPHA, EMB, [block(4)], WR1, WR2)
    r = RC / 2
    w = custom([[0.0, 0.0, 0.0], [r, 0.0, 0.0], [-r, 0.0, 0.0]], species=[0, 1, 1], n_species=2, mlip=net)
    E, _ = orc.mlip_energy_forces(w, net, w.q0)
    a = [ssp(C_F[f]) for f in range(F)]
    wf = [S_F2 * a[(f + H_F2) % F] * 0.5 for f in range(F)]

    def atom_energy(si, nbr_species):
        m = [0.0] * F
        for sj in nbr_species:
            for f in range(F):
                m[f] += S_IN * EMB[sj][(f + H_IN) % F] * wf[f]
        h = [S_O1 * m[(f + H_O1) % F] for f in range(F)]
        x = [EMB[si][f] + S_O2 * ssp(h[(f + H_O2) % F]) for f in range(F)]
        z = [sum(WR1[k][f] * x[f] for f in range(F)) for k in range(F // 2)]
        return sum(WR2[k] * ssp(z[k]) for k in range(F // 2))

    expect = ALPHA * (atom_energy(0, [1, 1]) + 2 * atom_energy(1, [0]))
    assert E == pytest.approx(expect, rel=1e-13)


def test_second_block_with_zero_input_matrix_adds_nothing(orc):
    """Block wiring: T = 2 with W_in of block 2 set to zero => y = 0 => m = 0 => ssp(0) = 0 => x unchanged, so the
    energy is that of the one-block network (closed form above) whatever the other matrices of block 2 are."""
    net2 = build(F, 2, R, RC, ALPHA, EMB, [block(4), block(2, zero_in=True)], WR1, WR2)
    w = two_atoms(RC / 2, net2)
    E2, _ = orc.mlip_energy_forces(w, net2, w.q0)
    assert E2 == pytest.approx(expected_pair_energy(1.0, 0.5, 0, 1), rel=1e-13)


def test_two_blocks_compose_in_order(orc):
    """T = 2, both blocks active on the same RBF: block 2 sees x after block 1 (y2 = W_in2 x1), written out by hand."""
    b1, b2 = block(4), block(4)
    b2["W_in"] = shift_matrix(F, 2, 0.25)
    net2 = build(F, 2, R, RC, ALPHA, EMB, [b1, b2], WR1, WR2)
    w = two_atoms(RC / 2, net2)
    E2, _ = orc.mlip_energy_forces(w, net2, w.q0)
    a = [ssp(C_F[f]) for f in range(F)]
    wf = [S_F2 * a[(f + H_F2) % F] * 0.5 for f in range(F)]                   # same filter in both blocks
    x = {0: list(EMB[0]), 1: list(EMB[1])}
    for t in range(2):
        new = {}
        for si, sj in ((0, 1), (1, 0)):
            if t == 0:
                y = [S_IN * x[sj][(f + H_IN) % F] for f in range(F)]
            else:
                y = [0.25 * x[sj][(f + 2) % F] for f in range(F)]
            m = [y[f] * wf[f] for f in range(F)]
            h = [S_O1 * m[(f + H_O1) % F] for f in range(F)]
            new[si] = [x[si][f] + S_O2 * ssp(h[(f + H_O2) % F]) for f in range(F)]
        x = new
    E = 0.0
    for s in (0, 1):
        z = [sum(WR1[k][f] * x[s][f] for f in range(F)) for k in range(F // 2)]
        E += sum(WR2[k] * ssp(z[k]) for k in range(F // 2))
    assert E2 == pytest.approx(ALPHA * E, rel=1e-13)
