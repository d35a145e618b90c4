"""Pin P1: the oracle's x = G(s) (readings R1-R3) against what the chemistry fixes.

Everything here measures the built coordinates back with formulas that do not appear in the
oracle (arccos bond angle, atan2 IUPAC dihedral), plus two closed-form structures (the planar
all-trans chain and the right-handed alpha-helix) that pin the dihedral sign convention.
"""
import math

import numpy as np
import pytest

import amh_inputs as gi


def angle(a, b, c):
    u, v = a - b, c - b
    return math.acos(float(u @ v) / (np.linalg.norm(u) * np.linalg.norm(v)))


def dihedral(a, b, c, d):
    """IUPAC dihedral a-b-c-d: atan2(|b2| b1.(b2 x b3), (b1 x b2).(b2 x b3))."""
    b1, b2, b3 = b - a, c - b, d - c
    n1, n2 = np.cross(b1, b2), np.cross(b2, b3)
    return math.atan2(np.linalg.norm(b2) * float(b1 @ n2), float(n1 @ n2))


def wrap(x):
    return (x + math.pi) % (2 * math.pi) - math.pi


@pytest.mark.parametrize("L,seed", [(2, 1), (5, 2), (64, 3), (257, 4)])
def test_ideal_geometry_is_preserved(orc, L, seed):
    s = gi.initial_states(1, 2 * L, seed)[0]
    N, CA, C, CB = orc.coords(s)
    g = orc.default_geom()
    tol = 1e-10
    assert np.abs(np.linalg.norm(CA - N, axis=1) - 1.458).max() < tol
    assert np.abs(np.linalg.norm(C - CA, axis=1) - 1.525).max() < tol
    if L > 1:
        assert np.abs(np.linalg.norm(N[1:] - C[:-1], axis=1) - 1.329).max() < tol
    for i in range(L):
        assert abs(angle(N[i], CA[i], C[i]) - math.radians(111.2)) < tol
        assert abs(np.linalg.norm(CB[i] - CA[i]) - 1.522) < tol
        assert abs(angle(N[i], CA[i], CB[i]) - 1.927) < tol
        assert abs(wrap(dihedral(C[i], N[i], CA[i], CB[i]) - (-2.143))) < 1e-9
    for i in range(L - 1):
        assert abs(angle(CA[i], C[i], N[i + 1]) - math.radians(116.2)) < tol
        assert abs(angle(C[i], N[i + 1], CA[i + 1]) - math.radians(121.7)) < tol
        assert abs(wrap(dihedral(N[i], CA[i], C[i], N[i + 1]) - float(s[2 * i + 1]))) < 1e-9      # psi_i
        assert abs(abs(dihedral(CA[i], C[i], N[i + 1], CA[i + 1])) - math.pi) < 1e-9            # omega
        assert abs(wrap(dihedral(C[i], N[i + 1], CA[i + 1], C[i + 1]) - float(s[2 * i + 2]))) < 1e-9  # phi_{i+1}
    assert abs(g.omega - math.pi) < 1e-15


def test_canonical_frame(orc):
    # R1/R4: N_0 at the origin, CA_0 on +x, C_0 in the xy plane with y > 0
    N, CA, C, CB = orc.coords(gi.initial_states(1, 12, 9)[0])
    assert np.all(N[0] == 0)
    assert CA[0, 0] == 1.458 and CA[0, 1] == 0 and CA[0, 2] == 0
    assert C[0, 2] == 0 and C[0, 1] > 0


def test_cbeta_is_the_L_amino_acid_hand(orc):
    # R3: chirality triple product > 0, and the internal-coordinate Cbeta sits within 0.02 A of the
    # widely used fixed linear combination of b = CA-N, c = C-CA, a = b x c for ideal L residues.
    N, CA, C, CB = orc.coords(gi.initial_states(1, 80, 11)[0])
    b, c = CA - N, C - CA
    a = np.cross(b, c)
    assert np.all(np.einsum("ij,ij->i", np.cross(N - CA, C - CA), CB - CA) > 0)
    lin = -0.58273431 * a + 0.56802827 * b - 0.54067466 * c + CA
    assert np.abs(np.linalg.norm(CB - lin, axis=1)).max() < 0.02


def test_all_trans_chain_is_planar(orc):
    L = 64
    s = np.full(2 * L, np.float32(math.pi))
    N, CA, C, CB = orc.coords(s)
    # fp32(pi) exceeds pi by 8.7e-8 rad, so the chain leaves the plane by ~1e-5 A over 64 residues
    assert max(np.abs(N[:, 2]).max(), np.abs(CA[:, 2]).max(), np.abs(C[:, 2]).max()) < 1e-4
    # trans peptide: CA-CA virtual bond 3.80 A (textbook 3.80 +- 0.01)
    d = np.linalg.norm(CA[1:] - CA[:-1], axis=1)
    assert np.ptp(d) < 1e-9 and abs(d[0] - 3.80) < 0.01
    # law of cosines through C-N with the two ideal angles and the trans dihedral
    # (closed form: planar zig-zag, so CA_i, C_i, N_{i+1}, CA_{i+1} is a planar trans 4-chain)
    a1, a2 = math.radians(116.2), math.radians(121.7)
    x = 1.525 + 1.329 * math.cos(math.pi - a1) + 1.458 * math.cos(a2 - a1)
    y = 1.329 * math.sin(math.pi - a1) + 1.458 * math.sin(a2 - a1)
    assert abs(d[0] - math.hypot(x, y)) < 1e-9


def test_alpha_helix_is_right_handed_with_textbook_pitch(orc):
    # phi = -57.8, psi = -47.0 deg: textbook alpha-helix, right-handed, rise 1.5 A and 100 deg per
    # residue (3.6 residues per turn).  A flipped dihedral sign gives a left-handed helix.
    L = 40
    s = np.empty(2 * L, np.float32)
    s[0::2] = math.radians(-57.8)
    s[1::2] = math.radians(-47.0)
    CA = orc.coords(s)[1]
    v = CA[1:] - CA[:-1]
    trip = np.einsum("ij,ij->i", np.cross(v[:-2], v[1:-1]), v[2:])
    assert np.all(trip > 0)                                    # right-handed
    # helix axis direction from second differences; rise = projection of CA steps on the axis
    w = np.cross(v[1:-1] - v[:-2], v[2:] - v[1:-1])
    axis = w.mean(axis=0)
    axis /= np.linalg.norm(axis)
    rise = np.abs(v @ axis)
    assert abs(rise.mean() - 1.5) < 0.1 and np.ptp(rise) < 1e-6
    perp = v - np.outer(v @ axis, axis)
    cosang = np.einsum("ij,ij->i", perp[:-1], perp[1:]) / (np.linalg.norm(perp[:-1], axis=1) * np.linalg.norm(perp[1:], axis=1))
    turn = np.degrees(np.arccos(cosang))
    assert abs(turn.mean() - 100.0) < 3.0


def test_first_phi_and_last_psi_are_inert(orc):
    # R1: phi_0 and psi_{L-1} do not enter any coordinate
    L = 9
    s = gi.initial_states(1, 2 * L, 21)[0]
    base = np.concatenate(orc.coords(s))
    s2 = s.copy(); s2[0] += 1.0; s2[2 * L - 1] -= 2.0
    assert np.array_equal(base, np.concatenate(orc.coords(s2)))
    s3 = s.copy(); s3[1] += 1e-3
    assert np.abs(base - np.concatenate(orc.coords(s3))).max() > 1e-5


def test_flip_moves_one_side_rigidly(orc):
    # PAPER.md:152 / R19: changing phi_c moves CB_c.. rigidly, psi_c moves CB_{c+1}.. rigidly
    L = 20
    s = gi.initial_states(1, 2 * L, 22)[0]
    CB0 = orc.coords(s)[3]
    D0 = np.linalg.norm(CB0[:, None] - CB0[None], axis=-1)
    for k in (6, 7, 21, 30):
        s2 = s.copy(); s2[k] = np.float32(wrap(float(s2[k]) + 1.3))
        CB1 = orc.coords(s2)[3]
        D1 = np.linalg.norm(CB1[:, None] - CB1[None], axis=-1)
        c = k // 2
        split = c if k % 2 == 0 else c + 1
        assert np.abs(CB1[:split] - CB0[:split]).max() < 1e-12          # upstream untouched in this frame
        assert np.abs(D1[:split, :split] - D0[:split, :split]).max() < 1e-10
        assert np.abs(D1[split:, split:] - D0[split:, split:]).max() < 1e-10
        assert np.abs(D1[:split, split:] - D0[:split, split:]).max() > 1e-3
