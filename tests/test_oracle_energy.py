"""Pins P2, P3, P5(i,ii,iv): the oracle's V (Eq. 3a) and V_local (Eq. 3b, :81-86)."""
import math

import numpy as np
import pytest

import amh_inputs as gi


def random_rotation(rng):
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def test_rigid_motion_invariance(orc, synth):
    # P2: V depends on |x_i - x_j| only (Eq. 3a)
    ref, p, edges, m = synth(64)
    rng = np.random.default_rng(0)
    for seed in range(3):
        CB = orc.coords(gi.initial_states(1, 128, seed)[0])[3]
        R, t = random_rotation(rng), rng.normal(size=3) * 50
        CB2 = CB @ R.T + t
        v, v2 = m.energy_cb(CB), m.energy_cb(CB2)
        assert abs(v - v2) < 1e-10 * abs(v)
        for k in (0, 17, 64, 127):
            a, b = m.energy_local_cb(CB, k, 8), m.energy_local_cb(CB2, k, 8)
            assert abs(a - b) < 1e-10 * max(1.0, abs(a))


def test_interpolation_at_and_between_bin_centres(orc, synth):
    # P3 / R8: at a bin centre e_ij(c_b) = E_ij(b) exactly; half way between two centres it is their
    # mean; beyond the end centres it is constant
    ref, p, edges, m = synth(16)
    e64 = edges.astype(np.float64)
    cen = 0.5 * (e64[:-1] + e64[1:])
    for (i, j) in ((0, 3), (2, 9), (5, 15)):
        E = -np.log(p[i, j].astype(np.float64) + 1e-8)
        for b in (0, 1, 17, 62, 63):
            assert m.pair(i, j, cen[b]) == pytest.approx(E[b], abs=1e-13)
        for b in (0, 30, 62):
            assert m.pair(i, j, 0.5 * (cen[b] + cen[b + 1])) == pytest.approx(0.5 * (E[b] + E[b + 1]), abs=1e-12)
            assert m.pair(i, j, 0.75 * cen[b] + 0.25 * cen[b + 1]) == pytest.approx(0.75 * E[b] + 0.25 * E[b + 1], abs=1e-12)
        for d in (0.0, 1.0, 2.0, cen[0]):
            assert m.pair(i, j, d) == pytest.approx(E[0], abs=1e-13)
        for d in (cen[-1], 22.0, 23.0, 500.0):
            assert m.pair(i, j, d) == pytest.approx(E[-1], abs=1e-13)


def test_linear_table_gives_closed_form_energy(orc):
    # If -log p is linear in distance for every pair, linear interpolation is exact and
    # V = sum_{i<j, j-i>=3} (a_ij d_ij + b_ij) for all distances inside the centre range.  a_ij is
    # asymmetric so a transposed table index, a wrong bin offset or a dropped pair shows up.
    L, nb = 12, 64
    edges = gi.bin_edges(nb)
    cen = 0.5 * (edges[:-1].astype(np.float64) + edges[1:].astype(np.float64))
    a = np.zeros((L, L)); b = np.zeros((L, L))
    for i in range(L):
        for j in range(L):
            a[i, j] = 0.02 + 0.003 * i + 0.011 * j
            b[i, j] = 0.5 + 0.07 * i - 0.01 * j
    p = np.exp(-(a[:, :, None] * cen[None, None, :] + b[:, :, None])).astype(np.float32)
    m = orc.Model(p, edges)
    # a compact helix-like state keeps all C-beta distances within [c_0, c_last]
    s = np.empty(2 * L, np.float32); s[0::2] = math.radians(-60); s[1::2] = math.radians(-45)
    CB = orc.coords(s)[3]
    D = np.linalg.norm(CB[:, None] - CB[None], axis=-1)
    iu = np.triu_indices(L, 3)
    assert D[iu].min() > cen[0] and D[iu].max() < cen[-1]
    want = float((a[iu] * D[iu] + b[iu]).sum())
    got = float(m.energy(s)[0])
    assert abs(got - want) < 2e-6 * len(iu[0])          # fp32 rounding of p: ~6e-8 relative per bin
    # the transposed reading would be far away
    assert abs(float((a.T[iu] * D[iu] + b.T[iu]).sum()) - want) > 0.1


def test_min_sep_and_pair_count(orc):
    # R9: unordered pairs with j - i >= min_sep; a constant table counts them
    L, nb = 10, 8
    p = np.full((L, L, nb), 0.125, np.float32)
    edges = gi.bin_edges(nb)
    s = gi.initial_states(1, 2 * L, 1)[0]
    e1 = -math.log(0.125 + 1e-8)
    for m_sep, cnt in ((1, 45), (2, 36), (3, 28), (9, 1), (10, 0)):
        m = orc.Model(p, edges, orc.default_geom(min_sep=m_sep))
        assert m.energy(s)[0] == pytest.approx(cnt * e1, abs=1e-10)
    # L < min_sep + 1 is valid: zero pairs, zero energy
    m = orc.Model(np.full((3, 3, nb), 0.125, np.float32), edges)
    assert m.energy(gi.initial_states(1, 6, 1)[0])[0] == 0.0


def test_zero_probability_bins_use_eps(orc):
    # E = -log(p + 1e-8): a zero bin scores -log 1e-8 = 18.42 (BASELINE.json:7)
    L, nb = 4, 4
    p = np.zeros((L, L, nb), np.float32)
    m = orc.Model(p, gi.bin_edges(nb))
    assert m.energy(gi.initial_states(1, 8, 1)[0])[0] == pytest.approx(-math.log(1e-8), abs=1e-12)


@pytest.mark.parametrize("L", [64, 128])
def test_reference_structure_scores_near_its_own_minimum(orc, synth, L):
    # P3: the seeded reference scores within 0.0125 per pair of sum_pairs min_b E_ij(b), and far
    # below a random state (BASELINE.json north_star)
    ref, p, edges, m = synth(L, 1000 + (L == 128))
    iu = np.triu_indices(L, 3)
    bound = float(m.E.min(axis=-1)[iu].sum())
    e_ref = float(m.energy(ref)[0])
    assert bound <= e_ref <= bound + 0.0125 * len(iu[0])
    e_rand = m.energy(gi.initial_states(4, 2 * L, 5))
    assert np.all(e_rand > 2.0 * e_ref)


def test_brute_force_double_loop(orc, synth):
    # numpy restatement of Eq. 3a with R8/R9 on a few states (a cross-check, not a pin)
    L = 40
    ref, p, edges, m = synth(L)
    e64 = edges.astype(np.float64)
    delta = (e64[-1] - e64[0]) / 64
    c0 = e64[0] + delta / 2
    E = -np.log(p.astype(np.float64) + 1e-8)
    for s in gi.initial_states(3, 2 * L, 8):
        CB = orc.coords(s)[3]
        tot = 0.0
        for i in range(L):
            for j in range(i + 3, L):
                t = min(max((np.linalg.norm(CB[i] - CB[j]) - c0) / delta, 0.0), 63.0)
                b = min(int(math.floor(t)), 62)
                tot += E[i, j, b] + (t - b) * (E[i, j, b + 1] - E[i, j, b])
        assert m.energy(s)[0] == pytest.approx(tot, rel=1e-12)


def test_local_energy_is_the_windowed_sum(orc, synth):
    # P5 (i), (ii): V_local(x,k,w) sums the pairs with both residues in [c-w, c+w] (Eq. 3b, R12);
    # with w >= L-1 it is V ("global MH, i.e. d = 2n")
    L = 48
    ref, p, edges, m = synth(L)
    s = gi.initial_states(1, 2 * L, 3)[0]
    CB = orc.coords(s)[3]
    full = m.energy_cb(CB)
    for k in (0, 1, 10, 47, 48, 94, 95):
        assert m.energy_local_cb(CB, k, L - 1) == pytest.approx(full, rel=1e-13)
        assert m.energy_local_cb(CB, k, 5 * L) == pytest.approx(full, rel=1e-13)
        for w in (0, 1, 2, 5, 8, 12):
            c = k // 2
            lo, hi = max(0, c - w), min(L - 1, c + w)
            want = sum(m.pair(i, j, np.linalg.norm(CB[i] - CB[j]))
                       for i in range(lo, hi + 1) for j in range(i + 3, hi + 1))
            assert m.energy_local_cb(CB, k, w) == pytest.approx(want, rel=1e-12, abs=1e-12)
            assert m.energy_local(s, k, w) == pytest.approx(want, rel=1e-12, abs=1e-12)
    # phi_c and psi_c share the window of residue c
    assert m.energy_local_cb(CB, 20, 8) == m.energy_local_cb(CB, 21, 8)


def test_delta_energy_equals_cross_segment_sum(orc, synth):
    # P5 (iv) / PAPER.md:152: a flip moves one side rigidly, so dV (and dV_local) is the sum over the
    # pairs that straddle the flipped bond only.  This is the identity the CUDA path relies on.
    L, w = 40, 8
    ref, p, edges, m = synth(L)
    s = gi.initial_states(1, 2 * L, 4)[0]
    rng = np.random.default_rng(1)
    for k in (0, 1, 2, 13, 40, 41, 78, 79):
        s2 = s.copy(); s2[k] = np.float32(rng.uniform(-math.pi, math.pi))
        CB, CB2 = orc.coords(s)[3], orc.coords(s2)[3]
        c = k // 2
        split = c if k % 2 == 0 else c + 1
        for lo, hi, dv in ((0, L - 1, m.energy_cb(CB2) - m.energy_cb(CB)),
                           (max(0, c - w), min(L - 1, c + w), m.energy_local_cb(CB2, k, w) - m.energy_local_cb(CB, k, w))):
            cross = sum(m.pair(i, j, np.linalg.norm(CB2[i] - CB2[j])) - m.pair(i, j, np.linalg.norm(CB[i] - CB[j]))
                        for i in range(lo, split) for j in range(max(split, i + 3), hi + 1))
            assert dv == pytest.approx(cross, abs=1e-9)
