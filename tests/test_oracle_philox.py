"""Pin P0: the oracle's Philox4x32-10 against published known-answer vectors (R6)."""
import os

import numpy as np

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers(orc):
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        w = [int(x, 16) for x in r]
        out = orc.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in out] == w[6:10]


def test_philox_is_a_bijection_in_the_counter(orc):
    # distinct counters under one key give distinct blocks (Philox is a keyed permutation)
    seen = set()
    for c in range(2000):
        seen.add(tuple(int(x) for x in orc.philox4x32_10([c, 0, 0, 0], [7, 9])))
    assert len(seen) == 2000


def test_uniform_proposal_lattice_statistics(orc, synth):
    # R5/R7: proposals lie on the 2^-23 * pi lattice in [-pi, pi), mean ~ 0, variance ~ pi^2/3
    ref, p, edges, m = synth(8)
    r = m.run(np.zeros((64, 16), np.float32), 8, n_global=1, n_local=0, seed=5, trace_steps=128)
    x = r["trace_prop"].astype(np.float64).ravel()
    assert x.min() >= -np.pi - 1e-6 and x.max() < np.pi
    assert abs(x.mean()) < 4 * np.pi / np.sqrt(3 * x.size)
    assert abs(x.var() - np.pi ** 2 / 3) < 0.15
    h = x / np.float64(np.float32(np.pi)) * 2 ** 23
    assert np.abs(h - np.round(h)).max() < 0.51   # one fp32 rounding away from the integer lattice
