"""Pins P4, P5(iii), P6, P7 and the R5/R7 draw formulas: the oracle's Alternating MH (Alg. 1,
PAPER.md:97-123; Eq. 1a-1c :27-37; Eq. 2a-2b :43-49) against what the mathematics fixes.

None of the expected values here come from the oracle's own run loop: the Boltzmann laws are
enumerated state by state, the schedule counts are arithmetic, the draw formulas are retyped in
numpy from the Philox words.
"""
import math

import numpy as np
import pytest
from scipy import stats

import amh_inputs as gi


def _chi2_p(counts, expect):
    """Pearson chi-square p-value with cells of expectation < 5 merged into one."""
    counts = np.asarray(counts, float)
    expect = np.asarray(expect, float)
    small = expect < 5.0
    c = np.concatenate([counts[~small], [counts[small].sum()]]) if small.any() else counts
    e = np.concatenate([expect[~small], [expect[small].sum()]]) if small.any() else expect
    keep = e > 0
    c, e = c[keep], e[keep]
    x2 = float(((c - e) ** 2 / e).sum())
    return float(stats.chi2.sf(x2, len(e) - 1)), len(e)


def _grid_value(m, G):
    return np.float32((2 * m - G) / np.float32(G)) * np.float32(math.pi)


@pytest.mark.parametrize("T", [1.0, 2.5])
def test_global_mh_samples_the_boltzmann_law_L4(orc, synth, T):
    # P4 (Eq. 1a-1c): L = 4, min_sep 3 -> one pair (0,3); phi_0 and psi_3 are inert (R1), the other six
    # torsions on a 4-point grid give 4^6 = 4096 states whose Boltzmann weights are enumerated.
    # Systematic-scan single-flip MH with a symmetric proposal leaves that law invariant.
    L, G, n = 4, 4, 8
    ref, p, edges, m = synth(L, 1000)
    eff = [1, 2, 3, 4, 5, 6]
    idx = np.stack(np.meshgrid(*[np.arange(G)] * 6, indexing="ij"), -1).reshape(-1, 6)
    states = np.zeros((len(idx), n), np.float32)
    states[:, 0] = _grid_value(1, G); states[:, 7] = _grid_value(2, G)
    for q, v in enumerate(eff):
        states[:, v] = _grid_value(idx[:, q], G)
    V = m.energy(states)
    assert V.max() - V.min() > 1.0            # the law is far from uniform, so the test has power
    w = np.exp(-(V - V.min()) / T)
    prob = w / w.sum()

    B = 65536
    start = gi.grid_states(B, n, G, seed=11)
    r = m.run(start, 40, n_global=1, n_local=0, window=0, t_start=T, t_end=T,
              prop_mode=orc.PROP_GRID, grid=G, seed=5)
    s = r["states"]
    cell = np.zeros(B, np.int64)
    for v in eff:
        mm = np.rint((s[:, v].astype(np.float64) / math.pi * G + G) / 2).astype(np.int64)
        assert np.all((mm >= 0) & (mm < G))
        cell = cell * G + mm
    counts = np.bincount(cell, minlength=G ** 6)
    pval, cells = _chi2_p(counts, B * prob)
    assert cells > 500
    assert pval > 0.01, pval
    # the inert variables are always accepted, hence uniform on the grid
    for v in (0, 7):
        mm = np.rint((s[:, v].astype(np.float64) / math.pi * G + G) / 2).astype(np.int64)
        pv, _ = _chi2_p(np.bincount(mm, minlength=G), np.full(G, B / G))
        assert pv > 0.001
    # a wrong acceptance (inverted ratio) would instead concentrate on HIGH energies: check the mean
    assert abs(float(V[cell].mean()) - float((prob * V).sum())) < 0.05


def test_global_mh_boltzmann_L3_three_pairs(orc):
    # P4, second case: L = 3 with min_sep = 1 -> three pairs; effective torsions psi_0, phi_1, psi_1, phi_2
    L, G, n = 3, 6, 6
    g = orc.default_geom(min_sep=1)
    ref = gi.reference_torsions(L, 77)
    CB = orc.coords(ref, g)[3]
    D = np.linalg.norm(CB[:, None] - CB[None], axis=-1)
    # C-beta distances at L = 3 only span ~3.5-7.5 A: use a narrow bin range so several bins matter
    p = gi.distogram_from_distances(D, n_bins=16, lo=3.0, hi=8.0, sigma=0.5)
    m = orc.Model(p, gi.bin_edges(16, 3.0, 8.0), g)
    eff = [1, 2, 3, 4]
    idx = np.stack(np.meshgrid(*[np.arange(G)] * 4, indexing="ij"), -1).reshape(-1, 4)
    states = np.zeros((len(idx), n), np.float32)
    for q, v in enumerate(eff):
        states[:, v] = _grid_value(idx[:, q], G)
    V = m.energy(states)
    assert V.max() - V.min() > 2.0
    prob = np.exp(-(V - V.min())); prob /= prob.sum()
    B = 40000
    r = m.run(gi.grid_states(B, n, G, seed=3), 30, n_global=1, n_local=0, window=0,
              prop_mode=orc.PROP_GRID, grid=G, seed=9)
    cell = np.zeros(B, np.int64)
    for v in eff:
        cell = cell * G + np.rint((r["states"][:, v].astype(np.float64) / math.pi * G + G) / 2).astype(np.int64)
    pval, cells = _chi2_p(np.bincount(cell, minlength=G ** 4), B * prob)
    assert cells > 100 and pval > 0.01, (cells, pval)


@pytest.mark.parametrize("k", [9, 14])
def test_fixed_k_local_chain_samples_exp_minus_Vlocal(orc, synth, k):
    # P5 (iii) (Eq. 2a-2b, 3b): proposing only variable k, the chain on s_k is plain MH for
    # exp(-V_local(G(s), k, w) / T) over the G grid values of s_k - enumerable.  All chains start from
    # the same state, so the burn-in (150 proposals of s_k) has to cover the slowest mode.
    L, w, G, T = 16, 3, 8, 3.0
    ref, p, edges, m = synth(L, 1000)
    base = gi.grid_states(1, 2 * L, G, seed=21)[0]
    cand = np.repeat(base[None], G, 0)
    cand[:, k] = _grid_value(np.arange(G), G)
    Vl = np.array([m.energy_local(c, k, w) for c in cand])
    assert Vl.max() - Vl.min() > 0.5
    prob = np.exp(-(Vl - Vl.min()) / T); prob /= prob.sum()
    B = 30000
    r = m.run(np.repeat(base[None], B, 0), 150, n_global=0, n_local=1, window=w, t_start=T, t_end=T,
              prop_mode=orc.PROP_GRID, grid=G, seed=4, only_k=k)
    s = r["states"]
    other = np.delete(np.arange(2 * L), k)
    assert np.array_equal(s[:, other], np.repeat(base[None, other], B, 0))     # nothing else moved
    mm = np.rint((s[:, k].astype(np.float64) / math.pi * G + G) / 2).astype(np.int64)
    pval, _ = _chi2_p(np.bincount(mm, minlength=G), B * prob)
    assert pval > 0.01, pval
    # and it is NOT the law of the global energy (the window matters)
    Vg = m.energy(cand)
    pg = np.exp(-(Vg - Vg.min()) / T); pg /= pg.sum()
    assert np.abs(pg - prob).max() > 0.02


def test_draw_formulas_R5_R7(orc, synth):
    # R5 (UNIFORM proposal) and R7 (u in (0,1]) retyped from the Philox words; R6 keying.
    # With w = 0 the window holds one residue, so every local dE is exactly 0 and g = log u.
    L, B, steps = 6, 3, 24
    ref, p, edges, m = synth(L, 1000)
    s0 = gi.initial_states(B, 2 * L, 2)
    seed = (0xDEADBEEF << 32) | 0x12345678
    r = m.run(s0, 2, n_global=0, n_local=1, window=0, seed=seed, chain_offset=5, trace_steps=steps)
    for b in range(B):
        for q in range(steps):
            key = [seed & 0xFFFFFFFF, seed >> 32]
            xp = orc.philox4x32_10([q, 0, 5 + b, 0], key)
            xa = orc.philox4x32_10([q, 0, 5 + b, 1], key)
            h = np.int64(xp[0] >> 8) - (1 << 23)
            want = np.float32(np.float32(h) * np.float32(2.0 ** -23)) * np.float32(math.pi)
            assert r["trace_prop"][b, q] == want
            u = (float(xa[0] >> 8) + 1.0) * 2.0 ** -24
            assert 0.0 < u <= 1.0
            assert r["trace_dE"][b, q] == 0.0
            assert r["trace_g"][b, q] == pytest.approx(math.log(u), abs=1e-15)
            assert r["trace_acc"][b, q] == 1
    assert np.array_equal(r["states"], r["trace_prop"][:, 12:24])    # all accepted: last sweep's proposals
    # the proposal value covers [-pi, pi) and never reaches +pi
    assert -math.pi <= float(r["trace_prop"].min()) and float(r["trace_prop"].max()) < math.pi


def test_schedule_counts_and_phase_order(orc, synth):
    # P6 / R10: cycle = n_global global sweeps then n_local local sweeps; n_sweeps counts all sweeps.
    # cfg 0 shape: the first 1000 steps are 128 global + 872 local proposals (R21).  With w = 0 every
    # local dE is exactly 0, so the trace shows which steps were judged on the global energy.
    c0 = gi.CONFIGS[0]
    ref, p, edges, m = synth(c0.L, c0.cfg_seed)
    s0 = gi.initial_states(2, c0.n, 1)
    r = m.run(s0, 22, n_global=c0.n_global, n_local=c0.n_local, window=0, seed=1, trace_steps=1000)
    assert np.all(r["n_prop_global"] == 2 * c0.n) and np.all(r["n_prop_local"] == 20 * c0.n)
    nz = r["trace_dE"] != 0.0
    assert np.all(nz[:, 1:127])             # global sweep: every variable but the two inert ones moves CB
    assert not nz[:, 0].any() and not nz[:, 127].any()      # phi_0, psi_{L-1} inert (R1)
    assert not nz[:, 128:].any()            # steps 128..999 are local
    # local-first ordering
    r2 = m.run(s0, 3, n_global=1, n_local=2, window=0, global_first=False, seed=1, trace_steps=3 * c0.n)
    nz2 = (r2["trace_dE"] != 0.0).reshape(2, 3, c0.n).any(axis=2)
    assert np.array_equal(nz2, np.array([[False, False, True]] * 2))
    # sweep_offset continues the cycle where it left off
    r3 = m.run(s0, 2, n_global=1, n_local=2, window=0, seed=1, sweep_offset=2, trace_steps=2 * c0.n)
    nz3 = (r3["trace_dE"] != 0.0).reshape(2, 2, c0.n).any(axis=2)
    assert np.array_equal(nz3, np.array([[False, True]] * 2))
    assert c0.proposals == 32 * 2200 * 128


def test_temperature_schedule(orc, synth):
    # P6 / R13: geometric per sweep with exact endpoints; per-chain constants override the ramp
    ref, p, edges, m = synth(8, 1000)
    S = 20001
    kw = dict(t_start=10.0, t_end=0.1, ramp_sweeps=S)
    assert m.temperature(0, **kw) == 10.0
    assert m.temperature(S - 1, **kw) == 0.1
    assert m.temperature(S + 50, **kw) == 0.1
    assert m.temperature((S - 1) // 2, **kw) == pytest.approx(1.0, rel=1e-13)
    assert m.temperature(5000, **kw) == pytest.approx(10.0 * 0.01 ** 0.25, rel=1e-13)
    assert m.temperature(7, t_start=1.0, t_end=1.0, ramp_sweeps=0) == 1.0
    pct = gi.per_chain_temperature(16, 8, 0.1, 5.0)
    assert pct[0] == np.float32(0.1) and pct[7] == np.float32(5.0) and pct[8] == pct[0]
    assert np.allclose(pct[1:8] / pct[0:7], 50.0 ** (1 / 7), rtol=1e-6)
    assert m.temperature(3, row=5, per_chain_T=pct, **kw) == float(pct[5])
    # a hot chain accepts more than a cold one
    L = 8
    s0 = np.repeat(gi.initial_states(1, 2 * L, 3), 64, 0)
    T = np.where(np.arange(64) < 32, 0.05, 50.0).astype(np.float32)
    r = m.run(s0, 20, n_global=1, n_local=0, window=0, per_chain_T=T, seed=2)
    assert r["n_accept_global"][32:].mean() > 1.5 * r["n_accept_global"][:32].mean()


def test_determinism_split_runs_and_chain_ids(orc, synth):
    # P7: counter-based RNG -> same seed, same trajectory; run(a) then run(b, offset=a) == run(a+b);
    # a row's trajectory depends on its chain id, not on its row index
    L = 12
    ref, p, edges, m = synth(L, 1000)
    s0 = gi.initial_states(6, 2 * L, 4)
    kw = dict(n_global=1, n_local=2, window=3, seed=17)
    a = m.run(s0, 9, **kw)
    b = m.run(s0, 9, **kw)
    assert np.array_equal(a["states"], b["states"]) and np.array_equal(a["energy"], b["energy"])
    h1 = m.run(s0, 4, **kw)
    h2 = m.run(h1["states"], 5, sweep_offset=4, **kw)
    assert np.array_equal(h2["states"], a["states"])
    assert np.array_equal(h2["energy"], a["energy"])
    assert np.all(np.minimum(h1["best_energy"], h2["best_energy"]) == a["best_energy"])
    assert np.array_equal(h1["n_accept_local"] + h2["n_accept_local"], a["n_accept_local"])
    assert np.array_equal(h1["n_accept_global"] + h2["n_accept_global"], a["n_accept_global"])
    c = m.run(s0[3:], 9, chain_offset=3, **kw)
    assert np.array_equal(c["states"], a["states"][3:])
    d = m.run(s0, 9, **dict(kw, seed=18))
    assert not np.array_equal(d["states"], a["states"])
    # energies reported are the energies of the returned states; best <= every sweep end
    assert np.allclose(a["energy"], m.energy(a["states"]), rtol=0, atol=1e-9)
    e = m.run(s0, 9, record_sweeps=True, **kw)
    assert np.array_equal(e["sweep_energy"].min(axis=1), e["best_energy"])
    assert np.allclose(m.energy(e["best_state"]), e["best_energy"], rtol=0, atol=1e-9)


def test_follow_mode_reproduces_the_free_run(orc, synth):
    # the parity protocol's replay: forcing the run's own decisions reproduces its trace
    L, steps = 10, 90
    ref, p, edges, m = synth(L, 1000)
    s0 = gi.initial_states(4, 2 * L, 6)
    kw = dict(n_global=1, n_local=3, window=2, seed=23, t_start=0.7, t_end=0.7)
    r = m.run(s0, 5, trace_steps=steps, **kw)
    f = m.follow(s0, steps, r["trace_acc"], **kw)
    assert np.array_equal(f["prop"], r["trace_prop"])
    assert np.array_equal(f["dE"], r["trace_dE"])
    assert np.array_equal(f["acc"], r["trace_acc"])
    assert np.array_equal(f["g"], r["trace_g"])
    # accept rule R14: accepted iff g = log u + dE/T <= 0
    assert np.array_equal(r["trace_acc"].astype(bool), r["trace_g"] <= 0.0)
    # forcing the opposite decision at one step changes the path from there on
    forced = r["trace_acc"].copy(); forced[:, 30] ^= 1
    f2 = m.follow(s0, steps, forced, **kw)
    assert np.array_equal(f2["dE"][:, :31], r["trace_dE"][:, :31])
    assert not np.array_equal(f2["states"], f["states"])


def test_gaussian_proposal_law_wrap_and_sigma_ramp(orc, synth):
    # P8 (NEXT-1; Eq. 1b, 129, 145): s'_k = wrap(s_k + sigma_t z), z ~ N(0, 1) by Box-Muller.
    # With every decision forced to "reject" the state never moves, so the recorded proposals expose z:
    # its law is tested against the normal distribution (Kolmogorov-Smirnov), its symmetry is what Eq. 1a
    # needs, the wrap keeps values in [-pi, pi) and is congruent mod 2 pi, and sigma_t hits both ends of its ramp.
    L, B, sweeps = 16, 8, 64
    n = 2 * L
    steps = sweeps * n
    ref, p, edges, m = synth(L, 1000)
    none = np.zeros((B, steps), np.uint8)
    s0 = np.full((B, n), 0.25, np.float32)
    kw = dict(n_global=0, n_local=1, window=2, seed=9, prop_mode=orc.PROP_GAUSSIAN)
    f = m.follow(s0, steps, none, sigma_start=0.3, sigma_end=0.3, **kw)
    z = (f["prop"].astype(np.float64) - 0.25) / 0.3
    assert np.array_equal(f["states"], s0)
    assert stats.kstest(z.ravel(), "norm").pvalue > 0.01
    assert abs(z.mean()) < 4.0 / math.sqrt(z.size) and abs(z.var() - 1.0) < 0.03
    assert abs((z > 0).mean() - 0.5) < 4 * 0.5 / math.sqrt(z.size)                # symmetric proposal (Eq. 1b)
    assert abs(np.corrcoef(z[:, :-1].ravel(), z[:, 1:].ravel())[0, 1]) < 0.02     # steps draw independently
    assert not np.array_equal(z[0], z[1])                                        # chains draw independently
    # wrap: the same draws from a start next to +pi land in [-pi, pi) and are congruent mod 2 pi
    s1 = np.full((B, n), 3.1, np.float32)
    f1 = m.follow(s1, steps, none, sigma_start=0.3, sigma_end=0.3, **kw)
    v = f1["prop"].astype(np.float64)
    assert np.all((v >= -math.pi - 1e-6) & (v < math.pi)) and (v < 0).mean() > 0.3
    d = v - (np.float64(np.float32(3.1)) + 0.3 * z)
    assert np.all(np.abs(d - 2 * math.pi * np.rint(d / (2 * math.pi))) < 1e-6)
    # sigma ramp, linear in the sweep index (the paper anneals 10 -> 4 degrees over a run)
    f2 = m.follow(s0, steps, none, sigma_start=math.radians(10), sigma_end=math.radians(4), ramp_sigma=sweeps, **kw)
    dz = (f2["prop"].astype(np.float64) - 0.25).reshape(B, sweeps, n)
    assert np.allclose(dz[:, 0] / math.radians(10), z.reshape(B, sweeps, n)[:, 0], atol=2e-6)
    assert np.allclose(dz[:, -1] / math.radians(4), z.reshape(B, sweeps, n)[:, -1], atol=2e-6)
    mid = sweeps // 2
    sig_mid = math.radians(10) + (math.radians(4) - math.radians(10)) * mid / (sweeps - 1)
    assert np.allclose(dz[:, mid] / sig_mid, z.reshape(B, sweeps, n)[:, mid], atol=2e-6)
    # teacher forcing: a forced proposal replaces the own one in the state, the own one is still reported
    forced = (f["prop"] + np.float32(0.01)).astype(np.float32)
    allacc = np.ones((B, n), np.uint8)
    f3 = m.follow(s0, n, allacc, sigma_start=0.3, sigma_end=0.3, forced_prop=forced[:, :n], **kw)
    assert np.array_equal(f3["states"], forced[:, :n]) and np.array_equal(f3["prop"], f["prop"][:, :n])


def test_replica_exchange_keeps_each_temperature_boltzmann_L4(orc, synth):
    # P9 (NEXT-3, R23): pairs of chains at T = 1 and T = 2.5 on the L = 4 grid system of P4, one global sweep per cycle,
    # an exchange attempt after every cycle.  A correct swap rule leaves the product law invariant, so the state that
    # holds temperature T at the end must follow the enumerated Boltzmann law of T - for both temperatures.  A wrong
    # sign or a swapped energy difference in the rule would pull the T = 1 holder towards the T = 2.5 law.
    L, G, n = 4, 4, 8
    ref, p, edges, m = synth(L, 1000)
    eff = [1, 2, 3, 4, 5, 6]
    idx = np.stack(np.meshgrid(*[np.arange(G)] * 6, indexing="ij"), -1).reshape(-1, 6)
    states = np.zeros((len(idx), n), np.float32)
    states[:, 0] = _grid_value(1, G); states[:, 7] = _grid_value(2, G)
    for q, v in enumerate(eff):
        states[:, v] = _grid_value(idx[:, q], G)
    V = m.energy(states)
    B = 2 * 32768
    T0 = np.tile(np.array([1.0, 2.5], np.float32), B // 2)
    start = gi.grid_states(B, n, G, seed=13)
    r = orc.run_pt(m, start, 30, T0, 2, n_global=1, n_local=0, window=0, seed=6, prop_mode=orc.PROP_GRID, grid=G)
    assert 0.2 < r["n_swap_accepted"] / r["n_swap_tried"] < 1.0        # the rule is exercised in both directions
    assert r["n_swap_tried"] == 15 * (B // 2)                          # pair (0, 1) is tested on even cycles only
    assert sorted(np.unique(r["T"]).tolist()) == [1.0, 2.5]
    assert np.all(np.sort(r["T"].reshape(-1, 2), axis=1) == np.array([1.0, 2.5], np.float32))   # a permutation per group
    s = r["states"]
    cell = np.zeros(B, np.int64)
    for v in eff:
        mm = np.rint((s[:, v].astype(np.float64) / math.pi * G + G) / 2).astype(np.int64)
        cell = cell * G + mm
    for T in (1.0, 2.5):
        w = np.exp(-(V - V.min()) / T)
        prob = w / w.sum()
        sel = r["T"] == np.float32(T)
        assert sel.sum() == B // 2
        counts = np.bincount(cell[sel], minlength=len(idx))
        pval, cells = _chi2_p(counts, prob * sel.sum())
        assert pval > 0.01, (T, pval)
    # the two laws differ enough for the test to have power: the T = 1 holders tested against the T = 2.5 law fail
    w = np.exp(-(V - V.min()) / 2.5); prob = w / w.sum()
    sel = r["T"] == np.float32(1.0)
    assert _chi2_p(np.bincount(cell[sel], minlength=len(idx)), prob * sel.sum())[0] < 1e-6
    # equal temperatures: every attempt is accepted (log u <= 0) and nothing observable changes
    Te = np.ones(8, np.float32)
    Tn, acc, gap = orc.exchange(np.arange(8, dtype=np.float32), Te, 4, 1, 3)
    assert list(acc.keys()) == [1, 5] and list(acc.values()) == [1, 1] and np.array_equal(Tn, Te)   # odd cycle: pair (1, 2) of each group


# ---------------------------------------------------------------------------------------------
# NEXT-4: the strided sweep order (a variant of Alg. 1; R26)
# ---------------------------------------------------------------------------------------------
def test_strided_order_is_a_permutation_in_colour_classes(orc):
    for L, s in ((10, 4), (64, 17), (7, 25), (33, 1)):
        order = orc.sweep_order(L, False, s)
        assert sorted(order.tolist()) == list(range(2 * L))                       # every variable once per sweep
        res = order[0::2] // 2
        assert np.array_equal(order[1::2], order[0::2] + 1) and np.all(order[0::2] % 2 == 0)     # phi_c, then psi_c
        cls = res % s
        assert np.all(np.diff(cls) >= 0)                                           # classes o = 0, 1, ... in turn
        for o in range(min(s, L)):
            assert np.array_equal(res[cls == o], np.arange(o, L, s))               # c = o, o + s, o + 2s, ...
        assert np.array_equal(orc.sweep_order(L, True, s), np.arange(2 * L))       # global sweeps keep Alg. 1's order
    assert np.array_equal(orc.sweep_order(12, False, 0), np.arange(24))
    assert np.array_equal(orc.sweep_order(12, False, 1), np.arange(24))            # stride 1 IS Alg. 1's order


def test_strided_run_with_stride_1_is_alg1_and_proposals_of_a_class_do_not_interact(orc, synth):
    L, w = 40, 3
    ref, p, edges, m = synth(L, 1000)
    s0 = gi.initial_states(6, 2 * L, seed=3)
    kw = dict(n_global=0, n_local=1, window=w, seed=11)
    a = m.run(s0, 3, **kw); b = m.run(s0, 3, local_stride=1, **kw)
    assert np.array_equal(a["states"], b["states"])
    # one strided local sweep, traced; stride 2w + 1: the windows of a class are disjoint
    sd = 2 * w + 1
    n = 2 * L
    r = m.run(s0, 1, local_stride=sd, trace_steps=n, **kw)
    order = orc.sweep_order(L, False, sd)
    assert not np.array_equal(r["states"], a["states"])                            # a different trajectory than Alg. 1's
    # R26: inside a class every decision can be taken against the state at the START of the class (phi) or after the
    # class's phi moves (psi): an accepted move turns everything right of it rigidly and leaves other windows' internal
    # distances alone.  Checked with the oracle's own V_local (pin P5) on reconstructed states.
    for row in range(2):
        s = s0[row].copy()
        pos = 0
        for o in range(sd):
            cs = list(range(o, L, sd))
            for par in (0, 1):
                base = s.copy()                                                     # state at the start of this half-class
                for idx, c in enumerate(cs):
                    q = pos + 2 * idx + par
                    k = 2 * c + par
                    assert order[q] == k
                    t = base.copy(); t[k] = r["trace_prop"][row, q]
                    want = m.energy_local(t, k, w) - m.energy_local(base, k, w)
                    assert abs(r["trace_dE"][row, q] - want) < 1e-8, (o, par, c)
                    if r["trace_acc"][row, q]:
                        s[k] = r["trace_prop"][row, q]
            pos += 2 * len(cs)
        assert np.array_equal(s, r["states"][row])
    # follow mode walks the same order
    f = m.follow(s0, n, r["trace_acc"], local_stride=sd, **kw)
    assert np.array_equal(f["states"], r["states"]) and np.array_equal(f["prop"], r["trace_prop"]) and np.array_equal(f["dE"], r["trace_dE"])
