"""Parity of the CUDA path for config 3 (NEXT-2: trRosetta2-style energy on the 5-slot state, R25) against the
fp64 oracle, through the C ABI (amh_create_tr5, amh_pair_geometry, amh_coords, amh_energy, amh_energy_local, amh_run).
The CUDA path is fp64 throughout, so dE must be the oracle's to rounding and every decision identical."""
import math

import numpy as np
import pytest

import amh_inputs as gi

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def amh():
    import paper_2211_03193_b200 as pkg
    pkg.lib()
    return pkg


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def tr5(amh, orc):
    cache = {}

    def make(L, cfg_seed=1003):
        if (L, cfg_seed) not in cache:
            ref = gi.reference_torsions_tr5(L, cfg_seed)
            D, OM, TH, PH = orc.tr5_pair_geometry(ref)
            maps = (gi.distogram_from_distances(D, n_bins=37, lo=2.0, hi=20.0),
                    gi.periodic_map_from_values(OM, 24, -math.pi, math.pi, True),
                    gi.periodic_map_from_values(TH, 24, -math.pi, math.pi, True),
                    gi.periodic_map_from_values(PH, 12, 0.0, math.pi, False))
            edges = gi.bin_edges(37, 2.0, 20.0)
            m = orc.TR5Model(maps[0], edges, maps[1], maps[2], maps[3])
            g = amh.AMH(maps[0], edges, orientation=maps[1:])
            cache[(L, cfg_seed)] = (ref, maps, edges, m, g)
        return cache[(L, cfg_seed)]
    return make


def _angdiff(a, b):
    d = np.abs(a - b)
    return np.minimum(d, np.abs(d - 2 * math.pi))


def test_tr5_degenerate_geometry_scores_like_libm_atan2(amh, torch):
    # cb_len = 0 puts every C-beta on its C-alpha: in omega = dihedral CA_i, CB_i, CB_j, CA_j the first bond vector
    # is the zero vector, in theta = dihedral N_i, CA_i, CB_i, CB_j the axis is, in phi = angle CA_i, CB_i, CB_j one arm
    # is: the device's branch-free atan2 is handed (+-0, +-0) exactly.  libm's atan2 (the oracle's) returns 0 or +-pi
    # there, never +-pi/4 or +-3 pi/4 (which a zero vector sorted into the "diagonal" octant would give).  The oracle's
    # own value is not compared: its projection form reaches the zero vector with other signs of zero, and its
    # acos(0/0) is NaN for phi.
    L = 7
    flat = [np.full((L, L, nb), 1.0 / nb, np.float32) for nb in (37, 24, 24, 12)]
    g = amh.AMH(flat[0], gi.bin_edges(37, 2.0, 20.0), amh.default_options(cb_len=0.0), orientation=flat[1:])
    s = gi.initial_states_tr5(3, L, 5)
    cb, at = g.coords(torch.from_numpy(s).cuda(), atoms=True)
    at = at.cpu().numpy()
    assert np.array_equal(at[:, :, 3], at[:, :, 1])                       # CB == CA, exactly
    d, om, th, ph = [x.cpu().numpy() for x in g.pair_geometry(torch.from_numpy(s).cuda())]
    off = ~np.eye(L, dtype=bool)
    for name, a in (("omega", om), ("theta", th), ("phi", ph)):
        v = np.abs(a[:, off])
        assert np.all((v == 0.0) | (np.abs(v - math.pi) < 1e-15)), (name, np.unique(np.round(v, 6)))
    assert np.all(d[:, off] > 1.0)                                        # the CAs themselves are apart
    e = g.energy(torch.from_numpy(s).cuda()).cpu().numpy()
    assert np.all(np.isfinite(e))
    g.close()


@pytest.mark.parametrize("L", [1, 2, 5, 33, 300])
def test_tr5_coords_and_pair_geometry_parity(amh, orc, torch, tr5, L):
    ref, maps, edges, m, g = tr5(L)
    assert g.n == 5 * L
    s = np.concatenate([gi.initial_states_tr5(5, L, 7), ref[None]])
    cb, at = g.coords(torch.from_numpy(s).cuda(), atoms=True)
    d, om, th, ph = [x.cpu().numpy() for x in g.pair_geometry(torch.from_numpy(s).cuda())]
    for b in range(len(s)):
        N, CA, Cc, CB = orc.tr5_coords(s[b])
        want = np.stack([N, CA, Cc, CB], axis=1)
        assert np.abs(at[b].cpu().numpy() - want).max() < 1e-9
        assert np.abs(cb[b].cpu().numpy() - CB).max() <= 1e-4
        if L > 1 and (b < 2 or b == len(s) - 1):
            D, OM, TH, PH = orc.tr5_pair_geometry(s[b])
            assert np.abs(d[b] - D).max() < 1e-9
            assert _angdiff(om[b], OM).max() < 1e-8 and _angdiff(th[b], TH).max() < 1e-8 and np.abs(ph[b] - PH).max() < 1e-7


@pytest.mark.parametrize("L,B", [(4, 64), (33, 200), (64, 200), (300, 24)])
def test_tr5_energy_parity(amh, orc, torch, tr5, L, B):
    ref, maps, edges, m, g = tr5(L)
    s = np.concatenate([gi.initial_states_tr5(B, L, 11), ref[None]])
    sd = torch.from_numpy(s).cuda()
    e = g.energy(sd).cpu().numpy().astype(np.float64)
    want = m.energy(s)
    rel = np.abs(e - want) / np.abs(want)
    assert rel.max() < 1e-5, rel.max()
    print("TR5 L=%d: energy rel err max %.3g" % (L, rel.max()))
    for k, w in ((0, 3), (5 * (L // 2) + 2, 4), (5 * L - 1, 2), (7, 10 * L)):
        el = g.energy_local(sd[:5], k, w).cpu().numpy().astype(np.float64)
        wl = np.array([m.energy_local(x, k, w) for x in s[:5]])
        assert np.all(np.abs(el - wl) <= 1e-5 * np.maximum(np.abs(wl), 1.0))
    assert np.array_equal(g.energy_host(s[:7]).astype(np.float64), e[:7])


def _follow(m, s0, r, steps, **kw):
    bits = r["trace_acc"].cpu().numpy()
    acc = bits & 1
    assert np.all(bits & 2)                                   # every decision of this path is an fp64 decision
    f = m.follow(s0, steps, acc, **kw)
    assert np.array_equal(f["prop"], r["trace_prop"].cpu().numpy()), "proposal values must be bit-identical (R5)"
    err = np.abs(r["trace_dE"].cpu().numpy() - f["dE"])
    diff = acc != f["acc"]
    assert np.all(np.abs(f["g"][diff]) < 1e-4)
    return dict(err=err, n_diff=int(diff.sum()), f=f, acc=acc)


def test_tr5_trajectory_parity_small(amh, orc, torch, tr5):
    L, B, sweeps = 40, 12, 4
    ref, maps, edges, m, g = tr5(L)
    s0 = gi.initial_states_tr5(B, L, 5)
    n = 5 * L
    for kw in (dict(n_global=1, n_local=2, window=5, seed=3, chain_offset=1),
               dict(n_global=0, n_local=1, window=100, seed=4, t_start=0.4, t_end=0.4),
               dict(n_global=1, n_local=1, window=3, seed=5, t_start=5.0, t_end=0.5, ramp_sweeps=6, sweep_offset=1)):
        st = torch.from_numpy(s0.copy()).cuda()
        r = g.run(st, sweeps, trace_steps=sweeps * n, **kw)
        chk = _follow(m, s0, r, sweeps * n, **kw)
        assert chk["n_diff"] == 0 and chk["err"].max() < 1e-8, chk["err"].max()
        assert np.array_equal(st.cpu().numpy(), chk["f"]["states"])
        free = m.run(s0, sweeps, **kw)
        assert np.array_equal(free["states"], st.cpu().numpy())
        assert np.array_equal(free["n_accept_local"], r["n_accept_local"].cpu().numpy())
        assert np.array_equal(free["n_accept_global"], r["n_accept_global"].cpu().numpy())
        e = r["energy"].cpu().numpy().astype(np.float64)
        assert np.all(np.abs(e - free["energy"]) < 1e-5 * np.abs(free["energy"]))
        assert np.array_equal(r["best_state"].cpu().numpy(), free["best_state"])
        k = np.arange(sweeps * n) % n
        inert = (k % 5 >= 3) | (k == 0) | (k == n - 4) | (k == n - 3)
        assert np.all(chk["acc"][:, inert] == 1) and 0 < chk["acc"][:, ~inert].mean() < 1
    # split runs compose, chain ids key the draws, the host entry point walks the same trajectory
    kw = dict(n_global=1, n_local=2, window=5, seed=3)
    a = torch.from_numpy(s0.copy()).cuda(); g.run(a, 6, **kw)
    b = torch.from_numpy(s0.copy()).cuda(); g.run(b, 2, **kw); g.run(b, 4, sweep_offset=2, **kw)
    assert torch.equal(a, b)
    c = torch.from_numpy(s0[3:].copy()).cuda(); g.run(c, 6, chain_offset=3, **kw)
    assert torch.equal(c, a[3:])
    hs = s0.copy(); g.run_host(hs, 6, **kw)
    assert np.array_equal(hs, a.cpu().numpy())


def test_tr5_trajectory_parity_config3_shape(amh, orc, torch, tr5):
    # config 3 at full width (L = 300, 2,048 chains, window 12): the first 1,000 proposals of the run (a global sweep) and
    # 1,000 proposals from the start of the first local sweep, traced for every chain and replayed by the oracle for sampled ones
    c = gi.CONFIGS[3]
    ref, maps, edges, m, g = tr5(c.L, c.cfg_seed)
    s0 = gi.initial_states_tr5(c.B, c.L, 1)
    kw = dict(n_global=c.n_global, n_local=c.n_local, window=c.window, seed=1)
    steps = 1000
    st = torch.from_numpy(s0.copy()).cuda()
    r = g.run(st, 1, trace_steps=steps, **kw)
    s1 = st.cpu().numpy().copy()
    r2 = g.run(st, 1, sweep_offset=1, trace_steps=steps, **kw)
    worst = 0.0
    for row in (0, 1023, 2047):
        for rr, start, off in ((r, s0, 0), (r2, s1, 1)):
            one = {k: rr[k][row:row + 1] for k in ("trace_acc", "trace_prop", "trace_dE")}
            chk = _follow(m, start[row:row + 1], one, steps, sweep_offset=off, chain_offset=row, **kw)
            assert chk["n_diff"] == 0
            worst = max(worst, float(chk["err"].max()))
    assert worst < 1e-7, worst
    pick = np.arange(0, c.B, c.B // 16)
    e = r2["energy"].cpu().numpy().astype(np.float64)[pick]
    want = m.energy(st.cpu().numpy()[pick])
    assert np.all(np.abs(e - want) < 1e-5 * np.abs(want))
    print("cfg3 shape: max |dE_gpu - dE_oracle| over 6 x 1000 traced steps = %.2e" % worst)


def test_tr5_boltzmann_on_device_L4(amh, orc, torch, tr5):
    from scipy import stats
    L, G, n, T = 4, 3, 20, 3.0
    ref, maps, edges, m, g = tr5(L)
    eff = [1, 2, 5, 6, 7, 10, 11, 12, 15]
    idx = np.stack(np.meshgrid(*[np.arange(G)] * 9, indexing="ij"), -1).reshape(-1, 9)
    states = np.zeros((len(idx), n), np.float32)
    for q, v in enumerate(eff):
        states[:, v] = np.float32((2 * idx[:, q] - G) / np.float32(G)) * np.float32(math.pi)
    V = m.energy(states)
    prob = np.exp(-(V - V.min()) / T); prob /= prob.sum()
    B = 98304
    st = torch.from_numpy(gi.grid_states(B, n, G, seed=21)).cuda()
    g.run(st, 100, n_global=1, n_local=0, window=0, prop_mode=amh.PROP_GRID, grid=G, seed=10, t_start=T, t_end=T, want=())
    s = st.cpu().numpy()
    cell = np.zeros(B, np.int64)
    for v in eff:
        cell = cell * G + np.rint((s[:, v].astype(np.float64) / math.pi * G + G) / 2).astype(np.int64)
    counts = np.bincount(cell, minlength=G ** 9).astype(float)
    expect = B * prob
    small = expect < 5
    cc = np.concatenate([counts[~small], [counts[small].sum()]]); ee = np.concatenate([expect[~small], [expect[small].sum()]])
    pval = float(stats.chi2.sf(((cc - ee) ** 2 / ee).sum(), len(ee) - 1))
    assert pval > 0.01, pval


def test_tr5_error_codes(amh, torch, tr5, synth):
    ref, maps, edges, m, g = tr5(5)
    bad = maps[2].copy(); bad[1, 2, 3] = np.nan
    with pytest.raises(amh.AMHError) as e:
        amh.AMH(maps[0], edges, orientation=(maps[1], bad, maps[3]))
    assert e.value.status == 1
    with pytest.raises(ValueError):
        amh.AMH(maps[0], edges, orientation=(maps[1][:4], maps[2], maps[3]))
    # amh_pair_geometry needs a TR5 context
    ref2, p2, edges2, m2 = synth(8, 1000)
    g2 = amh.AMH(p2, edges2)
    with pytest.raises(amh.AMHError):
        g2.pair_geometry(torch.zeros((1, 16), dtype=torch.float32, device="cuda"))
    # empty batch, zero sweeps
    st = torch.from_numpy(gi.initial_states_tr5(3, 5, 2)).cuda()
    r = g.run(st, 0)
    assert np.array_equal(r["energy"].cpu().numpy(), g.energy(st).cpu().numpy())
