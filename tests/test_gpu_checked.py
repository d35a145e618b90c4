"""The launch shapes of the parity tests through the CHECKED build of the library (-DAMH_CHECK: every table, ring and
shared-memory index of the pair loops is range-checked on the device; amh_check_status reports a failure).  This stands
in for compute-sanitizer's memcheck, which is closed on the GPU pool this was developed on (profiles/r2_sanitizer.md).
The checked library is loaded in a subprocess (AMH_B200_LIB) so that the other tests keep the product build."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r'''
import math, sys
import numpy as np, torch
sys.path.insert(0, %(root)r)
import amh_inputs as gi
import paper_2211_03193_b200 as pkg
code, checked = pkg.check_status()
assert checked and code == 0, (code, checked)

def model(L, seed, **opt):
    flat = np.full((L, L, 64), 1.0 / 64, np.float32)
    edges = gi.bin_edges(64)
    g0 = pkg.AMH(flat, edges)
    cb = g0.coords(torch.from_numpy(gi.reference_torsions(L, seed)[None]).cuda())[0].double().cpu().numpy()
    g0.close()
    D = np.linalg.norm(cb[:, None] - cb[None], axis=-1)
    return pkg.AMH(gi.distogram_from_distances(D), edges, pkg.default_options(**opt) if opt else None)

runs = 0
# config 0 in the eleven launch shapes of the trajectory test, plus strided sweeps and an unbounded guard
shapes = [(0, 0, 0, 0, 0, -1), (1, 0, 1, 0, 32, 1), (4, 1, 1, -1, 16, 0), (4, 0, 3, 0, 8, 1), (2, 0, 7, 0, 16, -1), (8, 3, 1, 0, 8, 1),
          (15, 0, 1, -1, 32, 0), (3, 2, 5, 11, 16, 1), (1, 0, 12, 12, 8, 0), (2, 16, 2, 0, 8, 0), (15, 0, 1, 0, 8, 1), (2, 0, 7, 0, 4, 1)]
for wpc, spec, cpc, ring, gl, sg in shapes:
    g = model(64, 1000, warps_per_chain=wpc, spec_local=spec, chains_per_cta=cpc, ring_cols=ring, lanes_per_step=gl, spec_global=sg)
    st = torch.from_numpy(gi.initial_states(32, 128, 1)).cuda()
    g.run(st, 24, n_global=1, n_local=10, window=8, seed=1, trace_steps=64)
    g.run(st, 5, n_global=1, n_local=3, window=8, seed=2, local_stride=17)
    g.close(); runs += 2
g = model(64, 1000, guard_scale=1e30)
st = torch.from_numpy(gi.initial_states(32, 128, 3)).cuda()
g.run(st, 3, n_global=1, n_local=2, window=8, seed=3); g.close(); runs += 1
# degenerate sizes and windows
for L in (1, 2, 3, 4, 5, 9, 33):
    g = model(L, 1000)
    st = torch.from_numpy(gi.initial_states(5, 2 * L, 2)).cuda()
    for w in (0, 1, 8, 100):
        g.run(st, 4, n_global=1, n_local=2, window=w, seed=5)
        g.run(st, 2, n_global=0, n_local=1, window=w, seed=6, local_stride=2 * min(w, max(L - 1, 0)) + 1)
        runs += 2
    g.energy(st); g.energy_local(st, 0, 3); g.close()
# the bench shapes of configs 1, 2 and 4 at full width, two cycles each
for cid in (1, 2, 4):
    c = gi.CONFIGS[cid]
    g = model(c.L, c.cfg_seed)
    st = torch.from_numpy(gi.initial_states(c.B, c.n, 1)).cuda()
    kw = dict(n_global=c.n_global, n_local=c.n_local, window=c.window, seed=1)
    if c.replicas:
        kw["per_chain_T"] = gi.per_chain_temperature(c.B, c.replicas, c.t_start, c.t_end)
    g.run(st, 2 * (c.n_global + c.n_local), **kw); g.close(); runs += 1
torch.cuda.synchronize()
code, checked = pkg.check_status()
print("checked build: %%d runs, status code %%d" %% (runs, code))
assert checked and code == 0, code
'''


def test_launch_shapes_through_the_checked_build():
    from paper_2211_03193_b200 import build
    lib = build.build_checked()
    env = dict(os.environ, AMH_B200_LIB=lib)
    out = subprocess.run([sys.executable, "-c", SCRIPT % dict(root=ROOT)], capture_output=True, text=True, env=env, timeout=1500)
    assert out.returncode == 0, (out.stdout[-2000:], out.stderr[-3000:])
    print(out.stdout.strip().splitlines()[-1])


def test_product_build_has_no_checks():
    import paper_2211_03193_b200 as pkg
    code, checked = pkg.check_status()
    assert not checked and code == 0
