"""NEXT-4: the paper's method-level experiments, re-run on synthetic inputs through the C ABI.

    python -m paper_2211_03193_b200.experiments [--L 41] [--sweeps 1000] [--seeds 10]

Two tables, printed as markdown (nothing is compared with the paper's VALUES: its proteins and distograms are
not available; only the SHAPE of the two findings is checked):

  chains   minimum energy over a run with 10 chains against 1,000 chains (PAPER.md:168 Fig. 4C, :184: "1000 parallel
           blocks reach 12.97 % lower energy than 10 blocks"), w = 5 (the paper's d = 10),
           1,000 sweeps (82,000 proposals at L = 41, the run length of PAPER.md:184), mean over seeds.
  beta     mean over 25 chains of the minimum energy of alternating MH (1 global : 10 local sweeps) against
           global-only MH at the same number of proposals, for inverse temperatures beta = 1/T from 0.1 to 5
           (Fig. 5).

Everything runs in the CUDA library (amh_run); this module only builds the synthetic inputs and prints.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import torch
    import amh_inputs as gi
    import paper_2211_03193_b200 as pkg

    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=41)
    ap.add_argument("--sweeps", type=int, default=1000)
    ap.add_argument("--seeds", type=int, default=10)
    ap.add_argument("--window", type=int, default=5)
    args = ap.parse_args()
    L, n = args.L, 2 * args.L
    pkg.lib()
    edges = gi.bin_edges(64)
    g0 = pkg.AMH(np.full((L, L, 64), 1.0 / 64, np.float32), edges)
    ref = gi.reference_torsions(L, 1000)
    cb = g0.coords(torch.from_numpy(ref[None]).cuda())[0].double().cpu().numpy()
    g0.close()
    D = np.linalg.norm(cb[:, None] - cb[None], axis=-1)
    g = pkg.AMH(gi.distogram_from_distances(D), edges)
    e_ref = float(g.energy(torch.from_numpy(ref[None]).cuda())[0])

    def best(B, seed, **kw):
        st = torch.from_numpy(gi.initial_states(B, n, seed=seed)).cuda()
        r = g.run(st, args.sweeps, window=args.window, seed=seed, want=("best_energy",), **kw)
        return r["best_energy"].double().cpu().numpy()

    print("synthetic protein L = %d (reference structure scores %.1f), %d sweeps = %d proposals per chain, window %d\n"
          % (L, e_ref, args.sweeps, args.sweeps * n, args.window))
    print("| chains | mean over %d seeds of min energy over the chains |" % args.seeds)
    print("|---|---|")
    out = {}
    for B in (10, 1000):
        out[B] = np.mean([best(B, 100 + s, n_global=1, n_local=10).min() for s in range(args.seeds)])
        print("| %d | %.1f |" % (B, out[B]))
    print("\n1,000 chains reach %.1f %% lower energy than 10 chains (excess over the reference structure: %.1f %% lower)\n"
          % (100 * (out[10] - out[1000]) / out[10], 100 * (out[10] - out[1000]) / max(out[10] - e_ref, 1e-9)))

    print("| beta = 1/T | alternating MH 1:10, mean min energy of 25 chains | global-only MH | AMH lower by |")
    print("|---|---|---|---|")
    for beta in (0.1, 0.2, 0.5, 1.0, 2.0, 5.0):
        T = 1.0 / beta
        a = np.mean([best(25, 200 + s, n_global=1, n_local=10, t_start=T, t_end=T).mean() for s in range(args.seeds)])
        b = np.mean([best(25, 200 + s, n_global=1, n_local=0, t_start=T, t_end=T).mean() for s in range(args.seeds)])
        print("| %.1f | %.1f | %.1f | %.1f %% |" % (beta, a, b, 100 * (b - a) / b))


if __name__ == "__main__":
    main()
