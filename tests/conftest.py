import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    """The fp64 CPU oracle (compiled on first use)."""
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def synth(orc):
    """Factory: (L, cfg_seed) -> (reference torsions, distogram fp32 [L][L][64], edges, oracle Model)."""
    import numpy as np
    import amh_inputs as gi
    cache = {}

    def make(L, cfg_seed=1000, n_bins=64):
        key = (L, cfg_seed, n_bins)
        if key not in cache:
            ref = gi.reference_torsions(L, cfg_seed)
            CB = orc.coords(ref)[3]
            D = np.linalg.norm(CB[:, None] - CB[None], axis=-1)
            p = gi.distogram_from_distances(D, n_bins=n_bins)
            edges = gi.bin_edges(n_bins)
            cache[key] = (ref, p, edges, orc.Model(p, edges))
        return cache[key]
    return make
