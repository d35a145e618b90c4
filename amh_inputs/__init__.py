"""Seeded synthetic inputs for the AMH hot path (shared by tests, bench.py and smoke()).

This module holds NONE of the method's arithmetic: no NeRF, no energy, no Philox, no
Metropolis test.  It only draws seeded numbers with numpy's own generator and turns a
caller-supplied distance matrix into a distogram with the recipe BASELINE.json:7 fixes
(`configs[0]`, "Common to all configs").  The distance matrix of the reference backbone is
supplied by the caller: tests pass the oracle's coordinates, the product path passes the
CUDA library's `amh_coords` output - so neither implementation leaks into the other.

The inputs stand in for the paper's CASP domains and AlphaFold1 distograms
(PAPER.md:73, 150, 168), which are not available here; see DESIGN.md "Input recipe".
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

__all__ = [
    "Config", "CONFIGS", "bin_edges", "reference_torsions", "initial_states",
    "distogram_from_distances", "grid_states", "per_chain_temperature", "periodic_map_from_values",
    "reference_torsions_tr5", "initial_states_tr5",
]


@dataclasses.dataclass(frozen=True)
class Config:
    """One workload of BASELINE.json `configs` with SURVEY.md section 8(c) readings R10/R11/R13."""
    name: str
    L: int                 # residues
    B: int                 # chains
    n_sweeps: int          # all sweeps, global + local (R10)
    n_global: int          # sweeps per cycle judged on the global energy (Alg. 1 first loop)
    n_local: int           # sweeps per cycle judged on the local energy (Alg. 1 second loop)
    window: int            # radius w in residues (R12)
    t_start: float = 1.0
    t_end: float = 1.0
    n_bins: int = 64
    d_lo: float = 2.0
    d_hi: float = 22.0
    replicas: int = 0      # >0: per-chain constant temperatures, geometric t_start..t_end (R13, cfg 4)
    cfg_seed: int = 1000
    slots: int = 2         # variables per residue: 2 = (phi, psi); 5 = config 3's (phi, psi, omega, two inert slots)

    @property
    def n(self) -> int:
        return self.slots * self.L

    @property
    def proposals(self) -> int:
        return self.B * self.n_sweeps * self.n


# BASELINE.json:8-12.  cfg 3 is the trRosetta2-style energy on the 5-slot state (n = 5 L; R25): 37 distance bins
# over 2-20 A plus 24/24/12-bin orientation maps; it gives no sweep count (R11: 33 sweeps = three cycles are used).
CONFIGS = {
    0: Config("cfg0", L=64, B=32, n_sweeps=2200, n_global=1, n_local=10, window=8, cfg_seed=1000),
    1: Config("cfg1", L=128, B=1024, n_sweeps=10000, n_global=1, n_local=10, window=8, cfg_seed=1001),
    2: Config("cfg2", L=256, B=4096, n_sweeps=20000, n_global=1, n_local=10, window=12,
              t_start=10.0, t_end=0.1, cfg_seed=1002),
    3: Config("cfg3", L=300, B=2048, n_sweeps=33, n_global=1, n_local=10, window=12, n_bins=37, d_lo=2.0, d_hi=20.0,
              cfg_seed=1003, slots=5),
    4: Config("cfg4", L=600, B=8192, n_sweeps=300, n_global=1, n_local=2, window=12,
              t_start=0.1, t_end=5.0, replicas=8, cfg_seed=1004),
}


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed) & (2**64 - 1), int(stream)]))


def bin_edges(n_bins: int = 64, lo: float = 2.0, hi: float = 22.0) -> np.ndarray:
    """fp32 edges evenly spaced over [lo, hi] (BASELINE.json:7: 64 bins over 2-22 A)."""
    return (lo + (hi - lo) * np.arange(n_bins + 1, dtype=np.float64) / n_bins).astype(np.float32)


def _uniform_angles(rng: np.random.Generator, shape) -> np.ndarray:
    """fp32 angles uniform on [-pi, pi) on a 2^-23 lattice (every value exactly representable)."""
    h = rng.integers(-(1 << 23), 1 << 23, size=shape, dtype=np.int64)
    return (h.astype(np.float32) * np.float32(2.0 ** -23)) * np.float32(math.pi)


def reference_torsions(L: int, cfg_seed: int) -> np.ndarray:
    """Reference backbone torsions, fp32 [2L], s[2i]=phi_i, s[2i+1]=psi_i, each ~ U[-pi, pi)."""
    return _uniform_angles(_rng(cfg_seed, 16), (2 * L,))


def initial_states(B: int, n: int, seed: int, chain_offset: int = 0) -> np.ndarray:
    """Seeded random start torsions fp32 [B][n] (BASELINE.json:7 "chains start from seeded random
    torsions").  Row b depends only on (seed, chain_offset + b), so sharded runs reproduce."""
    out = np.empty((B, n), dtype=np.float32)
    for b in range(B):
        out[b] = _uniform_angles(_rng(seed, (2 << 32) + chain_offset + b), (n,))
    return out


def grid_states(B: int, n: int, grid: int, seed: int) -> np.ndarray:
    """Start torsions on the coarse grid -pi + 2 pi m / grid used by the Boltzmann pins."""
    m = _rng(seed, 3 << 32).integers(0, grid, size=(B, n), dtype=np.int64)
    return ((2 * m - grid).astype(np.float32) / np.float32(grid)) * np.float32(math.pi)


def distogram_from_distances(dstar: np.ndarray, n_bins: int = 64, lo: float = 2.0, hi: float = 22.0,
                             sigma: float = 1.0, mix: float = 0.05) -> np.ndarray:
    """fp32 [L][L][n_bins]: p_ij(b) = (1-mix) softmax_b(-(c_b - d*_ij)^2 / 2 sigma^2) + mix / n_bins.

    BASELINE.json:7.  The softmax is taken in fp64 with the maximum subtracted (R18) so rows of
    far pairs (d* >> hi) put their mass in the last bin instead of underflowing to 0/0.
    `dstar` is symmetrised; the diagonal is filled like any other entry and never read.
    """
    d = np.asarray(dstar, dtype=np.float64)
    d = 0.5 * (d + d.T)
    edges = lo + (hi - lo) * np.arange(n_bins + 1, dtype=np.float64) / n_bins
    cen = 0.5 * (edges[:-1] + edges[1:])
    L = d.shape[0]
    out = np.empty((L, L, n_bins), dtype=np.float32)
    for i in range(L):                      # row blocks keep the fp64 temporary small at L=600
        logit = -((cen[None, :] - d[i, :, None]) ** 2) / (2.0 * sigma * sigma)
        logit -= logit.max(axis=-1, keepdims=True)
        p = np.exp(logit)
        p /= p.sum(axis=-1, keepdims=True)
        out[i] = ((1.0 - mix) * p + mix / n_bins).astype(np.float32)
    return out


def per_chain_temperature(B: int, replicas: int, t_lo: float, t_hi: float, chain_offset: int = 0) -> np.ndarray:
    """cfg 4 (R13): T_chain = t_lo * (t_hi/t_lo)^((chain mod replicas)/(replicas-1)), fp32 [B]."""
    r = (np.arange(B, dtype=np.int64) + chain_offset) % replicas
    return (t_lo * (t_hi / t_lo) ** (r.astype(np.float64) / (replicas - 1))).astype(np.float32)


def reference_torsions_tr5(L: int, cfg_seed: int) -> np.ndarray:
    """Reference state of config 3, fp32 [5L]: phi, psi ~ U[-pi, pi) as in every config (BASELINE.json:7), omega = 180
    degrees (trans), the two inert slots 0."""
    s = np.zeros((L, 5), dtype=np.float32)
    s[:, :2] = reference_torsions(L, cfg_seed).reshape(L, 2)
    s[:, 2] = np.float32(math.pi)
    return s.reshape(-1)


def initial_states_tr5(B: int, L: int, seed: int, chain_offset: int = 0) -> np.ndarray:
    """Seeded random start states of config 3, fp32 [B][5L]: every slot ~ U[-pi, pi) except omega, which starts within
    +-0.3 rad of trans (a peptide bond); row b depends only on (seed, chain_offset + b)."""
    out = np.empty((B, 5 * L), dtype=np.float32)
    for b in range(B):
        r = _rng(seed, (5 << 32) + chain_offset + b)
        s = _uniform_angles(r, (L, 5))
        om = np.float32(math.pi) + (s[:, 2] * np.float32(0.3 / math.pi))
        s[:, 2] = np.where(om >= np.float32(math.pi), om - np.float32(2 * math.pi), om).astype(np.float32)
        out[b] = s.reshape(-1)
    return out


def periodic_map_from_values(x: np.ndarray, n_bins: int, lo: float, hi: float, periodic: bool, sigma_bins: float = 1.0,
                             mix: float = 0.05) -> np.ndarray:
    """fp32 [L][L][n_bins] from a caller-supplied [L][L] array of reference values (angles in radians):
    p(b) = (1 - mix) softmax_b(-(c_b - x)^2 / 2 sigma^2) + mix / n_bins, sigma = sigma_bins bin widths, the difference
    c_b - x taken around the circle when `periodic` (config 3's "seeded Gaussian-smoothed softmax around the reference
    structure's values", BASELINE.json:11).  Entries are per ORDERED pair: no symmetrisation."""
    x = np.asarray(x, dtype=np.float64)
    width = (hi - lo) / n_bins
    cen = lo + (np.arange(n_bins) + 0.5) * width
    L = x.shape[0]
    out = np.empty((L, L, n_bins), dtype=np.float32)
    for i in range(L):
        d = cen[None, :] - x[i, :, None]
        if periodic:
            span = hi - lo
            d = (d + 0.5 * span) % span - 0.5 * span
        logit = -(d ** 2) / (2.0 * (sigma_bins * width) ** 2)
        logit -= logit.max(axis=-1, keepdims=True)
        p = np.exp(logit)
        p /= p.sum(axis=-1, keepdims=True)
        out[i] = ((1.0 - mix) * p + mix / n_bins).astype(np.float32)
    return out
