"""ctypes front end of the fp64 CPU oracle (oracle/amh_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports, links or calls
anything under paper_2211_03193_b200/ and the CUDA path never imports it.

The arithmetic lives in amh_oracle.c; this file only marshals numpy arrays.  See that file's header
for the passages of the paper each function follows and DESIGN.md for the readings R1-R22.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "amh_oracle.c")
_LIB = os.path.join(_HERE, "libamh_oracle.so")

PROP_UNIFORM, PROP_GRID, PROP_GAUSSIAN = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, -O2, OpenMP over chains)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp",
                               "-ffp-contract=off", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Geom(C.Structure):
    _fields_ = [(k, C.c_double) for k in (
        "len_n_ca", "len_ca_c", "len_c_n", "ang_n_ca_c", "ang_ca_c_n", "ang_c_n_ca",
        "omega", "cb_len", "cb_ang", "cb_dih", "eps")] + [("min_sep", C.c_int), ("pad_", C.c_int)]


class _Model(C.Structure):
    _fields_ = [("L", C.c_int), ("nb", C.c_int), ("E", C.c_void_p),
                ("c0", C.c_double), ("delta", C.c_double), ("g", Geom)]


class _RunParams(C.Structure):
    _fields_ = [("n_sweeps", C.c_longlong), ("sweep_offset", C.c_longlong),
                ("n_global", C.c_int), ("n_local", C.c_int), ("window", C.c_int), ("global_first", C.c_int),
                ("t_start", C.c_double), ("t_end", C.c_double), ("ramp_sweeps", C.c_longlong),
                ("per_chain_T", C.c_void_p),
                ("prop_mode", C.c_int), ("grid", C.c_int),
                ("sigma_start", C.c_double), ("sigma_end", C.c_double), ("ramp_sigma", C.c_longlong),
                ("seed", C.c_ulonglong), ("chain_offset", C.c_longlong),
                ("only_k", C.c_int), ("trace_steps", C.c_int), ("n_threads", C.c_int), ("local_stride", C.c_int)]


class _Outputs(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in (
        "energy", "best_energy", "best_state", "n_accept_local", "n_accept_global",
        "n_prop_local", "n_prop_global", "sweep_energy", "trace_prop", "trace_dE", "trace_g", "trace_acc")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.amho_pair.restype = C.c_double
        _lib.amho_pair.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double]
        _lib.amho_energy_cb.restype = C.c_double
        _lib.amho_energy_local_cb.restype = C.c_double
        _lib.amho_energy.restype = C.c_double
        _lib.amho_energy_local.restype = C.c_double
        _lib.amho_temperature.restype = C.c_double
        _lib.amho_temperature.argtypes = [C.c_void_p, C.c_longlong, C.c_longlong]
    return _lib


def _p(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def num_threads() -> int:
    return int(lib().amho_num_threads())


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().amho_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def sweep_order(n_res: int, is_global: bool, stride: int) -> np.ndarray:
    """The variables in the order a sweep visits them (NEXT-4): Alg. 1's 0..n-1, or the strided order of a local sweep."""
    return np.array([lib().amho_sweep_order(C.c_int(p), C.c_int(int(is_global)), C.c_int(n_res), C.c_int(stride))
                     for p in range(2 * n_res)], dtype=np.int64)


def default_geom(**over) -> Geom:
    g = Geom()
    lib().amho_default_geom(C.byref(g))
    for k, v in over.items():
        setattr(g, k, v)
    return g


def coords(s, geom: Geom | None = None):
    """N, CA, C, CB (each fp64 [L][3]) of one torsion vector s (fp32 [2L]) in the canonical frame (R1, R4)."""
    s = np.ascontiguousarray(s, dtype=np.float32)
    L = s.shape[0] // 2
    g = geom or default_geom()
    out = [np.zeros((L, 3), dtype=np.float64) for _ in range(4)]
    lib().amho_coords(C.byref(g), C.c_int(L), _p(s), *[_p(a) for a in out])
    return tuple(out)


class Model:
    """Energy model: table E = -log(p + eps) in fp64 plus the bin geometry (Eq. 3a, R8)."""

    def __init__(self, distogram, edges, geom: Geom | None = None):
        p = np.ascontiguousarray(distogram, dtype=np.float32)
        assert p.ndim == 3 and p.shape[0] == p.shape[1]
        self.L, self.nb = int(p.shape[0]), int(p.shape[2])
        e = np.asarray(edges, dtype=np.float32).astype(np.float64)
        assert e.shape[0] == self.nb + 1
        self.delta = float((e[-1] - e[0]) / self.nb)
        self.c0 = float(e[0] + 0.5 * self.delta)
        self.geom = geom or default_geom()
        self.E = np.empty(p.shape, dtype=np.float64)
        lib().amho_table(_p(p), C.c_longlong(p.size), C.c_double(self.geom.eps), _p(self.E))
        self._m = _Model(self.L, self.nb, self.E.ctypes.data, self.c0, self.delta, self.geom)

    @property
    def n(self):
        return 2 * self.L

    def pair(self, i: int, j: int, d: float) -> float:
        row = self.E[i, j]
        return float(lib().amho_pair(_p(row), self.nb, self.c0, self.delta, float(d)))

    def energy_cb(self, CB) -> float:
        CB = np.ascontiguousarray(CB, dtype=np.float64)
        return float(lib().amho_energy_cb(C.byref(self._m), _p(CB)))

    def energy_local_cb(self, CB, k: int, w: int) -> float:
        CB = np.ascontiguousarray(CB, dtype=np.float64)
        return float(lib().amho_energy_local_cb(C.byref(self._m), _p(CB), C.c_int(k), C.c_int(w)))

    def energy(self, states, n_threads: int = 0) -> np.ndarray:
        s = np.ascontiguousarray(states, dtype=np.float32).reshape(-1, self.n)
        out = np.zeros(s.shape[0], dtype=np.float64)
        lib().amho_energy_batch(C.byref(self._m), _p(s), C.c_longlong(s.shape[0]), _p(out), C.c_int(n_threads))
        return out

    def energy_local(self, s, k: int, w: int) -> float:
        s = np.ascontiguousarray(s, dtype=np.float32)
        return float(lib().amho_energy_local(C.byref(self._m), _p(s), C.c_int(k), C.c_int(w)))

    # -- Alg. 1 ---------------------------------------------------------------------------------
    def _params(self, n_sweeps, sweep_offset, n_global, n_local, window, global_first, t_start, t_end,
                ramp_sweeps, per_chain_T, prop_mode, grid, sigma_start, sigma_end, ramp_sigma, seed,
                chain_offset, only_k, trace_steps, n_threads, local_stride=0):
        return _RunParams(n_sweeps, sweep_offset, n_global, n_local, window, int(global_first),
                          t_start, t_end, ramp_sweeps,
                          None if per_chain_T is None else per_chain_T.ctypes.data,
                          prop_mode, grid, sigma_start, sigma_end, ramp_sigma, seed, chain_offset,
                          only_k, trace_steps, n_threads, local_stride)

    def run(self, states, n_sweeps, *, n_global=1, n_local=10, window=8, global_first=True,
            t_start=1.0, t_end=1.0, ramp_sweeps=0, per_chain_T=None, prop_mode=PROP_UNIFORM, grid=0,
            sigma_start=0.0, sigma_end=0.0, ramp_sigma=0, seed=1, chain_offset=0, sweep_offset=0,
            only_k=-1, trace_steps=0, n_threads=0, record_sweeps=False, local_stride=0):
        """Free-running AMH; returns a dict (states are returned, the input is not modified)."""
        s = np.array(states, dtype=np.float32, order="C").reshape(-1, self.n)
        B = s.shape[0]
        pct = None if per_chain_T is None else np.ascontiguousarray(per_chain_T, dtype=np.float32)
        prm = self._params(n_sweeps, sweep_offset, n_global, n_local, window, global_first, t_start, t_end,
                           ramp_sweeps, pct, prop_mode, grid, sigma_start, sigma_end, ramp_sigma, seed,
                           chain_offset, only_k, trace_steps, n_threads, local_stride)
        r = dict(
            energy=np.zeros(B), best_energy=np.zeros(B), best_state=np.zeros((B, self.n), np.float32),
            n_accept_local=np.zeros(B, np.int64), n_accept_global=np.zeros(B, np.int64),
            n_prop_local=np.zeros(B, np.int64), n_prop_global=np.zeros(B, np.int64),
            sweep_energy=np.zeros((B, n_sweeps)) if record_sweeps else None,
            trace_prop=np.zeros((B, trace_steps), np.float32) if trace_steps else None,
            trace_dE=np.zeros((B, trace_steps)) if trace_steps else None,
            trace_g=np.zeros((B, trace_steps)) if trace_steps else None,
            trace_acc=np.zeros((B, trace_steps), np.uint8) if trace_steps else None)
        o = _Outputs(*[None if r[k] is None else r[k].ctypes.data for k, _ in _Outputs._fields_])
        rc = lib().amho_run(C.byref(self._m), C.byref(prm), _p(s), C.c_longlong(B), C.byref(o))
        if rc != 0:
            raise ValueError("amho_run: invalid argument")
        r["states"] = s
        return r

    def follow(self, states, steps, forced_acc, *, n_global=1, n_local=10, window=8, global_first=True,
               t_start=1.0, t_end=1.0, ramp_sweeps=0, per_chain_T=None, prop_mode=PROP_UNIFORM, grid=0,
               sigma_start=0.0, sigma_end=0.0, ramp_sigma=0, seed=1, chain_offset=0, sweep_offset=0,
               n_threads=0, forced_prop=None, local_stride=0):
        """Follow mode: replay `steps` proposals taking the decisions in forced_acc [B][steps]; with
        forced_prop [B][steps] also the proposed values (Gaussian mode, R5) - "prop" in the result
        is still this implementation's own proposal."""
        s = np.array(states, dtype=np.float32, order="C").reshape(-1, self.n)
        B = s.shape[0]
        fa = np.ascontiguousarray(forced_acc, dtype=np.uint8).reshape(B, steps)
        pct = None if per_chain_T is None else np.ascontiguousarray(per_chain_T, dtype=np.float32)
        prm = self._params(0, sweep_offset, n_global, n_local, window, global_first, t_start, t_end,
                           ramp_sweeps, pct, prop_mode, grid, sigma_start, sigma_end, ramp_sigma, seed,
                           chain_offset, -1, 0, n_threads, local_stride)
        prop = np.zeros((B, steps), np.float32)
        dE = np.zeros((B, steps))
        g = np.zeros((B, steps))
        acc = np.zeros((B, steps), np.uint8)
        fp = None if forced_prop is None else np.ascontiguousarray(forced_prop, dtype=np.float32).reshape(B, steps)
        rc = lib().amho_follow(C.byref(self._m), C.byref(prm), _p(s), C.c_longlong(B), C.c_int(steps),
                               _p(fa), _p(fp), _p(prop), _p(dE), _p(g), _p(acc))
        if rc != 0:
            raise ValueError("amho_follow: invalid argument")
        return dict(states=s, prop=prop, dE=dE, g=g, acc=acc)

    def temperature(self, t, row=0, **kw) -> float:
        d = dict(n_sweeps=0, sweep_offset=0, n_global=1, n_local=1, window=0, global_first=True, t_start=1.0,
                 t_end=1.0, ramp_sweeps=0, per_chain_T=None, prop_mode=0, grid=0, sigma_start=0.0,
                 sigma_end=0.0, ramp_sigma=0, seed=0, chain_offset=0, only_k=-1, trace_steps=0, n_threads=0)
        d.update(kw)
        if d["per_chain_T"] is not None:
            d["per_chain_T"] = np.ascontiguousarray(d["per_chain_T"], dtype=np.float32)
        prm = self._params(**d)
        return float(lib().amho_temperature(C.byref(prm), C.c_longlong(t), C.c_longlong(row)))


# ---------------------------------------------------------------------------------------------------------
# NEXT-3: replica exchange between the temperatures of a group (PAPER.md:160 names parallel tempering as the
# companion of multi-block runs; BASELINE.json:12 gives config 4 eight temperature replicas).  DESIGN.md R23.
# Plain numpy on top of Model.run; test infrastructure like everything else in this package.
# ---------------------------------------------------------------------------------------------------------
PURPOSE_SWAP = 3


def exchange(energies, T, replicas: int, cycle: int, seed: int, chain_offset: int = 0):
    """One exchange step after cycle `cycle` (R23).  Chains chain_offset + b are grouped by `replicas` consecutive
    ids; the pairs (r, r+1) of a group with r = cycle (mod 2) are tested:
        accept iff log u <= (1/T_a - 1/T_b) (V_a - V_b),   u = ((x0 >> 8) + 1) 2^-24  (R7),
        x0 = word 0 of Philox(key = seed; counter = (cycle_lo, cycle_hi, chain id of r, 3)),
    evaluated in fp64 on the fp32 energies and temperatures; an accepted pair swaps its TEMPERATURES (the states stay
    in their rows).  Returns (new T fp32 [B], accept flags of the tested pairs as a dict row_a -> 0/1, gaps)."""
    V = np.asarray(energies, dtype=np.float32).astype(np.float64)
    Tn = np.array(T, dtype=np.float32, copy=True)
    B = V.shape[0]
    if replicas < 2 or B % replicas or chain_offset % replicas:
        raise ValueError("exchange: B and chain_offset must be multiples of replicas >= 2")
    acc, gap = {}, {}
    for g0 in range(0, B, replicas):
        for r in range(cycle % 2, replicas - 1, 2):
            a, b = g0 + r, g0 + r + 1
            chain = chain_offset + a
            ctr = np.array([[cycle & 0xffffffff, (cycle >> 32) & 0xffffffff, chain & 0xffffffff, PURPOSE_SWAP]], np.uint32)
            key = np.array([[seed & 0xffffffff, (seed >> 32) & 0xffffffff]], np.uint32)
            x0 = int(np.asarray(philox4x32_10(ctr, key)).reshape(-1)[0])
            lu = math.log(((x0 >> 8) + 1) * 2.0 ** -24)
            d = (1.0 / float(Tn[a]) - 1.0 / float(Tn[b])) * (V[a] - V[b])
            ok = lu <= d
            acc[a], gap[a] = int(ok), lu - d
            if ok:
                Tn[a], Tn[b] = Tn[b], Tn[a]
    return Tn, acc, gap


def run_pt(model: "Model", states, n_cycles: int, T, replicas: int, *, n_global=1, n_local=2, window=8, seed=1,
           chain_offset=0, cycle_offset=0, n_threads: int = 0, **run_kw):
    """Alternating MH with an exchange step after every cycle: Model.run for one cycle at the chains' current
    temperatures, then exchange() on the sweep-end energies.  Returns states, final T, energies, swap counts."""
    s = np.array(states, dtype=np.float32, order="C")
    Tn = np.array(T, dtype=np.float32, copy=True)
    cyc = n_global + n_local
    n_try = n_acc = 0
    e = None
    for y in range(cycle_offset, cycle_offset + n_cycles):
        r = model.run(s, cyc, n_global=n_global, n_local=n_local, window=window, per_chain_T=Tn, seed=seed,
                      chain_offset=chain_offset, sweep_offset=y * cyc, n_threads=n_threads, **run_kw)
        s, e = r["states"], r["energy"]
        Tn, acc, _ = exchange(e, Tn, replicas, y, seed, chain_offset)
        n_try += len(acc); n_acc += sum(acc.values())
    return dict(states=s, T=Tn, energy=e, n_swap_tried=n_try, n_swap_accepted=n_acc)


# ---------------------------------------------------------------------------------------------------------
# NEXT-2: config 3, trRosetta2-style energy on the 5-slot state (BASELINE.json:11; R25).  The arithmetic is
# in amh_oracle.c ("NEXT-2" section); this only marshals.
# ---------------------------------------------------------------------------------------------------------
class _TR5Model(C.Structure):
    _fields_ = [("L", C.c_int), ("nb_d", C.c_int), ("nb_o", C.c_int), ("nb_t", C.c_int), ("nb_p", C.c_int),
                ("Ed", C.c_void_p), ("Eo", C.c_void_p), ("Et", C.c_void_p), ("Ep", C.c_void_p),
                ("c0", C.c_double), ("delta", C.c_double), ("g", Geom)]


def dihedral(a, b, c, d) -> float:
    lib().amho_dihedral.restype = C.c_double
    v = [np.ascontiguousarray(x, dtype=np.float64) for x in (a, b, c, d)]
    return float(lib().amho_dihedral(*[_p(x) for x in v]))


def angle(a, b, c) -> float:
    lib().amho_angle.restype = C.c_double
    v = [np.ascontiguousarray(x, dtype=np.float64) for x in (a, b, c)]
    return float(lib().amho_angle(*[_p(x) for x in v]))


def interp_periodic(row, x: float) -> float:
    lib().amho_interp_periodic.restype = C.c_double
    lib().amho_interp_periodic.argtypes = [C.c_void_p, C.c_int, C.c_double]
    r = np.ascontiguousarray(row, dtype=np.float64)
    return float(lib().amho_interp_periodic(_p(r), int(r.shape[0]), float(x)))


def tr5_coords(s, geom: Geom | None = None):
    """N, CA, C, CB (fp64 [L][3]) of one 5-slot state s (fp32 [5L]): R1 with omega_i = s[5i+2]."""
    s = np.ascontiguousarray(s, dtype=np.float32)
    L = s.shape[0] // 5
    g = geom or default_geom()
    out = [np.zeros((L, 3), dtype=np.float64) for _ in range(4)]
    lib().amho_tr5_coords(C.byref(g), C.c_int(L), _p(s), *[_p(a) for a in out])
    return tuple(out)


def tr5_pair_geometry(s, geom: Geom | None = None):
    """d, omega, theta, phi as [L][L] arrays of one state: entry [i][j] is the ORDERED pair (i, j) (diagonal 0)."""
    N, CA, Cc, CB = tr5_coords(s, geom)
    L = N.shape[0]
    out = [np.zeros((L, L)) for _ in range(4)]
    v = [C.c_double() for _ in range(4)]
    f = lib().amho_tr5_pair_geometry
    for i in range(L):
        for j in range(L):
            if i != j:
                f(_p(N), _p(CA), _p(CB), C.c_int(i), C.c_int(j), *[C.byref(x) for x in v])
                for q in range(4):
                    out[q][i, j] = v[q].value
    return tuple(out)


def tr5_pair_geometry_atoms(N, CA, CB, i: int, j: int):
    """amho_tr5_pair_geometry on atoms given directly (fp64 [L][3] each): d, omega, theta, phi of the ORDERED pair (i, j).
    For pin P16, which places the atoms by hand."""
    a = [np.ascontiguousarray(x, dtype=np.float64) for x in (N, CA, CB)]
    v = [C.c_double() for _ in range(4)]
    lib().amho_tr5_pair_geometry(_p(a[0]), _p(a[1]), _p(a[2]), C.c_int(i), C.c_int(j), *[C.byref(x) for x in v])
    return tuple(x.value for x in v)


class TR5Model:
    """Config 3's energy: tables E = -log(p + eps) in fp64 for the distance, omega, theta and phi maps."""

    def __init__(self, dist_p, edges, omega_p, theta_p, phi_p, geom: Geom | None = None):
        self.geom = geom or default_geom()
        self.L = int(dist_p.shape[0])
        self.n = 5 * self.L
        e = np.asarray(edges, dtype=np.float32).astype(np.float64)
        self.nb = [int(a.shape[2]) for a in (dist_p, omega_p, theta_p, phi_p)]
        self.delta = float((e[-1] - e[0]) / self.nb[0])
        self.c0 = float(e[0] + 0.5 * self.delta)
        self.E = []
        for a in (dist_p, omega_p, theta_p, phi_p):
            a = np.ascontiguousarray(a, dtype=np.float32)
            assert a.shape[:2] == (self.L, self.L)
            E = np.empty(a.shape, dtype=np.float64)
            lib().amho_table(_p(a), C.c_longlong(a.size), C.c_double(self.geom.eps), _p(E))
            self.E.append(E)
        self._m = _TR5Model(self.L, *self.nb, *[x.ctypes.data for x in self.E], self.c0, self.delta, self.geom)
        lib().amho_tr5_energy.restype = C.c_double
        lib().amho_tr5_pair.restype = C.c_double

    def energy(self, states, n_threads: int = 0) -> np.ndarray:
        s = np.ascontiguousarray(states, dtype=np.float32).reshape(-1, self.n)
        out = np.zeros(s.shape[0])
        lib().amho_tr5_energy_batch(C.byref(self._m), _p(s), C.c_longlong(s.shape[0]), _p(out), C.c_int(n_threads))
        return out

    def energy_local(self, s, k: int, w: int) -> float:
        s = np.ascontiguousarray(s, dtype=np.float32)
        return float(lib().amho_tr5_energy(C.byref(self._m), _p(s), C.c_int(k), C.c_int(w), None))

    def energy_atoms(self, N, CA, CB) -> float:
        """V from given atoms (pins: rigid-motion invariance)."""
        N, CA, CB = [np.ascontiguousarray(x, dtype=np.float64) for x in (N, CA, CB)]
        v = 0.0
        for i in range(self.L):
            for j in range(i + self.geom.min_sep, self.L):
                v += float(lib().amho_tr5_pair(C.byref(self._m), _p(N), _p(CA), _p(CB), C.c_int(i), C.c_int(j)))
        return v

    def _params(self, n_sweeps, kw):
        d = dict(sweep_offset=0, n_global=1, n_local=10, window=12, global_first=True, t_start=1.0, t_end=1.0, ramp_sweeps=0,
                 per_chain_T=None, prop_mode=PROP_UNIFORM, grid=0, sigma_start=0.0, sigma_end=0.0, ramp_sigma=0, seed=1,
                 chain_offset=0, trace_steps=0, n_threads=0)
        bad = set(kw) - set(d)
        if bad:
            raise TypeError("unknown arguments %s" % sorted(bad))
        d.update(kw)
        pct = None if d["per_chain_T"] is None else np.ascontiguousarray(d["per_chain_T"], dtype=np.float32)
        prm = _RunParams(n_sweeps, d["sweep_offset"], d["n_global"], d["n_local"], d["window"], int(d["global_first"]),
                         d["t_start"], d["t_end"], d["ramp_sweeps"], None if pct is None else pct.ctypes.data,
                         d["prop_mode"], d["grid"], d["sigma_start"], d["sigma_end"], d["ramp_sigma"], d["seed"],
                         d["chain_offset"], -1, d["trace_steps"], d["n_threads"], 0)
        return prm, pct, d

    def run(self, states, n_sweeps, **kw):
        s = np.array(states, dtype=np.float32, order="C").reshape(-1, self.n)
        B = s.shape[0]
        prm, keep, d = self._params(n_sweeps, kw)
        ts = d["trace_steps"]
        r = dict(energy=np.zeros(B), best_energy=np.zeros(B), best_state=np.zeros((B, self.n), np.float32),
                 n_accept_local=np.zeros(B, np.int64), n_accept_global=np.zeros(B, np.int64), n_prop_local=None, n_prop_global=None,
                 sweep_energy=None, trace_prop=np.zeros((B, ts), np.float32) if ts else None,
                 trace_dE=np.zeros((B, ts)) if ts else None, trace_g=np.zeros((B, ts)) if ts else None,
                 trace_acc=np.zeros((B, ts), np.uint8) if ts else None)
        o = _Outputs(*[None if r[k] is None else r[k].ctypes.data for k, _ in _Outputs._fields_])
        if lib().amho_tr5_run(C.byref(self._m), C.byref(prm), _p(s), C.c_longlong(B), C.byref(o)) != 0:
            raise ValueError("amho_tr5_run: invalid argument")
        r["states"] = s
        return r

    def follow(self, states, steps, forced_acc, **kw):
        s = np.array(states, dtype=np.float32, order="C").reshape(-1, self.n)
        B = s.shape[0]
        fa = np.ascontiguousarray(forced_acc, dtype=np.uint8).reshape(B, steps)
        prm, keep, d = self._params(0, kw)
        prop = np.zeros((B, steps), np.float32); dE = np.zeros((B, steps)); g = np.zeros((B, steps)); acc = np.zeros((B, steps), np.uint8)
        if lib().amho_tr5_follow(C.byref(self._m), C.byref(prm), _p(s), C.c_longlong(B), C.c_int(steps), _p(fa),
                                 _p(prop), _p(dE), _p(g), _p(acc)) != 0:
            raise ValueError("amho_tr5_follow: invalid argument")
        return dict(states=s, prop=prop, dE=dE, g=g, acc=acc)
