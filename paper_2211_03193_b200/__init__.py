"""paper_2211_03193_b200 - thin Python binding of the AMH C-ABI library (include/amh.h).

Argument marshalling only: every step of the hot path (Philox draws, NeRF geometry, pair energies,
Metropolis test, book-keeping) runs in the CUDA kernels of csrc/.  PyTorch supplies device memory
and streams.  There is no CPU fallback: without the compiled library (python -m
paper_2211_03193_b200.build) or without a CUDA device every call raises.

Names follow include/amh.h: amh_create -> AMH(...), amh_run -> AMH.run, amh_energy -> AMH.energy,
amh_energy_local -> AMH.energy_local, amh_coords -> AMH.coords, amh_run_host -> AMH.run_host.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

__all__ = ["AMH", "AMHError", "RUN_PT_STATIC_MAX_CHAINS", "Options", "lib", "lib_path", "default_options", "philox4x32_10", "probe_l2_read", "probe_gather",
           "PROP_UNIFORM", "PROP_GRID", "PROP_GAUSSIAN", "EXPORTS"]

PROP_UNIFORM, PROP_GRID, PROP_GAUSSIAN = 0, 1, 2
RUN_PT_STATIC_MAX_CHAINS = 65536      # AMH_RUN_PT_STATIC_MAX_CHAINS of include/amh.h

# every symbol include/amh.h declares
EXPORTS = ["amh_default_options", "amh_default_launch_options", "amh_set_launch_options", "amh_create", "amh_destroy", "amh_energy", "amh_energy_local", "amh_coords",
           "amh_create_tr5", "amh_pair_geometry", "amh_run", "amh_run_host", "amh_run_pt", "amh_run_pt_static", "amh_exchange", "amh_energy_host", "amh_launch_info", "amh_launch_shape", "amh_philox_test",
           "amh_probe_l2_read", "amh_probe_gather", "amh_launch_variant", "amh_check_status", "amh_last_error", "amh_version"]


class AMHError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__("amh status %d: %s" % (status, msg))
        self.status = status


class _ModelOptions(C.Structure):          # amh_options
    _fields_ = [(k, C.c_double) for k in (
        "len_n_ca", "len_ca_c", "len_c_n", "ang_n_ca_c", "ang_ca_c_n", "ang_c_n_ca", "omega",
        "cb_len", "cb_ang", "cb_dih", "eps", "guard_scale")] + [("min_sep", C.c_int), ("pad_", C.c_int)]


class _LaunchOptions(C.Structure):         # amh_launch_options
    _fields_ = [(k, C.c_int) for k in ("warps_per_chain", "spec_local", "lanes_per_step", "spec_global", "chains_per_cta", "ring_cols")]


class Options:
    """amh_options (the model) and amh_launch_options (the launch shape) side by side; attribute access goes to
    whichever struct has the field."""

    def __init__(self):
        object.__setattr__(self, "model", _ModelOptions())
        object.__setattr__(self, "launch", _LaunchOptions())

    def __getattr__(self, k):
        for st in (self.model, self.launch):
            if k in dict(st._fields_):
                return getattr(st, k)
        raise AttributeError(k)

    def __setattr__(self, k, v):
        for st in (self.model, self.launch):
            if k in dict(st._fields_):
                return setattr(st, k, v)
        raise AttributeError(k)


class _OrientationMaps(C.Structure):       # amh_orientation_maps
    _fields_ = [("omega", C.c_void_p), ("theta", C.c_void_p), ("phi", C.c_void_p),
                ("nb_omega", C.c_int), ("nb_theta", C.c_int), ("nb_phi", C.c_int)]


class _Schedule(C.Structure):
    _fields_ = [("n_global", C.c_int), ("n_local", C.c_int), ("window", C.c_int), ("global_first", C.c_int), ("local_stride", C.c_int)]


class _Temperature(C.Structure):
    _fields_ = [("t_start", C.c_double), ("t_end", C.c_double), ("ramp_sweeps", C.c_longlong),
                ("per_chain_T", C.c_void_p)]


class _Proposal(C.Structure):
    _fields_ = [("mode", C.c_int), ("grid", C.c_int), ("sigma_start", C.c_double), ("sigma_end", C.c_double),
                ("ramp_sweeps", C.c_longlong)]


class _Outputs(C.Structure):
    _fields_ = [("energy", C.c_void_p), ("best_energy", C.c_void_p), ("best_state", C.c_void_p),
                ("n_accept_local", C.c_void_p), ("n_accept_global", C.c_void_p),
                ("first_hit_sweep", C.c_void_p), ("energy_threshold", C.c_float), ("trace_steps", C.c_int),
                ("trace_prop", C.c_void_p), ("trace_dE", C.c_void_p), ("trace_acc", C.c_void_p)]


_lib = None


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load csrc/libamh_b200.so (fails loudly when it has not been built)."""
    global _lib
    if _lib is None:
        path = os.environ.get("AMH_B200_LIB", _build.LIB)      # another build of the same library (kernel experiments)
        if not os.path.exists(path):
            raise ImportError("%s is missing: run `python -m paper_2211_03193_b200.build` (nvcc, sm_100a); "
                              "there is no CPU fallback" % path)
        L = C.CDLL(path)
        L.amh_last_error.restype = C.c_char_p
        L.amh_version.restype = C.c_char_p
        L.amh_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int,
                                 C.c_void_p, C.c_void_p]
        L.amh_create_tr5.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.amh_pair_geometry.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.amh_destroy.argtypes = [C.c_void_p]
        L.amh_energy.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p]
        L.amh_energy_host.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p]
        L.amh_energy_local.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.amh_coords.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p, C.c_void_p]
        run_args = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_longlong, C.c_longlong, C.c_longlong,
                    C.c_void_p, C.c_void_p, C.c_void_p, C.c_ulonglong, C.c_void_p, C.c_void_p]
        L.amh_run.argtypes = run_args
        L.amh_run_host.argtypes = run_args
        L.amh_exchange.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong, C.c_int, C.c_longlong, C.c_longlong,
                                   C.c_ulonglong, C.c_void_p, C.c_void_p, C.c_void_p]
        L.amh_run_pt.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_longlong, C.c_longlong, C.c_longlong, C.c_void_p,
                                 C.c_void_p, C.c_int, C.c_void_p, C.c_ulonglong, C.c_void_p, C.c_void_p, C.c_void_p,
                                 C.c_void_p, C.c_void_p]
        L.amh_run_pt_static.argtypes = L.amh_run_pt.argtypes
        L.amh_launch_info.argtypes = [C.c_void_p, C.c_longlong, C.c_int] + [C.POINTER(C.c_int)] * 4
        L.amh_launch_shape.argtypes = [C.c_void_p, C.c_longlong, C.c_int] + [C.POINTER(C.c_int)] * 4
        L.amh_probe_l2_read.argtypes = [C.c_longlong, C.c_int, C.POINTER(C.c_double), C.c_void_p]
        L.amh_probe_gather.argtypes = [C.c_longlong, C.c_int, C.POINTER(C.c_double), C.c_void_p]
        L.amh_launch_variant.argtypes = [C.c_void_p, C.c_longlong, C.c_int] + [C.POINTER(C.c_int)] * 5
        L.amh_check_status.argtypes = [C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.amh_philox_test.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p]
        L.amh_default_options.argtypes = [C.POINTER(_ModelOptions)]
        L.amh_default_launch_options.argtypes = [C.POINTER(_LaunchOptions)]
        L.amh_set_launch_options.argtypes = [C.c_void_p, C.POINTER(_LaunchOptions)]
        _lib = L
    return _lib


def _check(st: int):
    if st != 0:
        raise AMHError(st, lib().amh_last_error().decode())


def default_options(**over) -> Options:
    o = Options()
    _check(lib().amh_default_options(C.byref(o.model)))
    _check(lib().amh_default_launch_options(C.byref(o.launch)))
    for k, v in over.items():
        setattr(o, k, v)
    return o


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2211_03193_b200 needs a CUDA device (no CPU fallback)")
    return torch


def _stream_ptr(stream=None) -> int:
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _dev(t, dtype, name):
    torch = _torch()
    if not isinstance(t, torch.Tensor):
        t = torch.as_tensor(np.ascontiguousarray(t), device="cuda")
    if t.dtype != dtype or not t.is_cuda or not t.is_contiguous():
        t = t.to(device="cuda", dtype=dtype).contiguous()
    return t


def check_status():
    """amh_check_status: (code of the largest failed device-side range check or 0, whether this is the checked build)."""
    a, b = C.c_int(), C.c_int()
    _check(lib().amh_check_status(C.byref(a), C.byref(b)))
    return a.value, bool(b.value)


def probe_l2_read(n_bytes: int, reps: int = 20) -> float:
    """amh_probe_l2_read: GB/s of a read-only sweep of an n_bytes buffer by every SM (L1 bypassed)."""
    v = C.c_double()
    _check(lib().amh_probe_l2_read(int(n_bytes), int(reps), C.byref(v), _stream_ptr()))
    return v.value


def probe_gather(n_bytes: int, reps: int = 5) -> float:
    """amh_probe_gather: 8-byte gathers per second at random entries of an n_bytes table."""
    v = C.c_double()
    _check(lib().amh_probe_gather(int(n_bytes), int(reps), C.byref(v), _stream_ptr()))
    return v.value


def philox4x32_10(ctr, key):
    """Device Philox4x32-10 of the sweep kernel on arrays ctr [N][4], key [N][2] (test hook)."""
    torch = _torch()
    c = torch.as_tensor(np.ascontiguousarray(ctr, dtype=np.uint32).view(np.int32), device="cuda")
    k = torch.as_tensor(np.ascontiguousarray(key, dtype=np.uint32).view(np.int32), device="cuda")
    out = torch.empty_like(c)
    _check(lib().amh_philox_test(c.data_ptr(), k.data_ptr(), out.data_ptr(), c.shape[0], _stream_ptr()))
    return out.cpu().numpy().view(np.uint32)


class AMH:
    """amh_ctx: energy table on the device + geometry constants (amh_create / amh_destroy)."""

    def __init__(self, distogram, bin_edges, options: Options | None = None, stream=None, orientation=None):
        """orientation = (omega, theta, phi) maps, each [L][L][bins]: amh_create_tr5 (config 3, n = 5 L variables per chain)."""
        torch = _torch()
        self._h = C.c_void_p()
        if isinstance(distogram, torch.Tensor):
            d = distogram.to(dtype=torch.float32).contiguous()
            dptr, shape = d.data_ptr(), tuple(d.shape)
        else:
            d = np.ascontiguousarray(distogram, dtype=np.float32)
            dptr, shape = d.ctypes.data, d.shape
        if len(shape) != 3 or shape[0] != shape[1]:
            raise ValueError("distogram must be [L][L][n_bins]")
        e = np.ascontiguousarray(bin_edges, dtype=np.float32)
        if e.shape != (shape[2] + 1,):
            raise ValueError("bin_edges must be [n_bins + 1]")
        self.L, self.n_bins = int(shape[0]), int(shape[2])
        self.options = options
        optp = C.byref(options.model) if options is not None else None
        if orientation is None:
            self.n = 2 * self.L
            _check(lib().amh_create(C.byref(self._h), self.L, 0, dptr, e.ctypes.data, self.n_bins, optp, _stream_ptr(stream)))
        else:
            self.n = 5 * self.L
            keep = [np.ascontiguousarray(a, dtype=np.float32) for a in orientation]
            for a in keep:
                if a.ndim != 3 or a.shape[:2] != (self.L, self.L):
                    raise ValueError("orientation maps must be [L][L][bins]")
            om = _OrientationMaps(keep[0].ctypes.data, keep[1].ctypes.data, keep[2].ctypes.data,
                                  keep[0].shape[2], keep[1].shape[2], keep[2].shape[2])
            _check(lib().amh_create_tr5(C.byref(self._h), self.L, dptr, e.ctypes.data, self.n_bins, C.byref(om), optp,
                                        _stream_ptr(stream)))
        if options is not None:
            try:
                _check(lib().amh_set_launch_options(self._h, C.byref(options.launch)))
            except AMHError:
                self.close()
                raise

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().amh_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- amh_energy / amh_energy_local / amh_coords ---------------------------------------------
    def energy(self, states, stream=None):
        torch = _torch()
        s = _dev(states, torch.float32, "states").reshape(-1, self.n)
        out = torch.empty(s.shape[0], dtype=torch.float32, device="cuda")
        _check(lib().amh_energy(self._h, s.data_ptr(), s.shape[0], out.data_ptr(), _stream_ptr(stream)))
        return out

    def energy_host(self, states: np.ndarray) -> np.ndarray:
        s = np.ascontiguousarray(states, dtype=np.float32).reshape(-1, self.n)
        out = np.empty(s.shape[0], np.float32)
        _check(lib().amh_energy_host(self._h, s.ctypes.data, s.shape[0], out.ctypes.data, _stream_ptr()))
        return out

    def energy_local(self, states, k: int, window: int, stream=None):
        torch = _torch()
        s = _dev(states, torch.float32, "states").reshape(-1, self.n)
        out = torch.empty(s.shape[0], dtype=torch.float32, device="cuda")
        _check(lib().amh_energy_local(self._h, s.data_ptr(), s.shape[0], int(k), int(window), out.data_ptr(),
                                      _stream_ptr(stream)))
        return out

    def coords(self, states, atoms: bool = False, stream=None):
        """C-beta fp32 [B][L][3]; with atoms=True also fp64 [B][L][4][3] (N, CA, C, CB)."""
        torch = _torch()
        s = _dev(states, torch.float32, "states").reshape(-1, self.n)
        B = s.shape[0]
        cb = torch.empty((B, self.L, 3), dtype=torch.float32, device="cuda")
        at = torch.empty((B, self.L, 4, 3), dtype=torch.float64, device="cuda") if atoms else None
        _check(lib().amh_coords(self._h, s.data_ptr(), B, cb.data_ptr(), at.data_ptr() if atoms else None,
                                _stream_ptr(stream)))
        return (cb, at) if atoms else cb

    def pair_geometry(self, states, stream=None):
        """amh_pair_geometry (config 3): d, omega, theta, phi as fp64 [B][L][L] device tensors."""
        torch = _torch()
        s = _dev(states, torch.float32, "states").reshape(-1, self.n)
        B = s.shape[0]
        out = [torch.empty((B, self.L, self.L), dtype=torch.float64, device="cuda") for _ in range(4)]
        _check(lib().amh_pair_geometry(self._h, s.data_ptr(), B, *[o.data_ptr() for o in out], _stream_ptr(stream)))
        return tuple(out)

    def launch_info(self, B: int, window: int = 0) -> dict:
        v = [C.c_int() for _ in range(4)]
        _check(lib().amh_launch_info(self._h, int(B), int(window), *[C.byref(x) for x in v]))
        u = [C.c_int() for _ in range(4)]
        _check(lib().amh_launch_shape(self._h, int(B), int(window), *[C.byref(x) for x in u]))
        w = [C.c_int() for _ in range(5)]
        _check(lib().amh_launch_variant(self._h, int(B), int(window), *[C.byref(x) for x in w]))
        return dict(threads_per_chain=v[0].value, smem_bytes=v[1].value, ctas_per_sm=v[2].value, n_sm=v[3].value,
                    chains_per_cta=u[0].value, warps_per_chain=u[1].value, ring_cols=u[2].value, ring_rows=u[3].value,
                    spec_global=w[0].value, ring=w[1].value, cb64=w[2].value, nspec=w[3].value, lanes_per_step=w[4].value)

    # ---- amh_run ---------------------------------------------------------------------------------
    @staticmethod
    def _structs(n_global, n_local, window, global_first, t_start, t_end, ramp_sweeps, per_chain_T_ptr,
                 prop_mode, grid, sigma_start=0.0, sigma_end=0.0, ramp_sigma=0, local_stride=0):
        return (_Schedule(n_global, n_local, window, int(bool(global_first)), int(local_stride)),
                _Temperature(t_start, t_end, ramp_sweeps, per_chain_T_ptr),
                _Proposal(prop_mode, grid, sigma_start, sigma_end, ramp_sigma))

    def run(self, states, n_sweeps: int, *, n_global=1, n_local=10, window=8, global_first=True,
            t_start=1.0, t_end=1.0, ramp_sweeps=0, per_chain_T=None, prop_mode=PROP_UNIFORM, grid=0,
            sigma_start=0.0, sigma_end=0.0, ramp_sigma=0,
            seed=1, chain_offset=0, sweep_offset=0, trace_steps=0, energy_threshold=None, local_stride=0,
            want=("energy", "best_energy", "best_state", "n_accept_local", "n_accept_global"), stream=None):
        """amh_run on a DEVICE batch; `states` (torch.float32 [B][n], cuda) is updated in place.
        Returns a dict of device tensors for the outputs named in `want` (+ traces, first_hit_sweep)."""
        torch = _torch()
        if not (isinstance(states, torch.Tensor) and states.is_cuda and states.dtype == torch.float32
                and states.is_contiguous()):
            raise ValueError("states must be a contiguous cuda float32 tensor (it is updated in place)")
        s = states.view(-1, self.n)
        B = s.shape[0]
        r = {}
        o = _Outputs()
        f32, u64 = torch.float32, torch.int64

        def alloc(name, shape, dtype):
            r[name] = torch.empty(shape, dtype=dtype, device="cuda")
            return r[name].data_ptr()
        if "energy" in want: o.energy = alloc("energy", (B,), f32)
        if "best_energy" in want: o.best_energy = alloc("best_energy", (B,), f32)
        if "best_state" in want: o.best_state = alloc("best_state", (B, self.n), f32)
        if "n_accept_local" in want: o.n_accept_local = alloc("n_accept_local", (B,), u64)
        if "n_accept_global" in want: o.n_accept_global = alloc("n_accept_global", (B,), u64)
        if energy_threshold is not None:
            o.first_hit_sweep = alloc("first_hit_sweep", (1,), u64)
            o.energy_threshold = float(energy_threshold)
        if trace_steps:
            o.trace_steps = int(trace_steps)
            o.trace_prop = alloc("trace_prop", (B, trace_steps), f32)
            o.trace_dE = alloc("trace_dE", (B, trace_steps), torch.float64)
            o.trace_acc = alloc("trace_acc", (B, trace_steps), torch.uint8)
        pct = None
        if per_chain_T is not None:
            pct = _dev(per_chain_T, f32, "per_chain_T")
            if pct.numel() != B:
                raise ValueError("per_chain_T must have B entries")
        sc, tp, pr = self._structs(n_global, n_local, window, global_first, t_start, t_end, ramp_sweeps,
                                   pct.data_ptr() if pct is not None else None, prop_mode, grid,
                                   sigma_start, sigma_end, ramp_sigma, local_stride)
        _check(lib().amh_run(self._h, s.data_ptr(), B, int(n_sweeps), int(sweep_offset), int(chain_offset),
                             C.byref(sc), C.byref(tp), C.byref(pr), int(seed), C.byref(o), _stream_ptr(stream)))
        r["_keepalive"] = pct
        return r

    # ---- amh_exchange / amh_run_pt (NEXT-3) ---------------------------------------------------------
    def exchange(self, energies, per_chain_T, replicas: int, cycle: int, seed: int = 1, chain_offset: int = 0, stream=None):
        """amh_exchange: per_chain_T (cuda float32 [B]) is updated in place; returns (n_tried, n_accepted) device tensors."""
        torch = _torch()
        e = _dev(energies, torch.float32, "energies")
        if not (isinstance(per_chain_T, torch.Tensor) and per_chain_T.is_cuda and per_chain_T.dtype == torch.float32
                and per_chain_T.is_contiguous()):
            raise ValueError("per_chain_T must be a contiguous cuda float32 tensor (it is updated in place)")
        cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
        _check(lib().amh_exchange(self._h, e.data_ptr(), per_chain_T.data_ptr(), per_chain_T.numel(), int(replicas), int(cycle),
                                  int(chain_offset), int(seed), cnt[0:1].data_ptr(), cnt[1:2].data_ptr(), _stream_ptr(stream)))
        return cnt[0:1], cnt[1:2]

    def run_pt(self, states, n_cycles: int, per_chain_T, replicas: int, *, n_global=1, n_local=2, window=8, global_first=True,
               prop_mode=PROP_UNIFORM, grid=0, sigma_start=0.0, sigma_end=0.0, ramp_sigma=0, seed=1, chain_offset=0,
               cycle_offset=0, stream=None):
        """amh_run_pt on DEVICE tensors: states [B][n] and per_chain_T [B] (cuda float32) are updated in place."""
        torch = _torch()
        for t in (states, per_chain_T):
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
                raise ValueError("states and per_chain_T must be contiguous cuda float32 tensors (updated in place)")
        s = states.view(-1, self.n)
        B = s.shape[0]
        if per_chain_T.numel() != B:
            raise ValueError("per_chain_T must have B entries")
        energy = torch.empty(B, dtype=torch.float32, device="cuda")
        best = torch.empty(B, dtype=torch.float32, device="cuda")
        cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
        sc, _, pr = self._structs(n_global, n_local, window, global_first, 1.0, 1.0, 0, None, prop_mode, grid,
                                  sigma_start, sigma_end, ramp_sigma)
        _check(lib().amh_run_pt(self._h, s.data_ptr(), B, int(n_cycles), int(cycle_offset), int(chain_offset), C.byref(sc),
                                per_chain_T.data_ptr(), int(replicas), C.byref(pr), int(seed), energy.data_ptr(),
                                best.data_ptr(), cnt[0:1].data_ptr(), cnt[1:2].data_ptr(), _stream_ptr(stream)))
        return dict(energy=energy, best_energy=best, n_swap_tried=cnt[0:1], n_swap_accepted=cnt[1:2])

    def run_pt_static(self, states, n_cycles: int, per_chain_T, replicas: int, energy, best_energy=None, counters=None, *,
                      n_global=1, n_local=2, window=8, global_first=True, prop_mode=PROP_UNIFORM, grid=0, sigma_start=0.0,
                      sigma_end=0.0, ramp_sigma=0, seed=1, chain_offset=0, cycle_offset=0, stream=None):
        """amh_run_pt_static: run_pt for callers that may not allocate device memory while they sample (a sampler
        squeezed in beside a framework that owns nearly all of HBM, a latency-bound service that cannot take the
        device-wide stall of cudaMalloc / cudaFree, code under a fixed memory plan).  The library's per-cycle scratch is
        a fixed 256 KiB array inside the library instead of a staging arena, and this wrapper allocates nothing either:
        EVERY buffer is the caller's, made once at start-up and reused -
            states [B][n], per_chain_T [B], energy [B]   cuda float32, contiguous; updated / written in place
            best_energy [B]                              cuda float32 or None
            counters [2]                                 cuda int64 (swaps tried, swaps accepted; reset by the call) or None
        B <= RUN_PT_STATIC_MAX_CHAINS, else AMHError (status UNSUPPORTED).  Results equal run_pt's.  Calls share the
        library's array: do not let two of them run on the GPU at the same time (one stream, or events between them).
        Make the first call on a device at start-up, before any stream capture in the process.  Returns None."""
        torch = _torch()

        def own(t, dtype, count, name):
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.numel() == count):
                raise ValueError("%s must be a contiguous cuda %s tensor of %d elements (the caller owns every buffer)" % (name, dtype, count))
            return t.data_ptr()
        if not (isinstance(states, torch.Tensor) and states.numel() % self.n == 0):
            raise ValueError("states must be a cuda float32 tensor [B][n]")
        B = states.numel() // self.n
        sc, _, pr = self._structs(n_global, n_local, window, global_first, 1.0, 1.0, 0, None, prop_mode, grid,
                                  sigma_start, sigma_end, ramp_sigma)
        cnt = own(counters, torch.int64, 2, "counters") if counters is not None else 0
        _check(lib().amh_run_pt_static(self._h, own(states, torch.float32, B * self.n, "states"), B, int(n_cycles), int(cycle_offset),
                                       int(chain_offset), C.byref(sc), own(per_chain_T, torch.float32, B, "per_chain_T"),
                                       int(replicas), C.byref(pr), int(seed), own(energy, torch.float32, B, "energy"),
                                       own(best_energy, torch.float32, B, "best_energy") if best_energy is not None else None,
                                       cnt or None, (cnt + 8) if cnt else None, _stream_ptr(stream)))

    def run_host(self, states: np.ndarray, n_sweeps: int, *, n_global=1, n_local=10, window=8, global_first=True,
                 t_start=1.0, t_end=1.0, ramp_sweeps=0, per_chain_T=None, prop_mode=PROP_UNIFORM, grid=0,
                 sigma_start=0.0, sigma_end=0.0, ramp_sigma=0,
                 seed=1, chain_offset=0, sweep_offset=0, trace_steps=0, energy_threshold=None, local_stride=0,
                 want=("energy", "best_energy")):
        """amh_run_host: HOST numpy buffers in and out (states updated in place); synchronous."""
        if not (isinstance(states, np.ndarray) and states.dtype == np.float32 and states.flags.c_contiguous):
            raise ValueError("states must be a C-contiguous float32 numpy array (it is updated in place)")
        s = states.reshape(-1, self.n)
        B = s.shape[0]
        r = {}
        o = _Outputs()

        def alloc(name, shape, dtype):
            r[name] = np.empty(shape, dtype=dtype)
            return r[name].ctypes.data
        if "energy" in want: o.energy = alloc("energy", (B,), np.float32)
        if "best_energy" in want: o.best_energy = alloc("best_energy", (B,), np.float32)
        if "best_state" in want: o.best_state = alloc("best_state", (B, self.n), np.float32)
        if "n_accept_local" in want: o.n_accept_local = alloc("n_accept_local", (B,), np.uint64)
        if "n_accept_global" in want: o.n_accept_global = alloc("n_accept_global", (B,), np.uint64)
        if energy_threshold is not None:
            o.first_hit_sweep = alloc("first_hit_sweep", (1,), np.int64)
            o.energy_threshold = float(energy_threshold)
        if trace_steps:
            o.trace_steps = int(trace_steps)
            o.trace_prop = alloc("trace_prop", (B, trace_steps), np.float32)
            o.trace_dE = alloc("trace_dE", (B, trace_steps), np.float64)
            o.trace_acc = alloc("trace_acc", (B, trace_steps), np.uint8)
        pct = None
        if per_chain_T is not None:
            pct = np.ascontiguousarray(per_chain_T, dtype=np.float32)
        sc, tp, pr = self._structs(n_global, n_local, window, global_first, t_start, t_end, ramp_sweeps,
                                   pct.ctypes.data if pct is not None else None, prop_mode, grid,
                                   sigma_start, sigma_end, ramp_sigma, local_stride)
        _check(lib().amh_run_host(self._h, s.ctypes.data, B, int(n_sweeps), int(sweep_offset), int(chain_offset),
                                  C.byref(sc), C.byref(tp), C.byref(pr), int(seed), C.byref(o), _stream_ptr()))
        return r
