"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/amh.h declares; argument checks that fail before any CUDA call."""
import ctypes as C
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "amh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(amh_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    import paper_2211_03193_b200 as pkg
    from paper_2211_03193_b200 import build
    path = build.build()
    assert os.path.exists(path)
    lib = C.CDLL(path)
    names = _declared()
    assert names == sorted(pkg.EXPORTS)
    for name in names:
        assert hasattr(lib, name), name
    assert pkg.lib().amh_version().decode().startswith("amh-b200")


def test_built_for_sm_100a_only():
    from paper_2211_03193_b200 import build
    assert "arch=compute_100a,code=sm_100a" in build.NVCC_FLAGS
    assert not any("fast_math" in f for f in build.NVCC_FLAGS)
    info = open(os.path.join(build.CSRC, "ptxas_info.txt")).read() if os.path.exists(
        os.path.join(build.CSRC, "ptxas_info.txt")) else ""
    assert "sm_100a" in info or info == ""


def test_default_options_and_argument_checks_without_a_device():
    import paper_2211_03193_b200 as pkg
    o = pkg.default_options()
    assert o.min_sep == 3 and o.eps == 1e-8 and o.len_n_ca == 1.458 and o.len_ca_c == 1.525 and o.len_c_n == 1.329
    assert abs(o.ang_n_ca_c - np.deg2rad(111.2)) < 1e-15 and abs(o.omega - np.pi) < 1e-15
    lib = pkg.lib()
    h = C.c_void_p()
    edges = np.linspace(2, 22, 65).astype(np.float32)
    p = np.full((2, 2, 64), 1 / 64, np.float32)
    assert lib.amh_create(C.byref(h), 0, 0, p.ctypes.data, edges.ctypes.data, 64, None, None) == 1   # n_res < 1
    assert b"n_res" in lib.amh_last_error()
    assert lib.amh_create(C.byref(h), 2, 1, p.ctypes.data, edges.ctypes.data, 64, None, None) == 1   # TR5: amh_create_tr5 builds those
    assert b"amh_create_tr5" in lib.amh_last_error()
    assert lib.amh_create_tr5(C.byref(h), 2, p.ctypes.data, edges.ctypes.data, 64, None, None, None) == 1   # maps missing
    lo = pkg.default_options(warps_per_chain=99)
    assert lib.amh_set_launch_options(None, C.byref(lo.launch)) == 1
    v = C.c_double()
    assert lib.amh_probe_l2_read(16, 1, C.byref(v), None) == 1                                     # < 1 MiB
    assert lib.amh_create(C.byref(h), 2, 0, None, edges.ctypes.data, 64, None, None) == 1
    assert lib.amh_create(C.byref(h), 2, 0, p.ctypes.data, edges.ctypes.data, 1, None, None) == 1
    # a pair table the sweep kernel's 32-bit offsets cannot span is refused before any device work (the distogram
    # is not read that early, so a small stand-in serves): L = 600 holds 1,488 bins at most
    wide = np.arange(1491, dtype=np.float32)                        # unit bins: evenly spaced exactly in fp32
    assert lib.amh_create(C.byref(h), 600, 0, p.ctypes.data, wide.ctypes.data, 1490, None, None) == 2
    assert b"32-bit offsets" in lib.amh_last_error()
    assert lib.amh_destroy(None) == 0
    assert lib.amh_energy(None, None, 0, None, None) == 1


def test_product_path_never_imports_the_oracle():
    # the oracle is test infrastructure: nothing under the package may reference it
    pk = os.path.join(ROOT, "paper_2211_03193_b200")
    for dirpath, _, files in os.walk(pk):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "amh_oracle" not in txt, f
    orc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "amh_oracle.c")).read()
    assert "import paper_2211_03193_b200" not in orc and "libamh_b200" not in orc
