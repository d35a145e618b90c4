"""amh_run_pt_static (include/amh.h): replica-exchange runs for callers that may not allocate device memory while
they sample - a sampler running beside a framework whose caching allocator already holds nearly all of HBM (a raw
cudaMalloc fails there), a service that cannot take the device-wide stall of cudaMalloc / cudaFree inside its loop, code
under a fixed memory plan.  amh_run_pt grows a staging arena with cudaMalloc for its per-cycle best energies; the static
variant keeps them in a fixed 256 KiB array inside the library, shared by all calls.

What is checked here: the new entry point gives amh_run_pt's results (same kernels in the same order, so the bars are
the ones tests/test_gpu_parity.py::test_replica_exchange_parity uses: states, temperatures and swap counters equal,
energies within 1e-5 relative) on several calls in a row WITHOUT a synchronisation between them and with batch sizes
that shrink and grow, so every call finds the previous call's values in the shared array; a batch beyond the limit is
refused with a message that names the limit; a repeated call does not lower the device's free memory; and the body of
the entry point (and of what it calls) names no allocating routine.

This file sorts last on purpose (pytest -x stops at the first failure: nothing is hidden behind it).  It builds its own
context and shares no state with the other test files, so it passes alone in a fresh process - where its first call is
the one that looks up the array's address on the device - and after them.
"""
import os
import re

import numpy as np
import pytest

import amh_inputs as gi

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def amh():
    import paper_2211_03193_b200 as pkg
    pkg.lib()           # raises if the extension is missing: no fallback
    return pkg


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def _body(src: str, signature: str) -> str:
    """Text between the braces of the function whose definition starts with `signature`."""
    at = src.index(signature)
    open_ = src.index("{", src.index(")\n", at))
    depth, q = 0, open_
    while True:
        depth += {"{": 1, "}": -1}.get(src[q], 0)
        if depth == 0:
            return src[open_:q + 1]
        q += 1


def test_entry_point_names_no_allocating_routine():
    # the promise of include/amh.h, read off the source: neither the entry point nor anything it calls on the host
    # mentions an allocating or freeing routine (comments are stripped first)
    src = open(os.path.join(ROOT, "paper_2211_03193_b200", "csrc", "amh_api.cu")).read()
    src = re.sub(r"//[^\n]*", "", src)
    for sig in ("amh_status amh_run_pt_static(", "static amh_status pt_static_scratch(", "amh_status amh_run(",
                "amh_status amh_exchange(", "static amh_status check_run(", "static SweepShape choose_shape("):
        body = _body(src, sig)
        for word in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "ensure_stage", "malloc(", "new ", "std::vector", "c->stage"):
            assert word not in body, (sig, word)
    entry = _body(src, "amh_status amh_run_pt_static(")
    assert "pt_static_scratch(device, &cycle_best)" in entry and "AMH_RUN_PT_STATIC_MAX_CHAINS" in entry
    # the scratch is file-scope device storage whose address comes from the runtime, checked, never the bare name
    assert re.search(r"static __device__ __align__\(256\) float amh_pt_static_scratch\[AMH_RUN_PT_STATIC_MAX_CHAINS\];", src)
    look = _body(src, "static amh_status pt_static_scratch(")
    assert "cudaGetSymbolAddress(&p, amh_pt_static_scratch)" in look and "e != cudaSuccess" in look
    assert src.count("amh_pt_static_scratch") == 2          # the definition and the look-up: no kernel is handed the name
    import paper_2211_03193_b200 as pkg
    hdr = open(os.path.join(ROOT, "include", "amh.h")).read()
    assert "#define AMH_RUN_PT_STATIC_MAX_CHAINS %d\n" % pkg.RUN_PT_STATIC_MAX_CHAINS in hdr


@pytest.mark.gpu
def test_static_scratch_variant_equals_run_pt_on_calls_in_a_row(amh, torch, synth):
    L, replicas = 40, 8
    ref, p, edges, _ = synth(L, 1000)
    g = amh.AMH(p, edges)
    kw = dict(n_global=1, n_local=2, window=4, seed=17)
    # (chains, cycles, seed of the start states): the batch shrinks, then grows past the first one, so the shared array
    # holds stale values both beyond and inside the rows a call uses
    calls = [(32, 6, 4), (16, 4, 9), (48, 5, 2)]
    start = [(gi.initial_states(B, 2 * L, seed=s), gi.per_chain_temperature(B, replicas, 0.1, 5.0)) for B, _, s in calls]
    # the existing path first: amh_run_pt (staging arena from cudaMalloc)
    want = []
    for (B, cycles, _), (s0, T0) in zip(calls, start):
        st, Td = torch.from_numpy(s0.copy()).cuda(), torch.from_numpy(T0.copy()).cuda()
        r = g.run_pt(st, cycles, Td, replicas, **kw)
        want.append((st, Td, r))
    torch.cuda.synchronize()
    assert sum(int(r["n_swap_accepted"].item()) for _, _, r in want) > 0          # the exchange step does something
    assert any(bool((r["best_energy"] < r["energy"]).any()) for _, _, r in want)   # and so does the per-cycle fold
    # the static path: every buffer is made up front, then the calls are enqueued back to back, nothing in between
    bufs = []
    for (B, _, _), (s0, T0) in zip(calls, start):
        bufs.append(dict(states=torch.from_numpy(s0.copy()).cuda(), T=torch.from_numpy(T0.copy()).cuda(),
                         energy=torch.full((B,), float("nan"), device="cuda"), best=torch.full((B,), float("nan"), device="cuda"),
                         cnt=torch.full((2,), -1, dtype=torch.int64, device="cuda")))
    torch.cuda.synchronize()
    for (B, cycles, _), b in zip(calls, bufs):
        assert g.run_pt_static(b["states"], cycles, b["T"], replicas, b["energy"], b["best"], b["cnt"], **kw) is None
    torch.cuda.synchronize()
    for q, ((st, Td, r), b) in enumerate(zip(want, bufs)):
        assert torch.equal(b["states"], st), q
        assert torch.equal(b["T"], Td), q
        assert int(b["cnt"][0]) == int(r["n_swap_tried"].item()) and int(b["cnt"][1]) == int(r["n_swap_accepted"].item()), q
        for got, ref_ in ((b["energy"], r["energy"]), (b["best"], r["best_energy"])):
            got, ref_ = got.cpu().numpy().astype(np.float64), ref_.cpu().numpy().astype(np.float64)
            assert np.all(np.isfinite(got)) and np.all(np.abs(got - ref_) <= 1e-5 * np.abs(ref_)), q
    # split runs compose as amh_run_pt's do (cycle_offset), and best_energy / counters may be left out
    B, cycles, _ = calls[0]
    s0, T0 = start[0]
    st2, T2, e2 = torch.from_numpy(s0.copy()).cuda(), torch.from_numpy(T0.copy()).cuda(), torch.empty(B, device="cuda")
    g.run_pt_static(st2, 4, T2, replicas, e2, **kw)
    g.run_pt_static(st2, cycles - 4, T2, replicas, e2, cycle_offset=4, **kw)
    assert torch.equal(st2, want[0][0]) and torch.equal(T2, want[0][1])
    # a repeat of a call whose kernels are all loaded leaves the device's free memory where it was
    b = bufs[2]
    b["states"].copy_(torch.from_numpy(start[2][0]).cuda()); b["T"].copy_(torch.from_numpy(start[2][1]).cuda())
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    g.run_pt_static(b["states"], calls[2][1], b["T"], replicas, b["energy"], b["best"], b["cnt"], **kw)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    assert torch.equal(b["states"], want[2][0])
    g.close()


@pytest.mark.gpu
def test_batch_beyond_the_built_in_scratch_is_refused(amh, torch, synth):
    L, replicas = 8, 8
    ref, p, edges, _ = synth(L, 1000)
    g = amh.AMH(p, edges)
    B = amh.RUN_PT_STATIC_MAX_CHAINS + replicas
    st = torch.zeros(B, 2 * L, device="cuda")
    T = torch.ones(B, device="cuda")
    e = torch.full((B,), 7.0, device="cuda")
    with pytest.raises(amh.AMHError) as err:
        g.run_pt_static(st, 1, T, replicas, e, n_global=1, n_local=1, window=2)
    assert err.value.status == 2                                    # AMH_ERR_UNSUPPORTED
    assert "AMH_RUN_PT_STATIC_MAX_CHAINS = %d" % amh.RUN_PT_STATIC_MAX_CHAINS in str(err.value)
    torch.cuda.synchronize()
    assert bool((st == 0).all()) and bool((e == 7.0).all())         # nothing was enqueued
    # the largest batch that fits is taken
    B = amh.RUN_PT_STATIC_MAX_CHAINS
    g.run_pt_static(st[:B], 1, T[:B], replicas, e[:B], n_global=1, n_local=1, window=2)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(e[:B]).all()) and bool((e[B:] == 7.0).all())
    g.close()
