"""pv_find_static: the entry point for callers that cannot allocate device memory.

Some users of this library run where a cudaMalloc is not an option: as a plug-in of a framework that took the whole
GPU at start-up and serves memory only from its own arena, inside an event loop whose rules forbid cudaMalloc /
cudaFree after initialisation (both may stall the device for an unbounded time), or from plain C with nothing but the
input and output buffers they were handed.  For them the scratch of the kernels sits in a 16 MiB array inside the
library itself.  This file checks that the entry gives exactly what pv_find gives with a caller-owned workspace, on two
calls in a row that share that array, and that a batch too large for it is refused with its own error code.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a problem in this extra entry point
must not hide the parity tests.  It passes alone in a fresh process and after the other GPU tests alike (nothing here
depends on what earlier calls left in the array).
"""
import ctypes as C

import numpy as np
import pytest

from synth import events

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pv():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2412_14966_b200 import build as pvbuild
    pvbuild.build()
    import paper_2412_14966_b200 as pv
    return pv


def _assert_same(pv, p, got, ref, what):
    """The tolerance of the tests that compare one CUDA run with another (test_runs_are_reproducible,
    test_host_pipeline_matches_device_path): bit for bit, vertex slots beyond n_vtx being scratch."""
    m = np.arange(p.max_vtx_per_event)[None, :] < ref["n_vtx"][:, None]
    assert int(ref["n_vtx"].sum()) > 0, what
    for k in ref:
        a, b = (got[k][m], ref[k][m]) if k.startswith("vtx_") else (got[k], ref[k])
        assert np.array_equal(a, b, equal_nan=True), (what, k)


@pytest.mark.parametrize("mode", ["explicit", "multivertex"])
def test_static_workspace_entry_matches_pv_find_on_two_calls_in_a_row(pv, mode):
    import torch
    p = pv.default_params() if mode == "explicit" else pv.multivertex_params()
    # two different batches: 1000 events of configs[0], then 300 high pile-up events (other sizes, so the second call
    # finds the first one's records at other places of the shared array)
    batches = [events.generate(events.config(0)), events.generate(events.config(2, 300))]
    for d in batches:
        E, T = d["offsets"].size - 1, int(d["offsets"][-1])
        assert pv.workspace_bytes(E, T, p) <= pv.binding.STATIC_WORKSPACE_BYTES
    # the existing path, each batch with its own workspace
    want = [pv.find(d, p) for d in batches]
    # the new entry: both calls enqueued back to back on one stream (ordered, so they may share the array), read after
    runs = [pv.DeviceBatch(d, p) for d in batches]
    for b in runs:
        b.workspace = None                                   # nothing of the caller's serves as scratch
    s = torch.cuda.current_stream()
    for b in runs:
        b.find_static(stream=s)
    got = [b.results() for b in runs]
    for i in range(2):
        _assert_same(pv, p, got[i], want[i], f"{mode} call {i}")
    # once more in the other order: the array now holds the leftovers of the smaller batch on top of the larger one's
    for b in reversed(runs):
        for t in b.out.values():
            t.zero_()
        b.find_static(stream=s)
    got = [b.results() for b in runs]
    for i in range(2):
        _assert_same(pv, p, got[i], want[i], f"{mode} repeat {i}")
    info = pv.last_launch_info()
    assert info["n_kernels"] == 4, info


def test_static_workspace_entry_refuses_what_does_not_fit(pv):
    """A batch whose scratch exceeds the built-in 16 MiB is refused up front with PV_E_STATIC_LIMIT, nothing runs."""
    import torch
    p = pv.default_params()
    data = events.generate(events.config(1, 6000))            # ~700 k tracks: 28 MB of scratch
    E, T = data["offsets"].size - 1, int(data["offsets"][-1])
    assert pv.workspace_bytes(E, T, p) > pv.binding.STATIC_WORKSPACE_BYTES
    b = pv.DeviceBatch(data, p)
    b.out["n_vtx"].fill_(-7)
    with pytest.raises(pv.PvError) as err:
        b.find_static()
    assert "-6" in str(err.value) and "pv_find_static" in str(err.value)
    torch.cuda.synchronize()
    assert int((b.out["n_vtx"] != -7).sum()) == 0            # no kernel touched the outputs
    L = pv.lib()
    assert L.pv_error_string(pv.binding.E_STATIC_LIMIT).decode().startswith("batch needs more scratch")
    # an empty batch and invalid parameters behave as in pv_find
    args = [None] * 9 + [None, 0, 0, C.byref(p)] + [None] * 9 + [None]
    assert L.pv_find_static(*args) == 0
    q = pv.default_params(dz=0.3)
    args = [None] * 9 + [None, 0, 0, C.byref(q)] + [None] * 9 + [None]
    assert L.pv_find_static(*args) == -2
