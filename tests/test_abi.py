"""CPU-side checks of the C-ABI boundary (no GPU needed): the library builds, loads, exports every symbol
include/pv_finder.h declares, and validates its arguments before touching CUDA."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pv():
    from paper_2412_14966_b200 import build as pvbuild
    pvbuild.build()
    import paper_2412_14966_b200 as pv
    return pv


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "pv_finder.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+)?(?:int|float|char\s*\*|const char\s*\*)\s*\**\s*(pv_\w+)\s*\(", src, flags=re.M)
    return sorted(set(names))


def test_library_exports_every_declared_symbol(pv):
    declared = _declared_functions()
    assert len(declared) >= 12, declared
    L = pv.lib()
    for name in declared:
        assert hasattr(L, name), f"{name} declared in pv_finder.h but not exported"
    assert sorted(pv.EXPORTS) == declared


def test_default_params_are_the_papers(pv):
    p = pv.default_params()
    assert (p.z_min, p.z_max, p.dz) == (-550.0, 300.0, 0.25)
    assert p.z_split == -300.0                                                 # Table 2
    assert list(p.max_sigma_poca) == [1.5, 10.0]
    assert list(p.min_cluster_integral) == [2.5, 1.75]                         # Table 2
    assert list(p.min_tracks_seed) == [3, 2] and list(p.min_tracks_pv) == [4, 3]
    assert p.chi2_max == 12.0 and p.max_iter == 10
    assert abs(p.conv_dchi2 - 0.01) < 1e-9 and abs(p.conv_dz - 0.001) < 1e-9
    assert p.merge_ratio == 25.0 and abs(p.max_beam_dist - 0.3) < 1e-7
    assert pv.nbins(p) == 3400


def test_params_struct_matches_the_oracles_reading(pv, oracle):
    """Same field order and defaults on both sides of the parity tests (the two structs are declared
    independently)."""
    a, b = pv.default_params(), oracle.default_params()
    assert [f[0] for f in a._fields_] == [f[0] for f in b._fields_]
    assert bytes(a) == bytes(b)


def test_argument_validation_happens_before_cuda(pv):
    L = pv.lib()
    p = pv.default_params()
    out = C.c_size_t(0)
    assert L.pv_workspace_bytes(10, 1000, C.byref(p), C.byref(out)) == 0 and out.value >= 4
    assert L.pv_workspace_bytes(10, 1000, None, C.byref(out)) == -1            # PV_E_NULL
    assert L.pv_workspace_bytes(-1, 1000, C.byref(p), C.byref(out)) == -5      # PV_E_SIZE
    for bad in (dict(dz=0.0), dict(dz=-1.0), dict(dz=0.3), dict(z_max=-600.0), dict(dz=0.1),
                dict(max_vtx_per_event=0), dict(max_vtx_per_event=33), dict(max_iter=0), dict(max_iter=17),
                dict(chi2_max=0.0)):
        q = pv.default_params(**bad)
        assert L.pv_nbins(C.byref(q)) == -2, bad                              # PV_E_PARAM
        args = [None] * 9 + [None, 0, 0, C.byref(q)] + [None] * 9 + [None, 0, None]
        assert L.pv_find(*args) == -2, bad
    # template fill: the window of the widest class (2^(1/8) wider than the sigma cut) must fit the unit list too
    wide = dict(max_sigma_poca=(1.5, 127.0))
    assert L.pv_nbins(C.byref(pv.default_params(**wide))) == 3400             # polynomial window: 3052 bins <= 3072
    assert L.pv_nbins(C.byref(pv.default_params(fill_mode=1, **wide))) == -2  # class 51: 2 * 1654 + 1 = 3309 bins
    assert L.pv_nbins(C.byref(pv.default_params(fill_mode=1, max_sigma_poca=(1.5, 100.0)))) == 3400
    args = [None] * 9 + [None, 1, 0, C.byref(p)] + [None] * 9 + [None, 0, None]
    assert L.pv_find(*args) == -1                                             # NULL pointers
    assert L.pv_error_string(-2).decode() == "invalid parameter"
    assert L.pv_error_string(0).decode() == "ok"


def test_no_cpu_fallback(pv):
    """Without a CUDA device the compute entry fails loudly instead of computing on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from synth import events
    data = events.generate(events.config(0, 4))
    with pytest.raises(pv.PvError):
        pv.find(data)
    # and at the C level: valid arguments reach CUDA and come back as PV_E_CUDA
    L = pv.lib()
    p = pv.default_params()
    buf = np.zeros(1024, np.float32)
    ptr = buf.ctypes.data
    args = [ptr] * 9 + [ptr, 1, 1, C.byref(p)] + [ptr] * 9 + [ptr, 4096, None]
    assert L.pv_find(*args) == -4
    assert L.pv_last_cuda_error().decode() != ""


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2412_14966_b200")
    for dirpath, _d, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "pvref" not in src and "pv_oracle" not in src and "from oracle" not in src, f
