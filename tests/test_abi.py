"""CPU checks of the boundary: libgs.so builds, loads, exports every symbol include/gs.h declares,
fails loudly without a GPU (no CPU fallback), and the product never touches the oracle."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_01164_b200 import build, api
    build.build()
    return api.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "gs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gs_[a-z_]+)\s*\(", text)))


def test_exports_match_header(lib):
    from paper_2607_01164_b200 import api
    names = _declared()
    assert {"gs_preprocess", "gs_build_accel", "gs_sample_fwd", "gs_sample_bwd"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in gs.h but not exported"
    assert set(api.EXPORTS) == set(names)


def test_struct_layouts_match_header():
    from paper_2607_01164_b200 import api
    assert ctypes.sizeof(api._Gaussians) == 48
    assert ctypes.sizeof(api._Domain) == 24
    assert api._Query.num_points.offset == 64 and api._Query.xyz.offset == 72 and api._Query.jitter.offset == 84 and ctypes.sizeof(api._Query) == 96
    assert ctypes.sizeof(api._Grads) == 48
    assert ctypes.sizeof(api._RawParams) == 48 and api._RawParams.mean.offset == 8
    assert ctypes.sizeof(api._AdamCfg) == 36 and api._AdamCfg.step.offset == 32
    assert api._Loss.defined.offset == 16 and api._Loss.num_defined.offset == 24 and ctypes.sizeof(api._Loss) == 32
    assert ctypes.sizeof(api._StatusInfo) == 48 and api._StatusInfo.decode_repeats.offset == 40   # gs_status_info: six uint64


def test_fails_loudly_without_gpu(lib):
    import torch
    from paper_2607_01164_b200 import api
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = ctypes.c_void_p()
    assert lib.gs_create(0, None, ctypes.byref(h)) == api.GS_ERR_CUDA and not h.value
    with pytest.raises(api.GsLibraryError):
        api.Context()
    # NULL-context calls return an error code instead of crashing
    assert lib.gs_preprocess(None, None, None, ctypes.c_float(0.01)) == api.GS_ERR_INVALID_ARG
    assert lib.gs_build_accel(None, None) == api.GS_ERR_INVALID_ARG


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_01164_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                # no import, include, dlopen or path reference to anything under oracle/
                assert not re.search(r"(import\s+oracle|from\s+oracle|wveg_oracle|oracle/|#include.*oracle)", src), f
