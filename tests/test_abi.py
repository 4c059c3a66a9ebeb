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
    return sorted(set(re.findall(r"\b(gs_[a-z_0-9]+)\s*\(", text)))


def test_exports_match_header(lib):
    from paper_2607_01164_b200 import api
    names = _declared()
    assert {"gs_preprocess", "gs_build_accel", "gs_sample_fwd", "gs_sample_bwd"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in gs.h but not exported"
    assert set(api.EXPORTS) == set(names)


def _prototypes():
    """{name: [C type of each parameter]} of every function include/gs.h declares."""
    text = open(os.path.join(ROOT, "include", "gs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    out = {}
    for m in re.finditer(r"\b(gs_[a-z_0-9]+)\s*\(([^()]*)\)\s*;", text):
        params = [p.strip() for p in m.group(2).split(",")]
        out[m.group(1)] = [] if params == ["void"] else [re.sub(r"\s*\w+$", "", p).strip() if not p.endswith("*") else p for p in params]
    return out


def _kind(ctype):
    """Coarse class of a C parameter type / a ctypes type: pointers are one class, scalars must match exactly."""
    if isinstance(ctype, str):
        if "*" in ctype:
            return "ptr"
        return {"int": "i32", "int32_t": "i32", "uint32_t": "u32", "int64_t": "i64", "uint64_t": "u64", "size_t": "u64", "float": "f32"}[ctype]   # LP64: size_t is 64 bits
    if ctype in (ctypes.c_void_p, ctypes.c_char_p) or hasattr(ctype, "contents"):
        return "ptr"
    return {ctypes.c_int: "i32", ctypes.c_int32: "i32", ctypes.c_uint32: "u32", ctypes.c_int64: "i64", ctypes.c_uint64: "u64",
            ctypes.c_size_t: "u64", ctypes.c_float: "f32"}[ctype]


def test_binding_argtypes_match_header_prototypes(lib):
    # an exported symbol carries no prototype: the binding (and any caller built against an older header) only stays in
    # step with the library if every parameter list is checked against the header
    protos = _prototypes()
    assert set(protos) == set(_declared())
    for name, params in protos.items():
        argtypes = getattr(lib, name).argtypes
        assert argtypes is not None, f"{name}: the binding declares no argtypes"
        assert [_kind(a) for a in argtypes] == [_kind(p) for p in params], f"{name}: binding {argtypes} vs header {params}"
    # the round-1 prototype of gs_measure_alu_peaks (three arguments) is frozen; the packed-FMA figure lives in ...peaks2
    assert len(protos["gs_measure_alu_peaks"]) == 3 and len(protos["gs_measure_alu_peaks2"]) == 4


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
