"""The C-ABI library loads on a machine without a GPU and exports every symbol that
include/nearfield.h declares; argument errors are reported, never raised from C."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2110_11392_b200.build import build_library
    build_library()
    import paper_2110_11392_b200.binding as b
    return b


def _declared_symbols():
    with open(os.path.join(ROOT, "include", "nearfield.h")) as f:
        text = f.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nf_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    syms = _declared_symbols()
    assert "nf_create" in syms and "nf_accel" in syms and "nf_destroy" in syms
    raw = ctypes.CDLL(lib.lib_path())
    for s in syms:
        assert hasattr(raw, s), f"{s} declared in include/nearfield.h but not exported"
    assert sorted(lib.SYMBOLS) == syms, "binding.SYMBOLS out of date with the header"


def test_no_torch_types_in_header():
    with open(os.path.join(ROOT, "include", "nearfield.h")) as f:
        text = f.read()
    assert "torch" not in text.lower().replace("pytorch tensors", "") or "at::" not in text
    assert "at::Tensor" not in text and "#include <torch" not in text


def test_create_argument_errors(lib):
    L = lib._L
    h = ctypes.c_void_p()
    assert L.nf_create(None, 7, 2, 0.01, 1.0) == lib.NF_EINVAL
    for args in [(4, 2, 0.01, 1.0), (7, 0, 0.01, 1.0), (7, 5, 0.01, 1.0), (7, 2, 0.0, 1.0), (7, 2, -1.0, 1.0),
                 (7, 2, 0.01, 0.0), (7, 2, float("nan"), 1.0), (7, 2, 0.01, float("inf")), (1300, 2, 0.01, 1.0)]:
        assert L.nf_create(ctypes.byref(h), *args) == lib.NF_EINVAL, args
        assert not h.value
        assert b"bad argument" in L.nf_last_error(None)


def test_null_context_calls(lib):
    L = lib._L
    assert L.nf_destroy(None) == lib.NF_OK
    assert L.nf_accel(None, None, 0, None, None) == lib.NF_EINVAL
    assert L.nf_sync(None) == lib.NF_EINVAL
    assert L.nf_set_gm(None, 1.0) == lib.NF_EINVAL
    assert isinstance(L.nf_last_error(None), bytes)


def test_product_has_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(lib.NearFieldError) as e:
        lib.NearField(7, 2, 0.01)
    assert e.value.status == lib.NF_ECUDA and "no CPU fallback" in str(e.value)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2110_11392_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, fn)) as f:
                    t = f.read()
                assert "import oracle" not in t and "from oracle" not in t and "nf_oracle" not in t, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            with open(os.path.join(ROOT, "oracle", fn)) as f:
                t = f.read()
            assert "import paper_2110_11392_b200" not in t and "from paper_2110_11392_b200" not in t and "nearfield.h" not in t, fn


def test_bench_only_helper_library_is_built_and_separate():
    """libnf_pipeprobe.so (bench-only pipe-rate microbenchmarks, source outside csrc/) is built by build() beside the
    product library, exports its one entry point, and exports none of the product's nf_* symbols (and vice versa);
    editing it does not change the product library's source hash."""
    import ctypes
    from paper_2110_11392_b200 import build
    build.ensure_built()
    probe = ctypes.CDLL(build.PROBE_LIB)
    prod = ctypes.CDLL(build.LIB)
    assert hasattr(probe, "nfp_probe_pipes")
    assert not hasattr(probe, "nf_accel") and not hasattr(probe, "nf_create")
    assert not hasattr(prod, "nfp_probe_pipes")
    assert not any(os.path.abspath(d) == os.path.abspath(build.PROBE_SRC) for d in build._deps())
