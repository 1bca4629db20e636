"""Boundary checks that need no GPU: the C-ABI library loads, exports every symbol include/cobalt.h
declares, and validates its arguments / reports a missing device instead of falling back to a CPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "cobalt.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cobalt_[a-z0-9_]+)\s*\(", text)))


def test_header_and_binding_agree(cobalt):
    assert declared_symbols() == sorted(cobalt.ABI_SYMBOLS)


def test_library_exports_every_declared_symbol(cobalt):
    lib = ctypes.CDLL(cobalt.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_strerror_and_null_destroy(cobalt):
    lib = cobalt.load()
    assert lib.cobalt_strerror(0) == b"ok"
    assert lib.cobalt_strerror(cobalt.COBALT_ERR_BAD_ARG) == b"bad argument"
    assert lib.cobalt_destroy(None) == cobalt.COBALT_OK


@pytest.mark.parametrize("args", [
    (0, 1, 64, 16, 6400, 16),      # stations < 1
    (4, 0, 64, 16, 6400, 16),      # subbands < 1
    (4, 1, 32, 16, 6400, 16),      # channels not in {16, 64, 256}
    (4, 1, 64, 8, 6400, 16),       # taps != 16
    (4, 1, 64, 16, 63, 16),        # N < C
    (4, 1, 64, 16, 6400, 12),      # input_bits not in {4, 8, 16}
])
def test_plan_rejects_bad_arguments(cobalt, args):
    h = ctypes.c_void_p(1234)
    rc = cobalt.load().cobalt_plan(ctypes.byref(h), *args)
    assert rc == cobalt.COBALT_ERR_BAD_ARG
    assert h.value is None                      # *out = NULL on failure
    assert cobalt.load().cobalt_last_error(None)


def test_plan_null_out(cobalt):
    assert cobalt.load().cobalt_plan(None, 4, 1, 64, 16, 6400, 16) == cobalt.COBALT_ERR_BAD_ARG


def test_no_device_is_an_error_not_a_fallback(cobalt):
    """On a box without a GPU a valid plan request must fail loudly (there is no CPU path)."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(cobalt.CobaltError) as e:
        cobalt.cobalt_plan(4, 1, 16, 16, 4096, 16)
    assert e.value.status in (cobalt.COBALT_ERR_UNSUPPORTED_DEVICE, cobalt.COBALT_ERR_CUDA)


def test_null_plan_calls(cobalt):
    lib = cobalt.load()
    assert lib.cobalt_process(None, None, None, None, None, None) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_process_host(None, None, None, None, None) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_process_ex(None, None, None) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_set_dumps(None, 2) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_set_phase_offsets(None, None) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_set_coarse_delays(None, None, 0) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_set_input_layout(None, 1) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_reset(None) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_info(None, None) == cobalt.COBALT_ERR_BAD_ARG
    assert lib.cobalt_debug_unpack(None, 12, None, 0, None) == cobalt.COBALT_ERR_BAD_ARG


def test_product_does_not_import_the_oracle():
    """The package and its CUDA sources never reference oracle/ (parity would be void otherwise)."""
    pkg = os.path.join(ROOT, "paper_1801_04834_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "cobalt_oracle" not in text, f
