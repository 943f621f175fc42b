"""CPU-side checks of the C-ABI boundary: the library builds, loads without a GPU and exports
every symbol include/polargrav.h declares; host-only argument validation works; the binding has
the same names.  No compute calls here (those are the -m gpu tests)."""
import ctypes
import os
import re

import pytest

from paper_2409_02294_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "polargrav.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pg3?n?_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for must in ("pg_create", "pg_set_density", "pg_potential", "pg_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    raw = ctypes.CDLL(binding.LIB_PATH)
    for name in declared_functions():
        assert hasattr(raw, name), f"{name} declared in polargrav.h but not exported"


def test_binding_has_the_same_names(lib):
    names = declared_functions()
    assert sorted(binding.EXPORTS) == names
    for name in names:
        if name in ("pg_status_string", "pg_last_error", "pg_version"):
            continue
        assert callable(getattr(binding, name)), name


def test_status_strings_and_version(lib):
    assert binding.status_string(0) == "PG_OK"
    assert binding.status_string(-2) == "PG_ERR_UNSUPPORTED"
    assert binding.status_string(-5) == "PG_ERR_STATE"
    assert "sm_100a" in binding.version()


def test_argument_validation_needs_no_gpu(lib):
    # these fail in host-side checks before any CUDA call
    with pytest.raises(binding.PolargravError) as e:
        binding.pg_create(64, 64, 1.0, 0.5, 0.01)           # r_out <= r_in
    assert e.value.status == binding.PG_ERR_INVALID_ARG
    with pytest.raises(binding.PolargravError) as e:
        binding.pg_create(64, 64, 1.0, 100.0, 0.0)          # eps <= 0
    assert e.value.status == binding.PG_ERR_INVALID_ARG
    with pytest.raises(binding.PolargravError) as e:
        binding.pg_create(96, 64, 1.0, 100.0, 0.01)         # not a power of two
    assert e.value.status == binding.PG_ERR_UNSUPPORTED
    with pytest.raises(binding.PolargravError) as e:
        binding.pg_create(4096, 64, 1.0, 100.0, 0.01)       # above PG_MAX_N
    assert e.value.status == binding.PG_ERR_UNSUPPORTED
    assert binding.lib().pg_destroy(None) == binding.PG_OK   # no-op
    assert binding.lib().pg_set_density(None, None, 1, 0) == binding.PG_ERR_INVALID_ARG
    # the 3-D mesh calls (NEXT-2)
    with pytest.raises(binding.PolargravError) as e:
        binding.pg3_create(48, 1.0)                          # not a supported mesh size
    assert e.value.status == binding.PG_ERR_UNSUPPORTED
    with pytest.raises(binding.PolargravError) as e:
        binding.pg3_create(64, 0.0)                          # box <= 0
    assert e.value.status == binding.PG_ERR_INVALID_ARG
    assert binding.lib().pg3_destroy(None) == binding.PG_OK
    assert binding.lib().pg3_set_density(None, None, 0) == binding.PG_ERR_INVALID_ARG


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.PolargravError) as e:
        binding.pg_create(64, 64, 1.0, 100.0, 0.01)
    assert e.value.status in (binding.PG_ERR_CUDA, binding.PG_ERR_UNSUPPORTED)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2409_02294_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "polar_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2409_02294_b200" not in text and "from paper_2409_02294_b200" not in text, f
            assert "polargrav.h" not in text and "libpolargrav" not in text, f
