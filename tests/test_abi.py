"""The C-ABI boundary without a GPU: libecpush.so builds, loads, exports every symbol that
include/ecpush.h declares, and its host-side argument checks answer with status codes instead of
crashing.  No compute call is made here."""
from __future__ import annotations

import ctypes
import os

import pytest

import paper_2603_16624_b200 as pk
from paper_2603_16624_b200 import binding, build


@pytest.fixture(scope="module")
def L():
    build.build()
    return pk.lib()


def test_library_is_in_tree():
    path = build.build()
    assert os.path.dirname(path) == os.path.dirname(os.path.abspath(pk.__file__))


def test_every_declared_symbol_is_exported_and_bound(L):
    names = pk.declared_symbols()
    for required in ("ecsim_init_grid", "ecsim_load_particles", "ecsim_push_and_moments", "ecsim_sort_particles"):
        assert required in names            # the calls BASELINE.json's north_star lists
    raw = ctypes.CDLL(pk.lib_path())
    for n in names:
        assert hasattr(raw, n), f"{n} declared in ecpush.h but not exported"
        assert n in binding._PROTOS, f"{n} has no Python prototype"
    assert set(binding._PROTOS) == set(names)


def test_strerror_and_status_codes(L):
    assert L.ecsim_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5, -6):
        assert len(L.ecsim_strerror(code)) > 0
    assert L.ecsim_strerror(-99) == b"unknown status"


def test_init_grid_rejects_bad_arguments(L):
    h = ctypes.c_void_p()
    assert L.ecsim_init_grid(None, 4, 4, 4, 1.0, 1.0, 1.0, 1, None) == -1
    assert L.ecsim_init_grid(ctypes.byref(h), 1, 4, 4, 1.0, 1.0, 1.0, 1, None) == -1     # dims >= 2
    assert L.ecsim_init_grid(ctypes.byref(h), 4, 4, 4, 0.0, 1.0, 1.0, 1, None) == -1     # spacing > 0
    assert L.ecsim_init_grid(ctypes.byref(h), 4, 4, 4, 1.0, 1.0, 1.0, 0, None) == -1     # species >= 1
    assert L.ecsim_init_grid(ctypes.byref(h), 4096, 4096, 4096, 1.0, 1.0, 1.0, 1, None) == -1
    assert not h.value


def test_null_context_is_an_error_not_a_crash(L):
    assert L.ecsim_set_workspace(None, None, 0) == -1
    assert L.ecsim_workspace_bytes(None, 10) == 0
    assert L.ecsim_push_and_moments(None, 0, None, None, 0.1, 0.5, None, None, None, 0) == -1
    assert L.ecsim_push_and_moments_all(None, None, None, 0.1, 0.5, None, None, None, 0) == -1
    assert L.ecsim_sort_particles(None, 0, None, None) == -1
    assert L.ecsim_build_segments(None, 0) == -1
    assert L.ecsim_cell_index(None, 0, None) == -1
    assert L.ecsim_set_variant(None, 0) == -1
    assert L.ecsim_enable_timing(None, 1) == -1
    assert L.ecsim_launch_count(None) == 0
    assert L.ecsim_moments(None, 0, None, 0.1, None, None, None, 0) == -1
    assert L.ecsim_moments_all(None, None, 0.1, None, None, None, 0) == -1
    assert L.ecsim_push(None, 0, None, None, 0.1, 0.5) == -1
    assert L.ecsim_push_all(None, None, None, 0.1, 0.5) == -1
    assert L.ecsim_make_resident(None, 0, None, 0, 0.25) == -1
    assert L.ecsim_export_particles(None, 0, None, None, None, None, None, None, None) == -1
    assert L.ecsim_resident_bytes(None, 10, 0.25) == 0
    assert L.ecsim_apply_M(None, None, None, None, 0) == -1
    assert L.ecsim_set_m_layout(None, 0) == -1
    assert L.ecsim_relayout_count(None) == 0
    assert L.ecsim_set_overflow_capacity(None, 0, 10) == -1
    assert L.ecsim_validate_particles(None, 0) == -1
    assert L.ecsim_destroy(None) == 0


def test_no_cpu_fallback_without_a_device(L):
    """On a box without a GPU the product path must fail loudly (ECSIM_ERR_CUDA), never compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = ctypes.c_void_p()
    rc = L.ecsim_init_grid(ctypes.byref(h), 8, 8, 8, 1.0, 1.0, 1.0, 2, None)
    assert rc == -4 and not h.value
    assert b"cuda" in L.ecsim_last_error().lower()
    with pytest.raises(pk.EcsimError):
        pk.Ecsim(8, 8, 8, 1.0, 1.0, 1.0, 2)


def test_product_does_not_import_the_oracle():
    """Neither side imports the other (the oracle is test infrastructure)."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for dirpath, _, files in os.walk(os.path.join(root, "paper_2603_16624_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "ecsim_oracle" not in text and "liboracle" not in text, f
    for f in os.listdir(os.path.join(root, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(root, "oracle", f)).read()
            assert "import paper_2603_16624_b200" not in text and "libecpush" not in text
            assert "from paper_2603_16624_b200" not in text
