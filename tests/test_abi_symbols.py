"""CPU-side checks of the C-ABI boundary (no compute calls: there is no GPU here).

The library builds with nvcc (cross-compiled for sm_100a), loads, exports every function include/m3dk.h declares, its
pure host entry points (workspace sizes, argument validation) behave, and without a CUDA device it fails loudly instead
of falling back to anything."""
import ctypes as C

import pytest

import paper_2107_13663_b200 as m3dk


@pytest.fixture(scope="module")
def libs():
    m3dk.build_all()
    return [m3dk.lib(False), m3dk.lib(True)]


def test_every_declared_symbol_is_exported(libs):
    names = m3dk.exported_symbols()
    assert {"m3dk_fields_create", "m3dk_particles_init", "m3dk_push", "m3dk_sort"} <= set(names)
    assert len(names) >= 19
    for L in libs:
        for n in names:
            assert getattr(L, n) is not None
        assert L.m3dk_version() >= 100


def test_workspace_queries_are_pure_host_functions(libs):
    L = libs[0]
    b = C.c_size_t()
    assert L.m3dk_fields_workspace_bytes(1089, 2048, 1, C.byref(b)) == 0
    one = b.value
    assert one % 256 == 0 and one > 2048 * 432 * 8           # the tiles alone: 432 doubles per element with one mode
    assert L.m3dk_fields_workspace_bytes(1089, 2048, 0, C.byref(b)) == 0 and b.value < one
    assert L.m3dk_fields_workspace_bytes(1089, 2048, 5, C.byref(b)) == -1      # more than M3DK_MAX_MODES
    assert L.m3dk_fields_workspace_bytes(2, 2048, 1, C.byref(b)) == -1         # fewer than 3 nodes
    assert L.m3dk_fields_workspace_bytes(1089, 2048, 1, None) == -1
    s = C.c_size_t()
    assert L.m3dk_sort_workspace_bytes(0, 2048, C.byref(s)) == 0 and s.value % 256 == 0
    small = s.value
    assert L.m3dk_sort_workspace_bytes(1 << 20, 2048, C.byref(s)) == 0
    assert s.value >= small + (1 << 20) * (2 * 64 + 2 * 8 + 2 * 4)            # two record buffers, two order lists, key, rank
    assert L.m3dk_sort_workspace_bytes(-1, 2048, C.byref(s)) == -1


def test_null_context_is_rejected_not_dereferenced(libs):
    L = libs[0]
    assert L.m3dk_push(None, 1, 0.1) == -1
    assert L.m3dk_sort(None, None, 0) == -1
    assert L.m3dk_destroy(None) == -1
    assert L.m3dk_set_options(None, 0, 0, 0.0) == -1


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(m3dk.M3DKError):
        m3dk.Pusher(device=0)
    L = m3dk.lib(False)
    h = C.c_void_p()
    rc = L.m3dk_create(C.byref(h), 0, None)
    assert rc == -4 and not h.value                       # M3DK_ECUDA, no context
    assert b"cuda" in L.m3dk_last_error(None).lower()
