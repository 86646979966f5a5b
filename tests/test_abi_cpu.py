"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/dsk.h declares, and
its host-only logic (argument validation, workspace sizing, constants, the fp64 lattice tensors of the
periodic far field) is right.  No compute call is made (there is no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1407_2600_b200 import build, dsk
    build.build()
    return dsk.load_library()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "dsk.h")).read()
    declared = set(re.findall(r"\b(dsk_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 18
    from paper_1407_2600_b200 import dsk
    assert declared == set(dsk.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_constants_match_oracle_conventions(lib, orc):
    from paper_1407_2600_b200 import dsk
    assert dsk.get_param("NLEAF") == orc.NLEAF and dsk.get_param("NCRIT") == orc.NCRIT
    assert dsk.get_param("WS") == orc.WS and dsk.get_param("KEY_LEVELS") == orc.KEY_LEVELS
    assert dsk.get_param("FAR_ORDER") == orc.FAR_ORDER
    with pytest.raises(dsk.DskError):
        dsk.get_param("NOPE")


def test_task_widths_cover_every_group_size(lib):
    """Host logic of the force kernels' task split: for every group size the widths tile the sink
    lanes exactly, respect the warp width, and no split of <= 4 parts is cheaper under the stated cost model."""
    import functools
    from paper_1407_2600_b200 import dsk
    ncrit = int(dsk.get_param("NCRIT"))

    def cost(w):                                       # 1/S + c in units of 1/960, S = sub-groups of a w-lane task
        return 960 // (32 // w) + 40

    @functools.lru_cache(None)
    def best(lanes, k):
        if lanes == 0:
            return 0
        if k == 0:
            return 10 ** 9
        return min(cost(w) + best(lanes - w, k - 1) for w in range(1, min(32, lanes) + 1))

    for n in range(1, ncrit + 1):
        w = dsk.get_task_widths(n)
        lanes = (n + 1) // 2
        assert 1 <= len(w) <= 4 and all(1 <= x <= 32 for x in w), (n, w)
        assert sum(w) == lanes, (n, w)
        assert sum(cost(x) for x in w) == best(lanes, 4), (n, w)
    # the examples DESIGN.md quotes
    assert sorted(dsk.get_task_widths(65)) == [1, 32] and sorted(dsk.get_task_widths(37)) == [3, 16]
    for bad in (0, -1, ncrit + 1):
        with pytest.raises(dsk.DskError):
            dsk.get_task_widths(bad)


def test_create_validation_and_workspace(lib):
    h = C.c_void_p(0)
    bad = [(0, 1.0, 0, 1e-3, 0.5, 4), (10, -1.0, 0, 1e-3, 0.5, 4), (10, 1.0, 0, 0.0, 0.5, 4),
           (10, 1.0, 0, 1e-3, 0.0, 4), (10, 1.0, 0, 1e-3, 1.5, 4), (10, 1.0, 0, 1e-3, 0.5, 7), (10, 1.0, 0, 1e-3, 0.5, 1),
           (10, 1.0, 0, 1e-3, 0.5, 10)]
    for a in bad:
        assert lib.dsk_create(C.byref(h), *a) == -1
    assert lib.dsk_create(C.byref(h), 1 << 20, 1.0, 0, 1e-4, 0.5, 4) == 0
    b1 = lib.dsk_workspace_bytes(h)
    assert 200e6 < b1 < 4e9                     # ~2 kB per particle
    # calls that need a workspace / tree fail cleanly without touching the device
    assert lib.dsk_build_tree(h, C.c_void_p(256), C.c_void_p(256)) == -2
    assert lib.dsk_accel(h, C.c_void_p(256), C.c_void_p(256), C.c_void_p(256), None) == -2
    assert lib.dsk_bind_workspace(h, C.c_void_p(0), b1) == -2
    assert lib.dsk_bind_workspace(h, C.c_void_p(257), b1) == -2
    # p may be lowered but not raised above dsk_create's p (the workspace is sized for it)
    assert lib.dsk_set_params(h, 1e-4, 0.3, 2) == 0 and lib.dsk_set_params(h, 1e-4, 0.3, 3) == 0 and lib.dsk_set_params(h, 1e-4, 0.3, 7) == -1
    assert lib.dsk_set_params(h, 1e-4, 0.3, 8) == -2
    # switches validate their argument without touching the device
    lib.dsk_set_walk_sharing.argtypes = [C.c_void_p, C.c_int]
    assert lib.dsk_set_walk_sharing(h, 8) == 0 and lib.dsk_set_walk_sharing(h, 0) == 0
    assert lib.dsk_set_walk_sharing(h, 9) == -1 and lib.dsk_set_walk_sharing(h, -1) == -1
    assert lib.dsk_set_background(h, 1) == -1                    # isolated context
    assert lib.dsk_destroy(h) == 0
    assert lib.dsk_strerror(-4).decode().startswith("position outside")
    assert "maximum" in lib.dsk_strerror(-9).decode()
    # the no-allocation entry point rejects sizes beyond its fixed scratch before any device work
    lib.dsk_sort_keys_noalloc.argtypes = [C.c_void_p, C.c_int64, C.c_float, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    assert lib.dsk_sort_keys_noalloc(C.c_void_p(256), (1 << 20) + 1, 1.0, 0, C.c_void_p(256), C.c_void_p(256), None) == -9
    assert lib.dsk_sort_keys_noalloc(C.c_void_p(256), 0, 1.0, 0, C.c_void_p(256), C.c_void_p(256), None) == -1
    assert lib.dsk_sort_keys_noalloc(None, 10, 1.0, 0, C.c_void_p(256), C.c_void_p(256), None) == -1
    h2 = C.c_void_p(0)
    assert lib.dsk_create(C.byref(h2), 1 << 21, 1.0, 0, 1e-4, 0.5, 4) == 0
    assert 1.8 < lib.dsk_workspace_bytes(h2) / b1 < 2.2
    lib.dsk_destroy(h2)


def test_lattice_tensors_match_oracle(lib, orc):
    """the library's own fp64 host computation of T_n (farfield.cu) against the pinned oracle"""
    for box in (1.0, 2.0):
        h = C.c_void_p(0)
        assert lib.dsk_create(C.byref(h), 100, box, 1, 1e-3, 0.5, 4) == 0
        T = np.empty(165)
        assert lib.dsk_get_lattice_tensors(h, T.ctypes.data_as(C.c_void_p)) == 0
        ref = orc.farfield_T(box, orc.WS, 8)
        assert np.max(np.abs(T - ref)) < 1e-10 * max(1.0, np.abs(ref).max())
        lib.dsk_destroy(h)
    h = C.c_void_p(0)
    lib.dsk_create(C.byref(h), 100, 1.0, 0, 1e-3, 0.5, 4)
    assert lib.dsk_get_lattice_tensors(h, T.ctypes.data_as(C.c_void_p)) == -1     # isolated: none
    lib.dsk_destroy(h)


def test_sort_threshold_is_the_same_on_both_sides_of_the_accounting():
    """bench.py's algorithmic bytes of the sort (accounting.sort_bytes) switch where the library switches its sort form"""
    import re
    from paper_1407_2600_b200 import accounting
    src = open(os.path.join(os.path.dirname(__file__), "..", "paper_1407_2600_b200", "csrc", "dsk_internal.cuh")).read()
    m = re.search(r"#define DSK_SORT_ONESWEEP_NMAX \(1 << (\d+)\)", src)
    assert m and (1 << int(m.group(1))) == accounting.SORT_ONESWEEP_NMAX
    assert accounting.sort_bytes(1 << 20) == 200 and accounting.sort_bytes(1 << 24) == 256
