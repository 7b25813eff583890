"""CPU-side checks of the boundary: libwl.so builds, loads, exports every symbol include/wl.h
declares, and the host-only logic (field creation, argument validation, workspace plan) behaves
as the header says.  No kernel is launched here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "wl.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1407_7486_b200 import build
    return C.CDLL(build.build())


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(wl_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_calls_of_survey_8b():
    names = declared_symbols()
    for want in ("wl_field_create", "wl_field_destroy", "wl_loops_generate", "wl_eval_workspace_bytes",
                 "wl_eval", "wl_jackknife_finalize", "wl_status_string", "wl_eval_host", "wl_eval_per_loop"):
        assert want in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_every_declared_call_cites_the_paper():
    src = open(HEADER).read()
    assert src.count("PAPER.md:") >= 10


def test_field_create_validation(lib):
    lib.wl_field_create.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_void_p)]
    lib.wl_field_destroy.argtypes = [C.c_void_p]

    def create(profile, params):
        arr = (C.c_double * max(len(params), 1))(*params)
        h = C.c_void_p()
        st = lib.wl_field_create(profile, arr, len(params), C.byref(h))
        return st, h

    st, h = create(0, [1.0])
    assert st == 0 and h.value
    lib.wl_field_destroy(h)
    st, h = create(1, [1.0, 0.5])
    assert st == 0 and h.value
    lib.wl_field_destroy(h)
    st, h = create(2, [10.0, 1.0])                                   # flux tube, eq. (68)
    assert st == 0 and h.value
    lib.wl_field_destroy(h)
    lib.wl_field_create_particle.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_int, C.c_int, C.POINTER(C.c_void_p)]
    arr, h = (C.c_double * 2)(1.0, 1.0), C.c_void_p()
    assert lib.wl_field_create_particle(1, arr, 2, 1, C.byref(h)) == 0 and h.value          # scalar loop
    lib.wl_field_destroy(h)
    assert lib.wl_field_create_particle(1, arr, 2, 2, C.byref(h)) == 1 and not h.value      # unknown particle
    for profile, params in ((0, [1.0, 2.0]), (1, [1.0]), (1, [1.0, 0.0]), (1, [1.0, -1.0]), (2, [1.0]), (2, [1.0, 0.0]),
                            (1, [float("nan"), 1.0]), (0, [float("inf")]), (7, [1.0])):
        st, h = create(profile, params)
        assert st == 1 and not h.value
    lib.wl_field_destroy(None)


def test_status_strings(lib):
    lib.wl_status_string.restype = C.c_char_p
    seen = {lib.wl_status_string(i) for i in range(5)}
    assert len(seen) == 5 and all(seen)
    assert lib.wl_status_string(99)


def test_workspace_plan_is_a_function_of_sizes_only(lib):
    f = lib.wl_eval_workspace_bytes
    f.restype = C.c_size_t
    f.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
    # config 3: 16384 loops, 64x64 grid, G = 64: units of 4 loops -> 4096 x 4096 doubles
    assert f(16384, 2048, 64, 64, 64, 0) == 4096 * 4096 * 8
    # a partial is never coarser than a group and never finer than a loop
    for (nl, g, nt, nr) in ((1024, 16, 16, 16), (4096, 32, 32, 8), (65536, 256, 64, 64), (12, 4, 3, 5), (7, 7, 1, 1)):
        b = f(nl, 64, nt, nr, g, 1)
        units = b // (8 * nt * nr)
        assert b % (8 * nt * nr) == 0 and g <= units <= nl and units % g == 0
    # invalid sizes -> 0
    assert f(10, 64, 4, 4, 3, 0) == 0          # 10 % 3 != 0 (equal groups)
    assert f(0, 64, 4, 4, 1, 0) == 0
    assert f(8, 64, 0, 4, 1, 0) == 0
    assert f(8, 64, 4, 4, 1, 5) == 0


def test_compute_calls_reject_bad_arguments_without_a_gpu(lib):
    lib.wl_eval.restype = C.c_int
    vp = C.c_void_p
    lib.wl_eval.argtypes = [vp, vp, C.c_int, C.c_int64, C.c_int, vp, C.c_int, vp, vp, C.c_int, C.c_int, C.c_int,
                            vp, vp, vp, C.c_size_t, vp]
    assert lib.wl_eval(None, None, 0, 1, 1, None, 1, None, None, 1, 1, 0, None, None, None, 0, None) == 1
    lib.wl_loops_generate.restype = C.c_int
    lib.wl_loops_generate.argtypes = [vp, C.c_int, C.c_int64, C.c_int64, C.c_int, C.c_uint64, vp]
    dummy = C.c_void_p(16)
    assert lib.wl_loops_generate(dummy, 1, 0, 4, 100, 1, None) == 1      # not a power of two
    assert lib.wl_loops_generate(dummy, 1, 0, 4, 131072, 1, None) == 1   # above the generator limit (65536)
    assert lib.wl_loops_generate(dummy, 1, 0, -1, 64, 1, None) == 1
    assert lib.wl_loops_generate(dummy, 1, 0, 0, 64, 1, None) == 0       # empty: no-op
    lib.wl_jackknife_finalize.restype = C.c_int
    lib.wl_jackknife_finalize.argtypes = [vp, C.c_int, C.c_int64, C.c_int, C.c_int, vp, vp, vp, vp]
    assert lib.wl_jackknife_finalize(dummy, 1, 8, 2, 2, dummy, dummy, None, None) == 1   # G < 2
    assert lib.wl_jackknife_finalize(dummy, 3, 8, 2, 2, dummy, dummy, None, None) == 1   # 8 % 3


def test_proper_time_nodes_host_call(lib):
    """wl_proper_time_nodes is host-only: x = 1/(1 + T/Tmax) is uniform on (0, x_a]."""
    lib.wl_proper_time_nodes.restype = C.c_int
    lib.wl_proper_time_nodes.argtypes = [C.c_double, C.c_double, C.c_int, C.POINTER(C.c_double)]
    n, a, Tmax = 12, 0.05, 3.0
    T = (C.c_double * n)()
    assert lib.wl_proper_time_nodes(a, Tmax, n, T) == 0
    x = [1.0 / (1.0 + t / Tmax) for t in T]
    xa = 1.0 / (1.0 + a / Tmax)
    assert T[0] == a and all(abs(x[j] - xa * (n - j) / n) < 1e-15 for j in range(n))
    assert lib.wl_proper_time_nodes(a, Tmax, 7, T) == 1 and lib.wl_proper_time_nodes(0.0, Tmax, 8, T) == 1
    assert lib.wl_proper_time_nodes(a, Tmax, 8, None) == 1
