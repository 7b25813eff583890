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


HOUSEKEEPING = {"wl_field_destroy", "wl_eval_options_default", "wl_eval_host_trim", "wl_eval_launch_count", "wl_version"}


def test_every_declared_call_cites_the_paper():
    """Each prototype's own comment (the block comment that precedes it) names the passage that defines the
    operation: a PAPER.md line, or the DESIGN.md reading / SURVEY.md section that stands for it.  Calls that
    compute nothing of the method (HOUSEKEEPING) are exempt."""
    src = open(HEADER).read()
    comment, uncited, seen = None, [], set()
    for m in re.finditer(r"/\*.*?\*/|\b(wl_[a-z_0-9]+)\s*\(", src, flags=re.S):
        if m.group(0).startswith("/*"):
            line_start = src.rfind("\n", 0, m.start()) + 1
            if src[line_start:m.start()].strip() == "":           # a block comment of its own, not a trailing remark
                comment = m.group(0)
            continue
        name = m.group(1)
        seen.add(name)
        if name in HOUSEKEEPING:
            continue
        if not (comment and ("PAPER.md:" in comment or "DESIGN.md" in comment or "SURVEY.md" in comment)):
            uncited.append(name)
    assert not uncited, uncited
    assert seen == set(declared_symbols())


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
    seen = {lib.wl_status_string(i) for i in range(7)}
    assert len(seen) == 7 and all(seen)
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
    # the CTA bound follows the real launch shape: 2^24 loops on a 128 x 128 grid are 2^21 units x 16 tiles = 2^25 CTAs
    assert f(1 << 24, 64, 128, 128, 16, 0) == (1 << 21) * 128 * 128 * 8
    # ... and what no kernel shape can launch is refused: 2^40 loops x 4 tiles of 1024 points, in units of 8
    assert f(1 << 40, 64, 64, 64, 16, 0) == 0


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


class _Options(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("quadrature_order", C.c_int), ("seeded", C.c_int),
                ("seed", C.c_uint64), ("loop_begin", C.c_int64), ("shuffle_groups", C.c_int), ("staging", C.c_int),
                ("shuffle_seed", C.c_uint64), ("ensemble_loops", C.c_int64), ("event_wilson_begin", C.c_void_p),
                ("event_wilson_end", C.c_void_p)]


def test_options_block_and_its_workspace_sizes(lib):
    """struct wl_eval_options (NEXT-4 options): defaults, validation and the workspace each option needs -- host only."""
    o = _Options()
    lib.wl_eval_options_default.restype = None
    lib.wl_eval_options_default(C.byref(o))
    assert o.struct_size == C.sizeof(_Options) and o.quadrature_order == 1
    assert (o.seeded, o.shuffle_groups, o.staging, o.ensemble_loops) == (0, 0, 0, 0)
    lib.wl_eval_options_default(None)                                  # NULL is ignored
    f = lib.wl_eval_opt_workspace_bytes
    f.restype = C.c_size_t
    f.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(_Options)]
    base = f(16384, 2048, 64, 64, 64, 0, None)
    assert base == f(16384, 2048, 64, 64, 64, 0, C.byref(o)) == 4096 * 4096 * 8
    o.quadrature_order = 3
    assert f(16384, 2048, 64, 64, 64, 0, C.byref(o)) == base           # the order needs no workspace
    o.quadrature_order = 4
    assert f(16384, 2048, 64, 64, 64, 0, C.byref(o)) == 0
    o.quadrature_order = 1
    o.shuffle_groups = 1                                               # W per loop + the membership table
    assert f(16384, 2048, 64, 64, 64, 0, C.byref(o)) == 16384 * 4096 * 8 + 64 * 16384 * 4
    o.shuffle_groups = 0
    o.seeded = 1
    assert f(16384, 2048, 64, 64, 64, 0, C.byref(o)) == base
    assert f(16384, 2000, 64, 64, 64, 0, C.byref(o)) == 0              # seeded: N must be a power of two
    assert f(16384, 131072, 4, 4, 64, 0, C.byref(o)) == 0              # ... of at most 65536
    o.seeded = 0
    o.ensemble_loops = 8 * 16384                                       # a shard of a 131072-loop ensemble: units of 8 loops
    assert f(16384, 2048, 64, 64, 64, 0, C.byref(o)) == 2048 * 4096 * 8
    o.ensemble_loops = 100                                             # smaller than the shard
    assert f(16384, 2048, 64, 64, 64, 0, C.byref(o)) == 0
    o.ensemble_loops = 0
    o.struct_size = 8                                                  # another ABI generation
    assert f(16384, 2048, 64, 64, 64, 0, C.byref(o)) == 0


def test_grid_validate_and_permutation_argument_checks(lib):
    dp = C.POINTER(C.c_double)
    lib.wl_grid_validate.restype = C.c_int
    lib.wl_grid_validate.argtypes = [dp, C.c_int, dp, C.c_int]
    T = (C.c_double * 3)(0.01, 1.0, 10.0)
    rho = (C.c_double * 2)(0.0, 4.0)
    assert lib.wl_grid_validate(T, 3, rho, 2) == 0
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        Tb = (C.c_double * 3)(0.01, bad, 10.0)
        assert lib.wl_grid_validate(Tb, 3, rho, 2) == 1
    assert lib.wl_grid_validate(T, 3, (C.c_double * 2)(0.0, -1e-12), 2) == 1
    assert lib.wl_grid_validate(None, 3, rho, 2) == 1 and lib.wl_grid_validate(T, 0, rho, 2) == 1
    lib.wl_group_permutation.restype = C.c_int
    lib.wl_group_permutation.argtypes = [C.c_uint64, C.c_int64, C.c_int, C.c_void_p, C.c_void_p]
    dummy = C.c_void_p(16)
    assert lib.wl_group_permutation(1, 0, 4, dummy, None) == 1
    assert lib.wl_group_permutation(1, 1 << 31, 4, dummy, None) == 1
    assert lib.wl_group_permutation(1, 8, 0, dummy, None) == 1
    assert lib.wl_group_permutation(1, 8, 4, None, None) == 1
    lib.wl_version.restype = C.c_char_p
    assert lib.wl_version() == b"2.1"


def test_binding_never_writes_into_the_callers_options_block():
    """api.wl_eval_seeded / wl_eval(wilson_events=...) / shard.wl_eval_sharded set fields (seeded, event handles,
    ensemble_loops) on a private copy: a block the caller reuses for a later plain call keeps its own values."""
    from paper_1407_7486_b200 import api
    mine = api.wl_eval_options(quadrature_order=2, shuffle_seed=5)
    copy = api._own_options(mine)
    copy.ensemble_loops, copy.seeded, copy.seed = 99, 1, 7
    assert (mine.ensemble_loops, mine.seeded, mine.seed) == (0, 0, 0)
    assert (copy.quadrature_order, copy.shuffle_groups, copy.shuffle_seed, copy.struct_size) == (2, 1, 5, mine.struct_size)
    fresh = api._own_options(None)
    assert fresh.quadrature_order == 1 and fresh.struct_size == mine.struct_size and fresh.seeded == 0
