"""ctypes binding of oracle/wl_oracle.c (FP64 CPU oracle).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs import this module.  It does not
import the product package and the product package does not import it.

Argument marshalling only; all arithmetic is in wl_oracle.c (each function there
cites the PAPER.md passage it follows).
"""
import ctypes as C

import numpy as np

from . import build as _build

UNIFORM = 0
SECH2 = 1
FLUXTUBE = 2

_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.wlo_field_g.restype = C.c_double
        L.wlo_field_g.argtypes = [C.c_int, _dp, C.c_double]
        L.wlo_field_b.restype = C.c_double
        L.wlo_field_b.argtypes = [C.c_int, _dp, C.c_double]
        L.wlo_loop_phase_spin.restype = None
        L.wlo_loop_phase_spin.argtypes = [C.c_int, _dp, _dp, C.c_int, C.c_double, C.c_double,
                                          C.c_double, _dp, _dp]
        L.wlo_eval.restype = C.c_int
        L.wlo_eval.argtypes = [C.c_int, _dp, _dp, C.c_int64, C.c_int, _dp, C.c_int, _dp, _dp,
                               C.c_int, C.c_int, _dp, _dp, _dp, _dp, _dp]
        L.wlo_eval_particle.restype = C.c_int
        L.wlo_eval_particle.argtypes = [C.c_int, _dp, C.c_int, _dp, C.c_int64, C.c_int, _dp, C.c_int, _dp, _dp,
                                        C.c_int, C.c_int, _dp, _dp, _dp, _dp, _dp]
        L.wlo_eval_discretization.restype = C.c_int
        L.wlo_eval_discretization.argtypes = [C.c_int, _dp, C.c_int, _dp, C.c_int64, C.c_int, _dp, C.c_int, _dp,
                                              _dp, C.c_int, C.c_int, _dp, _dp]
        L.wlo_extrapolate.restype = None
        L.wlo_extrapolate.argtypes = [_dp, C.c_int64, _dp, _dp]
        L.wlo_proper_time_nodes.restype = C.c_int
        L.wlo_proper_time_nodes.argtypes = [C.c_double, C.c_double, C.c_int, _dp]
        L.wlo_small_T_integral.restype = C.c_double
        L.wlo_small_T_integral.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int]
        L.wlo_action_density.restype = C.c_int
        L.wlo_action_density.argtypes = [C.c_int, _dp, C.c_int, _dp, C.c_int, C.c_int64, _dp, C.c_int, _dp, C.c_int,
                                         C.c_double, C.c_double, C.c_double, _dp]
        L.wlo_action_radial.restype = C.c_int
        L.wlo_action_radial.argtypes = [_dp, C.c_int, _dp, C.c_int, _dp]
        L.wlo_finalize.restype = C.c_int
        L.wlo_finalize.argtypes = [_dp, C.c_int, C.c_int64, C.c_int64, _dp, _dp, _dp]
        L.wlo_philox4x32_10.restype = None
        L.wlo_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.wlo_normal_pair.restype = None
        L.wlo_normal_pair.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, _dp, _dp]
        L.wlo_generate_loops.restype = C.c_int
        L.wlo_generate_loops.argtypes = [C.c_uint64, C.c_int64, C.c_int64, C.c_int, _dp]
        L.wlo_num_threads.restype = C.c_int
        L.wlo_gauss_legendre_01.restype = C.c_int
        L.wlo_gauss_legendre_01.argtypes = [C.c_int, _dp, _dp]
        L.wlo_loop_phase_spin_q.restype = C.c_int
        L.wlo_loop_phase_spin_q.argtypes = [C.c_int, _dp, _dp, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                            _dp, _dp]
        L.wlo_eval_quadrature.restype = C.c_int
        L.wlo_eval_quadrature.argtypes = [C.c_int, _dp, C.c_int, C.c_int, _dp, C.c_int64, C.c_int, _dp, C.c_int, _dp,
                                          _dp, C.c_int, C.c_int, _dp, _dp, _dp, _dp, _dp]
        L.wlo_shuffle_index.restype = C.c_int64
        L.wlo_shuffle_index.argtypes = [C.c_uint64, C.c_int, C.c_int64, C.c_int64]
        L.wlo_group_permutation.restype = C.c_int
        L.wlo_group_permutation.argtypes = [C.c_uint64, C.c_int64, C.c_int, C.POINTER(C.c_int64)]
        L.wlo_regroup_shuffled.restype = C.c_int
        L.wlo_regroup_shuffled.argtypes = [_dp, C.c_int64, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int64), _dp, _dp]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def field_g(profile, params, rho):
    """g(rho) = e A_phi(rho)/rho, vectorised over rho."""
    pr = _f64(params)
    r = np.atleast_1d(_f64(rho))
    return np.array([lib().wlo_field_g(profile, _p(pr), float(x)) for x in r.ravel()]).reshape(r.shape)


def field_b(profile, params, rho):
    """b(rho) = e B_z(rho), vectorised over rho."""
    pr = _f64(params)
    r = np.atleast_1d(_f64(rho))
    return np.array([lib().wlo_field_b(profile, _p(pr), float(x)) for x in r.ravel()]).reshape(r.shape)


def loop_phase_spin(profile, params, y, T, cx, cy):
    """(phase, spin) of one unit loop y[N][2] at proper time T and centre (cx, cy)."""
    pr = _f64(params)
    y = _f64(y)
    assert y.ndim == 2 and y.shape[1] == 2
    ph, sp = C.c_double(), C.c_double()
    lib().wlo_loop_phase_spin(profile, _p(pr), _p(y), y.shape[0], float(T), float(cx), float(cy),
                              C.byref(ph), C.byref(sp))
    return ph.value, sp.value


def evaluate(profile, params, loops, T, rho_cm, phi_cm=None, n_groups=1, per_loop=False, scalar=False):
    """Whole-ensemble evaluation (scalar=True: scalar QED, W = cos(phase), eq. (19)-(20), (43)).

    loops [n_loops][N][2] (float32 storage is promoted exactly to float64).
    Returns dict(W_mean [n_T][n_rho], group_sums [G][n_T][n_rho]) and, if per_loop,
    W, phase, spin of shape [n_loops][n_T][n_rho].
    """
    pr = _f64(params)
    y = _f64(loops)
    assert y.ndim == 3 and y.shape[2] == 2
    T = _f64(T)
    rho = _f64(rho_cm)
    phi = _f64(phi_cm) if phi_cm is not None else None
    nl, N = y.shape[0], y.shape[1]
    nT, nr = T.shape[0], rho.shape[0]
    if phi is not None:
        assert phi.shape == rho.shape
    mean = np.empty((nT, nr))
    gs = np.empty((n_groups, nT, nr))
    W = ph = sp = None
    if per_loop:
        W, ph, sp = (np.empty((nl, nT, nr)) for _ in range(3))
    rc = lib().wlo_eval_particle(profile, _p(pr), 1 if scalar else 0, _p(y), nl, N, _p(T), nT, _p(rho), _p(phi),
                                 nr, n_groups, _p(mean), _p(gs), _p(W), _p(ph), _p(sp))
    if rc != 0:
        raise ValueError("wlo_eval: invalid argument")
    out = {"W_mean": mean, "group_sums": gs}
    if per_loop:
        out.update(W=W, phase=ph, spin=sp)
    return out


def gauss_legendre_01(Q):
    """(nodes, weights) of the Q-point Gauss-Legendre rule on [0, 1] as the oracle uses them (Q = 1, 2, 3)."""
    t, w = np.empty(3), np.empty(3)
    if lib().wlo_gauss_legendre_01(int(Q), _p(t), _p(w)) != 0:
        raise ValueError("Q must be 1, 2 or 3")
    return t[:Q].copy(), w[:Q].copy()


def loop_phase_spin_q(profile, params, y, T, cx, cy, Q):
    """(phase, spin) of one unit loop with the Q-point rule for the t-integral of eq. (24), eq. (25)-(28)."""
    pr = _f64(params)
    y = _f64(y)
    assert y.ndim == 2 and y.shape[1] == 2
    ph, sp = C.c_double(), C.c_double()
    if lib().wlo_loop_phase_spin_q(profile, _p(pr), _p(y), y.shape[0], float(T), float(cx), float(cy), int(Q),
                                   C.byref(ph), C.byref(sp)) != 0:
        raise ValueError("Q must be 1, 2 or 3")
    return ph.value, sp.value


def evaluate_quadrature(profile, params, loops, T, rho_cm, phi_cm=None, n_groups=1, per_loop=False, scalar=False,
                        Q=1):
    """`evaluate` with the Q-point Gauss-Legendre rule for the t-integral of eq. (24)."""
    pr = _f64(params)
    y = _f64(loops)
    assert y.ndim == 3 and y.shape[2] == 2
    T = _f64(T)
    rho = _f64(rho_cm)
    phi = _f64(phi_cm) if phi_cm is not None else None
    nl, N = y.shape[0], y.shape[1]
    nT, nr = T.shape[0], rho.shape[0]
    mean = np.empty((nT, nr))
    gs = np.empty((n_groups, nT, nr))
    W = ph = sp = None
    if per_loop:
        W, ph, sp = (np.empty((nl, nT, nr)) for _ in range(3))
    rc = lib().wlo_eval_quadrature(profile, _p(pr), 1 if scalar else 0, int(Q), _p(y), nl, N, _p(T), nT, _p(rho),
                                   _p(phi), nr, n_groups, _p(mean), _p(gs), _p(W), _p(ph), _p(sp))
    if rc != 0:
        raise ValueError("wlo_eval_quadrature: invalid argument")
    out = {"W_mean": mean, "group_sums": gs}
    if per_loop:
        out.update(W=W, phase=ph, spin=sp)
    return out


def shuffle_index(seed, t, n_loops, i):
    """pi_t(i): the loop at position i of the shuffled order used at proper-time index t."""
    return int(lib().wlo_shuffle_index(int(seed), int(t), int(n_loops), int(i)))


def group_permutation(seed, n_loops, n_T):
    """perm [n_T][n_loops] (int64): perm[t][i] = pi_t(i)."""
    perm = np.empty((n_T, n_loops), dtype=np.int64)
    if lib().wlo_group_permutation(int(seed), int(n_loops), int(n_T),
                                   perm.ctypes.data_as(C.POINTER(C.c_int64))) != 0:
        raise ValueError("wlo_group_permutation: invalid argument")
    return perm


def regroup_shuffled(W_loop, n_groups, perm):
    """(W_mean [n_T][n_rho], group_sums [G][n_T][n_rho]) from per-loop W [n_loops][n_T][n_rho] with the
    per-T group membership of `perm` [n_T][n_loops] (eq. (60) with shuffled groups)."""
    W = _f64(W_loop)
    nl, nT, nr = W.shape
    perm = np.ascontiguousarray(perm, dtype=np.int64)
    assert perm.shape == (nT, nl)
    mean = np.empty((nT, nr))
    gs = np.empty((n_groups, nT, nr))
    if lib().wlo_regroup_shuffled(_p(W), nl, nT, nr, int(n_groups), perm.ctypes.data_as(C.POINTER(C.c_int64)),
                                  _p(gs), _p(mean)) != 0:
        raise ValueError("wlo_regroup_shuffled: invalid argument")
    return mean, gs


def evaluate_discretization(profile, params, loops, T, rho_cm, phi_cm=None, n_groups=1, per_loop=False,
                            scalar=False):
    """Sec. IV.A, eq. (48)-(50): group sums [3][G][n_T][n_rho] at the levels (N/4, N/2, N) of the paper's
    interleaved sub-worldline scheme (and per-loop W [3][n_loops][n_T][n_rho] if per_loop)."""
    pr = _f64(params)
    y = _f64(loops)
    assert y.ndim == 3 and y.shape[2] == 2
    T = _f64(T)
    rho = _f64(rho_cm)
    phi = _f64(phi_cm) if phi_cm is not None else None
    nl, N = y.shape[0], y.shape[1]
    gs = np.empty((3, n_groups, T.shape[0], rho.shape[0]))
    W = np.empty((3, nl, T.shape[0], rho.shape[0])) if per_loop else None
    rc = lib().wlo_eval_discretization(profile, _p(pr), 1 if scalar else 0, _p(y), nl, N, _p(T), T.shape[0],
                                       _p(rho), _p(phi), rho.shape[0], n_groups, _p(gs), _p(W))
    if rc != 0:
        raise ValueError("wlo_eval_discretization: invalid argument (N must be a multiple of 4)")
    return (gs, W) if per_loop else gs


def extrapolate(levels):
    """eq. (51)-(52): levels [3][...] (N/4, N/2, N) -> (W_inf, delta = |W_N - W_inf|)."""
    a = _f64(levels)
    n = int(np.prod(a.shape[1:])) if a.ndim > 1 else 1
    out = np.empty(n)
    delta = np.empty(n)
    lib().wlo_extrapolate(_p(a), n, _p(out), _p(delta))
    return out.reshape(a.shape[1:]), delta.reshape(a.shape[1:])


def proper_time_nodes(a, Tmax, n):
    """Simpson nodes of x = 1/(1 + T/Tmax) on [0, x_a] as proper times T_0 = a < T_1 < ...."""
    T = np.empty(n)
    if lib().wlo_proper_time_nodes(float(a), float(Tmax), int(n), _p(T)) != 0:
        raise ValueError("proper_time_nodes: a > 0, Tmax > 0, n even >= 2")
    return T


def small_T_integral(eB, m2, a, scalar=False):
    """int_0^a of the small-T expansion eq. (44) (fermion) / (45) (scalar)."""
    return lib().wlo_small_T_integral(float(eB), float(m2), float(a), 1 if scalar else 0)


def action_density(profile, params, group_sums, n_loops, T, rho_cm, m2, a, Tmax, scalar=False):
    """Per-group proper-time integral of eq. (12)/(70): density [G][n_rho] (eq. (47))."""
    pr = _f64(params)
    gs = _f64(group_sums)
    T = _f64(T)
    rho = _f64(rho_cm)
    G = gs.shape[0]
    assert gs.shape == (G, T.shape[0], rho.shape[0])
    out = np.empty((G, rho.shape[0]))
    rc = lib().wlo_action_density(profile, _p(pr), 1 if scalar else 0, _p(gs), G, int(n_loops), _p(T), T.shape[0],
                                  _p(rho), rho.shape[0], float(m2), float(a), float(Tmax), _p(out))
    if rc != 0:
        raise ValueError("wlo_action_density: invalid argument")
    return out


def action_radial(density, rho_cm):
    """eq. (12): (1/4 pi) int rho density d rho per group, Simpson on a uniform grid (n_rho odd)."""
    d = _f64(density)
    rho = _f64(rho_cm)
    out = np.empty(d.shape[0])
    if lib().wlo_action_radial(_p(d), d.shape[0], _p(rho), rho.shape[0], _p(out)) != 0:
        raise ValueError("wlo_action_radial: n_rho must be odd >= 3")
    return out


def finalize(group_sums, n_loops, delete_one=False):
    """eq. (60)-(63): (mean, err[, delete-one-group means]) from group sums [G][...]."""
    gs = _f64(group_sums)
    G = gs.shape[0]
    grid_shape = gs.shape[1:]
    n_grid = int(np.prod(grid_shape)) if grid_shape else 1
    mean = np.empty(n_grid)
    err = np.empty(n_grid)
    d1 = np.empty((G, n_grid)) if delete_one else None
    rc = lib().wlo_finalize(_p(gs), G, n_loops, n_grid, _p(mean), _p(err), _p(d1))
    if rc != 0:
        raise ValueError("wlo_finalize: invalid argument")
    res = (mean.reshape(grid_shape), err.reshape(grid_shape))
    if delete_one:
        res += (d1.reshape((G,) + grid_shape),)
    return res


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    lib().wlo_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def normal_pair(seed, loop, point):
    a, b = C.c_double(), C.c_double()
    lib().wlo_normal_pair(seed, loop, point, C.byref(a), C.byref(b))
    return a.value, b.value


def generate_loops(seed, n_loops, n_ppl, loop_begin=0):
    """Unit d-loops [n_loops][n_ppl][2], FP64, centre of mass at the origin."""
    out = np.empty((n_loops, n_ppl, 2))
    rc = lib().wlo_generate_loops(seed, loop_begin, n_loops, n_ppl, _p(out))
    if rc != 0:
        raise ValueError("wlo_generate_loops: n_ppl must be a power of two >= 2")
    return out


def num_threads():
    return lib().wlo_num_threads()
