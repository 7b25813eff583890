"""Thin Python binding of libwl.so (include/wl.h): argument marshalling only.

Every function has the name of the C entry point it calls.  Tensors are PyTorch CUDA tensors
(device memory and streams are PyTorch's; all arithmetic runs in the library's kernels).
There is no CPU fallback: importing this module raises if libwl.so is missing or does not
load, and each call raises WLError on a non-zero status.
"""
import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libwl.so")

WL_OK = 0
PROFILE_UNIFORM = 0
PROFILE_SECH2 = 1
PROFILE_FLUXTUBE = 2
FERMION = 0
SCALAR = 1
F32 = 0
F64 = 1

if not os.path.exists(LIB_PATH):
    # a fresh checkout (the .so is not in the history): compile the CUDA sources once, in-tree; no CPU fallback
    try:
        from . import build as _build
        _build.build()
    except Exception as exc:
        raise ImportError("%s not found and `python -m paper_1407_7486_b200.build` failed (%s): "
                          "there is no CPU fallback" % (LIB_PATH, exc))
_lib = C.CDLL(LIB_PATH)

_vp, _dp, _i64, _int, _u64, _sz = C.c_void_p, C.c_void_p, C.c_int64, C.c_int, C.c_uint64, C.c_size_t
_lib.wl_field_create.restype = _int
_lib.wl_field_create.argtypes = [_int, C.POINTER(C.c_double), _int, C.POINTER(_vp)]
_lib.wl_field_create_particle.restype = _int
_lib.wl_field_create_particle.argtypes = [_int, C.POINTER(C.c_double), _int, _int, C.POINTER(_vp)]
_lib.wl_field_destroy.restype = None
_lib.wl_field_destroy.argtypes = [_vp]
_lib.wl_loops_generate.restype = _int
_lib.wl_loops_generate.argtypes = [_vp, _int, _i64, _i64, _int, _u64, _vp]
_lib.wl_eval_workspace_bytes.restype = _sz
_lib.wl_eval_workspace_bytes.argtypes = [_i64, _int, _int, _int, _int, _int]
_lib.wl_eval_launch_count.restype = _int
_lib.wl_eval_launch_count.argtypes = [_i64, _int, _int, _int, _int, _int]
_lib.wl_eval.restype = _int
_lib.wl_eval.argtypes = [_vp, _vp, _int, _i64, _int, _dp, _int, _dp, _dp, _int, _int, _int, _dp, _dp,
                         _vp, _sz, _vp]
_lib.wl_eval_static.restype = _int
_lib.wl_eval_static.argtypes = list(_lib.wl_eval.argtypes[:14]) + [_vp]
_lib.wl_eval_static_max_bytes.restype = _sz
_lib.wl_eval_static_max_bytes.argtypes = []
_lib.wl_eval_instrumented.restype = _int
_lib.wl_eval_instrumented.argtypes = list(_lib.wl_eval.argtypes) + [_vp, _vp]


class _Options(C.Structure):
    """struct wl_eval_options of include/wl.h."""
    _fields_ = [("struct_size", C.c_size_t), ("quadrature_order", C.c_int), ("seeded", C.c_int),
                ("seed", C.c_uint64), ("loop_begin", C.c_int64), ("shuffle_groups", C.c_int), ("staging", C.c_int),
                ("shuffle_seed", C.c_uint64), ("ensemble_loops", C.c_int64), ("event_wilson_begin", C.c_void_p), ("event_wilson_end", C.c_void_p)]


_op = C.POINTER(_Options)
_lib.wl_eval_options_default.restype = None
_lib.wl_eval_options_default.argtypes = [_op]
_lib.wl_eval_opt_workspace_bytes.restype = _sz
_lib.wl_eval_opt_workspace_bytes.argtypes = [_i64, _int, _int, _int, _int, _int, _op]
_lib.wl_eval_opt.restype = _int
_lib.wl_eval_opt.argtypes = list(_lib.wl_eval.argtypes) + [_op]
_lib.wl_eval_seeded.restype = _int
_lib.wl_eval_seeded.argtypes = [_vp, _u64, _i64, _int, _i64, _int, _dp, _int, _dp, _dp, _int, _int, _int, _dp, _dp,
                                _vp, _sz, _vp]
_lib.wl_group_permutation.restype = _int
_lib.wl_group_permutation.argtypes = [_u64, _i64, _int, _vp, _vp]
_lib.wl_grid_validate.restype = _int
_lib.wl_grid_validate.argtypes = [C.POINTER(C.c_double), _int, C.POINTER(C.c_double), _int]
_lib.wl_eval_discretization_workspace_bytes.restype = _sz
_lib.wl_eval_discretization_workspace_bytes.argtypes = [_i64, _int, _int, _int, _int, _int]
_lib.wl_eval_discretization.restype = _int
_lib.wl_eval_discretization.argtypes = [_vp, _vp, _int, _i64, _int, _dp, _int, _dp, _dp, _int, _int, _int, _dp,
                                        _vp, _sz, _vp]
_lib.wl_extrapolate.restype = _int
_lib.wl_extrapolate.argtypes = [_dp, _i64, _dp, _dp, _vp]
_lib.wl_proper_time_nodes.restype = _int
_lib.wl_proper_time_nodes.argtypes = [C.c_double, C.c_double, _int, C.POINTER(C.c_double)]
_lib.wl_action_density.restype = _int
_lib.wl_action_density.argtypes = [_vp, _dp, _int, _i64, _dp, _int, _dp, _int, C.c_double, C.c_double, C.c_double,
                                   _dp, _vp]
_lib.wl_action_radial.restype = _int
_lib.wl_action_radial.argtypes = [_dp, _int, _dp, _int, _dp, _vp]
_lib.wl_eval_per_loop.restype = _int
_lib.wl_eval_per_loop.argtypes = [_vp, _vp, _int, _i64, _int, _dp, _int, _dp, _dp, _int, _int, _dp, _dp,
                                  _dp, _vp]
_lib.wl_eval_per_loop_opt.restype = _int
_lib.wl_eval_per_loop_opt.argtypes = list(_lib.wl_eval_per_loop.argtypes) + [_op]
_lib.wl_jackknife_finalize.restype = _int
_lib.wl_jackknife_finalize.argtypes = [_dp, _int, _i64, _int, _int, _dp, _dp, _dp, _vp]
_lib.wl_eval_host.restype = _int
_lib.wl_eval_host.argtypes = [_vp, _vp, _int, _i64, _int, _dp, _int, _dp, _dp, _int, _int, _int, _dp, _dp,
                              _dp]
_lib.wl_eval_host_trim.restype = _int
_lib.wl_eval_host_trim.argtypes = []
_lib.wl_pipe_probe.restype = _int
_lib.wl_pipe_probe.argtypes = [_int, _i64, _vp, _vp, C.POINTER(C.c_int64), C.POINTER(C.c_int)]
_lib.wl_status_string.restype = C.c_char_p
_lib.wl_status_string.argtypes = [_int]
_lib.wl_version.restype = C.c_char_p
_lib.wl_version.argtypes = []


class WLError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        super().__init__("%s: %s (status %d)" % (where, wl_status_string(status), status))


def _check(status, where):
    if status != WL_OK:
        raise WLError(status, where)


def wl_status_string(status) -> str:
    return _lib.wl_status_string(int(status)).decode()


def wl_version() -> str:
    return _lib.wl_version().decode()


def _dtype_code(dt) -> int:
    if isinstance(dt, int) and not isinstance(dt, bool) and dt in (F32, F64):
        return dt
    s = str(dt)
    if "float32" in s or s == "f32":
        return F32
    if "float64" in s or s == "f64":
        return F64
    raise ValueError("dtype must be float32 or float64, got %r" % (dt,))


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _cuda_f64(t, name, numel=None):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise ValueError("%s must be a contiguous float64 CUDA tensor" % name)
    if numel is not None and t.numel() != numel:
        raise ValueError("%s must have %d elements" % (name, numel))
    return t


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


class Field:
    """Owns a wl_field* (wl_field_create / wl_field_destroy)."""

    def __init__(self, profile, params, particle=FERMION):
        arr = (C.c_double * len(params))(*[float(p) for p in params])
        h = C.c_void_p()
        _check(_lib.wl_field_create_particle(int(profile), arr, len(params), int(particle), C.byref(h)),
               "wl_field_create_particle")
        self._h = h
        self.profile = int(profile)
        self.params = tuple(float(p) for p in params)
        self.particle = int(particle)

    def __del__(self, _destroy=_lib.wl_field_destroy):
        h, self._h = getattr(self, "_h", None), None
        if h:
            _destroy(h)


def wl_field_create(profile, params) -> Field:
    return Field(profile, params)


def wl_field_create_particle(profile, params, particle) -> Field:
    """particle = FERMION (W = cos(phase) cosh(spin)) or SCALAR (W = cos(phase))."""
    return Field(profile, params, particle)


def wl_loops_generate(n_loops, n_ppl, seed, dtype=torch.float64, loop_begin=0, out=None, device="cuda",
                      stream=None) -> torch.Tensor:
    """Unit d-loops [n_loops][n_ppl][2] of ensemble `seed`, loops loop_begin .. loop_begin+n_loops-1."""
    if out is None:
        out = torch.empty((n_loops, n_ppl, 2), dtype=dtype, device=device)
    if not (out.is_cuda and out.is_contiguous() and out.shape == (n_loops, n_ppl, 2)):
        raise ValueError("out must be a contiguous CUDA tensor [n_loops][n_ppl][2]")
    with torch.cuda.device(out.device):
        _check(_lib.wl_loops_generate(_ptr(out), _dtype_code(out.dtype), int(loop_begin), int(n_loops),
                                      int(n_ppl), int(seed), _stream(stream)), "wl_loops_generate")
    return out


def wl_eval_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, compute) -> int:
    return int(_lib.wl_eval_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, _dtype_code(compute)))


def wl_eval_launch_count(n_loops, n_ppl, n_T, n_rho, n_groups, compute) -> int:
    return int(_lib.wl_eval_launch_count(n_loops, n_ppl, n_T, n_rho, n_groups, _dtype_code(compute)))


def _loops_arg(loops):
    if not (isinstance(loops, torch.Tensor) and loops.is_cuda and loops.is_contiguous() and loops.dim() == 3
            and loops.shape[2] == 2 and loops.dtype in (torch.float32, torch.float64)):
        raise ValueError("loops must be a contiguous CUDA tensor [n_loops][n_ppl][2], float32 or float64")
    return loops.shape[0], loops.shape[1]


def _event_handle(ev, stream):
    if ev is None:
        return None
    if not ev.cuda_event:          # torch creates the cudaEvent_t lazily, on the first record()
        ev.record(stream if stream is not None else torch.cuda.current_stream())
    return C.c_void_p(ev.cuda_event)


def wl_eval_options(quadrature_order=1, seed=None, loop_begin=0, shuffle_seed=None, staging=0,
                    ensemble_loops=0) -> _Options:
    """struct wl_eval_options: seed != None sets `seeded`, shuffle_seed != None sets `shuffle_groups`;
    ensemble_loops = size of the whole ensemble when the call evaluates one shard of it."""
    o = _Options()
    _lib.wl_eval_options_default(C.byref(o))
    o.quadrature_order = int(quadrature_order)
    if seed is not None:
        o.seeded, o.seed, o.loop_begin = 1, int(seed), int(loop_begin)
    if shuffle_seed is not None:
        o.shuffle_groups, o.shuffle_seed = 1, int(shuffle_seed)
    o.staging = int(staging)
    o.ensemble_loops = int(ensemble_loops)
    return o


def _own_options(options) -> _Options:
    """A private copy of the caller's options block (or fresh defaults): the wrappers below set fields of it
    (seeded, ensemble_loops, event handles) and must not leave them behind in an object the caller may reuse."""
    o = _Options()
    if options is None:
        _lib.wl_eval_options_default(C.byref(o))
    else:
        C.memmove(C.byref(o), C.byref(options), C.sizeof(_Options))
    return o


def _scratch(nbytes, dev, stream):
    """Scratch bytes for kernels enqueued on `stream`: allocated under that stream, so that PyTorch's caching
    allocator does not hand the block to another stream's tensor while those kernels still use it."""
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    with torch.cuda.stream(st):
        return torch.empty(max(int(nbytes), 8), dtype=torch.uint8, device=dev)


def wl_eval_opt_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, compute, options=None) -> int:
    return int(_lib.wl_eval_opt_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, _dtype_code(compute),
                                                C.byref(options) if options is not None else None))


def wl_eval(field, loops, T, rho_cm, phi_cm=None, n_groups=1, compute=torch.float64, W_mean=None,
            group_sums=None, workspace=None, stream=None, wilson_events=None, options=None):
    """Returns (W_mean [n_T][n_rho], group_sums [G][n_T][n_rho]); see include/wl.h.

    wilson_events = (begin, end) torch.cuda.Event pair (enable_timing=True): recorded around the k_wilson
    launch.  options = wl_eval_options(...): calls wl_eval_opt (quadrature order, shuffled groups, staging)."""
    n_loops, n_ppl = _loops_arg(loops)
    T = _cuda_f64(T, "T")
    rho_cm = _cuda_f64(rho_cm, "rho_cm")
    n_T, n_rho = T.numel(), rho_cm.numel()
    phi_cm = _cuda_f64(phi_cm, "phi_cm", n_rho)
    dev = loops.device
    if W_mean is None:
        W_mean = torch.empty((n_T, n_rho), dtype=torch.float64, device=dev)
    if group_sums is None:
        group_sums = torch.empty((n_groups, n_T, n_rho), dtype=torch.float64, device=dev)
    _cuda_f64(W_mean, "W_mean", n_T * n_rho)
    _cuda_f64(group_sums, "group_sums", n_groups * n_T * n_rho)
    cc = _dtype_code(compute)
    if workspace is None:
        workspace = _scratch(wl_eval_opt_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, cc, options), dev, stream)
    args = (field._h, _ptr(loops), _dtype_code(loops.dtype), n_loops, n_ppl, _ptr(T), n_T,
            _ptr(rho_cm), _ptr(phi_cm), n_rho, int(n_groups), cc, _ptr(W_mean),
            _ptr(group_sums), _ptr(workspace), workspace.numel() * workspace.element_size())
    with torch.cuda.device(dev):
        if options is not None:
            if wilson_events is not None:
                options = _own_options(options)
                e0, e1 = (_event_handle(ev, stream) for ev in wilson_events)
                options.event_wilson_begin, options.event_wilson_end = e0, e1
            _check(_lib.wl_eval_opt(*args, _stream(stream), C.byref(options)), "wl_eval_opt")
        elif wilson_events is None:
            _check(_lib.wl_eval(*args, _stream(stream)), "wl_eval")
        else:
            e0, e1 = (_event_handle(ev, stream) for ev in wilson_events)
            _check(_lib.wl_eval_instrumented(*args, _stream(stream), e0, e1), "wl_eval_instrumented")
    return W_mean, group_sums


def wl_eval_static_max_bytes() -> int:
    """Size of the library's built-in scratch array, the ceiling of wl_eval_static (bytes)."""
    return int(_lib.wl_eval_static_max_bytes())


def wl_eval_static(field, loops, T, rho_cm, phi_cm, n_groups, compute, W_mean, group_sums, stream=None):
    """wl_eval for callers that may not allocate device memory (include/wl.h, wl_eval_static).

    Nothing is allocated here either, in the library or in this binding: W_mean [n_T][n_rho] and group_sums
    [G][n_T][n_rho] must be float64 CUDA tensors the caller already owns, and the partial sums go to a 16 MiB
    array built into libwl.so (sizes that need more raise WLError with status WL_ERR_STATIC_LIMIT = 5).
    That array is shared by every call on the device: keep calls on one stream, or otherwise ordered."""
    n_loops, n_ppl = _loops_arg(loops)
    T = _cuda_f64(T, "T")
    rho_cm = _cuda_f64(rho_cm, "rho_cm")
    n_T, n_rho = T.numel(), rho_cm.numel()
    phi_cm = _cuda_f64(phi_cm, "phi_cm", n_rho)
    if W_mean is None or group_sums is None:
        raise ValueError("wl_eval_static allocates nothing: pass W_mean and group_sums")
    _cuda_f64(W_mean, "W_mean", n_T * n_rho)
    _cuda_f64(group_sums, "group_sums", n_groups * n_T * n_rho)
    with torch.cuda.device(loops.device):
        _check(_lib.wl_eval_static(field._h, _ptr(loops), _dtype_code(loops.dtype), n_loops, n_ppl, _ptr(T), n_T,
                                   _ptr(rho_cm), _ptr(phi_cm), n_rho, int(n_groups), _dtype_code(compute),
                                   _ptr(W_mean), _ptr(group_sums), _stream(stream)), "wl_eval_static")
    return W_mean, group_sums


def wl_eval_seeded(field, seed, n_loops, n_ppl, T, rho_cm, phi_cm=None, n_groups=1, compute=torch.float64,
                   storage=torch.float32, loop_begin=0, W_mean=None, group_sums=None, workspace=None, stream=None,
                   options=None):
    """wl_eval without an ensemble buffer: loops [loop_begin, loop_begin + n_loops) of ensemble `seed` are
    regenerated inside the kernel; same bits as wl_loops_generate(storage) + wl_eval.
    options (quadrature order, shuffled groups) goes through wl_eval_opt with `seeded` set."""
    T = _cuda_f64(T, "T")
    rho_cm = _cuda_f64(rho_cm, "rho_cm")
    n_T, n_rho = T.numel(), rho_cm.numel()
    phi_cm = _cuda_f64(phi_cm, "phi_cm", n_rho)
    dev = T.device
    if W_mean is None:
        W_mean = torch.empty((n_T, n_rho), dtype=torch.float64, device=dev)
    if group_sums is None:
        group_sums = torch.empty((n_groups, n_T, n_rho), dtype=torch.float64, device=dev)
    cc, sc = _dtype_code(compute), _dtype_code(storage)
    if options is not None:
        options = _own_options(options)
        options.seeded, options.seed, options.loop_begin = 1, int(seed), int(loop_begin)
    if workspace is None:
        workspace = _scratch(wl_eval_opt_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, cc, options), dev, stream)
    wsb = workspace.numel() * workspace.element_size()
    with torch.cuda.device(dev):
        if options is None:
            _check(_lib.wl_eval_seeded(field._h, int(seed), int(loop_begin), sc, int(n_loops), int(n_ppl), _ptr(T), n_T,
                                       _ptr(rho_cm), _ptr(phi_cm), n_rho, int(n_groups), cc, _ptr(W_mean),
                                       _ptr(group_sums), _ptr(workspace), wsb, _stream(stream)), "wl_eval_seeded")
        else:
            _check(_lib.wl_eval_opt(field._h, None, sc, int(n_loops), int(n_ppl), _ptr(T), n_T, _ptr(rho_cm),
                                    _ptr(phi_cm), n_rho, int(n_groups), cc, _ptr(W_mean), _ptr(group_sums),
                                    _ptr(workspace), wsb, _stream(stream), C.byref(options)), "wl_eval_opt")
    return W_mean, group_sums


def wl_group_permutation(shuffle_seed, n_loops, n_T, device="cuda", stream=None) -> torch.Tensor:
    """perm [n_T][n_loops] int32: perm[t][i] = pi_t(i), the group membership of shuffle_groups (include/wl.h)."""
    perm = torch.empty((n_T, n_loops), dtype=torch.int32, device=device)
    with torch.cuda.device(perm.device):
        _check(_lib.wl_group_permutation(int(shuffle_seed), int(n_loops), int(n_T), _ptr(perm), _stream(stream)),
               "wl_group_permutation")
    return perm


def wl_grid_validate(T, rho_cm) -> None:
    """Host check of grid values (T > 0, rho_cm >= 0, finite); raises WLError(WL_ERR_INVALID_ARG) otherwise."""
    T = np.ascontiguousarray(T, dtype=np.float64)
    rho = np.ascontiguousarray(rho_cm, dtype=np.float64)
    dp = C.POINTER(C.c_double)
    _check(_lib.wl_grid_validate(T.ctypes.data_as(dp), T.size, rho.ctypes.data_as(dp), rho.size), "wl_grid_validate")


def wl_eval_discretization(field, loops, T, rho_cm, phi_cm=None, n_groups=1, compute=torch.float64, stream=None):
    """Group sums [3][G][n_T][n_rho] at the levels (N/4, N/2, N) of Sec. IV.A, eq. (48)-(50)."""
    n_loops, n_ppl = _loops_arg(loops)
    T = _cuda_f64(T, "T")
    rho_cm = _cuda_f64(rho_cm, "rho_cm")
    n_T, n_rho = T.numel(), rho_cm.numel()
    phi_cm = _cuda_f64(phi_cm, "phi_cm", n_rho)
    cc = _dtype_code(compute)
    gs3 = torch.empty((3, n_groups, n_T, n_rho), dtype=torch.float64, device=loops.device)
    need = int(_lib.wl_eval_discretization_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, cc))
    ws = _scratch(need, loops.device, stream)
    with torch.cuda.device(loops.device):
        _check(_lib.wl_eval_discretization(field._h, _ptr(loops), _dtype_code(loops.dtype), n_loops, n_ppl, _ptr(T),
                                           n_T, _ptr(rho_cm), _ptr(phi_cm), n_rho, int(n_groups), cc, _ptr(gs3),
                                           _ptr(ws), need, _stream(stream)), "wl_eval_discretization")
    return gs3


def wl_extrapolate(levels3, want_delta=True, stream=None):
    """eq. (51)-(52) element-wise on levels3 [3][...] -> (W_inf, delta)."""
    lv = _cuda_f64(levels3, "levels3")
    if lv.shape[0] != 3:
        raise ValueError("levels3 must be [3][...]")
    n = lv.numel() // 3
    out = torch.empty(lv.shape[1:], dtype=torch.float64, device=lv.device)
    delta = torch.empty_like(out) if want_delta else None
    with torch.cuda.device(lv.device):
        _check(_lib.wl_extrapolate(_ptr(lv), n, _ptr(out), _ptr(delta), _stream(stream)), "wl_extrapolate")
    return out, delta


def wl_eval_per_loop(field, loops, T, rho_cm, phi_cm=None, compute=torch.float64, want_phase_spin=True,
                     stream=None, options=None, n_loops=None, n_ppl=None, storage=torch.float32):
    """Per-loop (W, phase, spin), each [n_loops][n_T][n_rho] (phase/spin None if not wanted).
    options: quadrature order / seeded (then loops may be None and n_loops, n_ppl, storage say what to generate)."""
    if loops is None:
        if options is None or not options.seeded:
            raise ValueError("loops=None needs seeded options")
    else:
        n_loops, n_ppl = _loops_arg(loops)
    T = _cuda_f64(T, "T")
    rho_cm = _cuda_f64(rho_cm, "rho_cm")
    n_T, n_rho = T.numel(), rho_cm.numel()
    phi_cm = _cuda_f64(phi_cm, "phi_cm", n_rho)
    dev = T.device
    W = torch.empty((n_loops, n_T, n_rho), dtype=torch.float64, device=dev)
    ph = torch.empty_like(W) if want_phase_spin else None
    sp = torch.empty_like(W) if want_phase_spin else None
    ldt = _dtype_code(loops.dtype if loops is not None else storage)
    with torch.cuda.device(dev):
        _check(_lib.wl_eval_per_loop_opt(field._h, _ptr(loops), ldt, int(n_loops), int(n_ppl), _ptr(T),
                                         n_T, _ptr(rho_cm), _ptr(phi_cm), n_rho, _dtype_code(compute), _ptr(W),
                                         _ptr(ph), _ptr(sp), _stream(stream),
                                         C.byref(options) if options is not None else None), "wl_eval_per_loop_opt")
    return W, ph, sp


def wl_jackknife_finalize(group_sums, n_loops, delete_one=False, stream=None):
    """(mean, err[, delete-one-group means]) from group_sums [G][n_T][n_rho]; eq. (60)-(63)."""
    gs = _cuda_f64(group_sums, "group_sums")
    if gs.dim() != 3:
        raise ValueError("group_sums must be [G][n_T][n_rho]")
    G, n_T, n_rho = gs.shape
    mean = torch.empty((n_T, n_rho), dtype=torch.float64, device=gs.device)
    err = torch.empty_like(mean)
    d1 = torch.empty_like(gs) if delete_one else None
    with torch.cuda.device(gs.device):
        _check(_lib.wl_jackknife_finalize(_ptr(gs), G, int(n_loops), n_T, n_rho, _ptr(mean), _ptr(err),
                                          _ptr(d1), _stream(stream)), "wl_jackknife_finalize")
    return (mean, err, d1) if delete_one else (mean, err)


def wl_eval_host(field, loops, T, rho_cm, phi_cm=None, n_groups=2, compute=torch.float64):
    """End-to-end call on HOST buffers (numpy arrays or CPU tensors; pinned memory is used as given).

    Returns numpy (W_mean, err, group_sums).  All copies happen inside the C call.
    """
    def host(a, dt=None):
        if isinstance(a, torch.Tensor):
            if a.is_cuda:
                raise ValueError("wl_eval_host takes host buffers")
            a = a.numpy()
        a = np.ascontiguousarray(a) if dt is None else np.ascontiguousarray(a, dtype=dt)
        return a
    y = host(loops)
    if y.dtype not in (np.float32, np.float64) or y.ndim != 3 or y.shape[2] != 2:
        raise ValueError("loops must be [n_loops][n_ppl][2], float32 or float64")
    T = host(T, np.float64)
    rho = host(rho_cm, np.float64)
    phi = host(phi_cm, np.float64) if phi_cm is not None else None
    n_T, n_rho = T.size, rho.size
    mean = np.empty((n_T, n_rho))
    err = np.empty((n_T, n_rho))
    gs = np.empty((n_groups, n_T, n_rho))
    p = lambda a: C.c_void_p(a.ctypes.data) if a is not None else None
    _check(_lib.wl_eval_host(field._h, p(y), _dtype_code(y.dtype.type), y.shape[0], y.shape[1], p(T), n_T,
                             p(rho), p(phi), n_rho, int(n_groups), _dtype_code(compute), p(mean), p(err),
                             p(gs)), "wl_eval_host")
    return mean, err, gs


def wl_eval_host_trim():
    """Returns the unused memory of wl_eval_host's private pool to the device."""
    _check(_lib.wl_eval_host_trim(), "wl_eval_host_trim")


def wl_pipe_probe(pipe, iters, sink, stream=None):
    """Enqueues the single-pipe instruction stream `pipe` (0 FFMA, 1 MUFU.EX2, 2 DFMA); returns (lane_ops, n_sms)."""
    ops, sms = C.c_int64(0), C.c_int(0)
    with torch.cuda.device(sink.device):
        _check(_lib.wl_pipe_probe(int(pipe), int(iters), _ptr(sink), _stream(stream), C.byref(ops), C.byref(sms)),
               "wl_pipe_probe")
    return int(ops.value), int(sms.value)


def wl_proper_time_nodes(a, Tmax, n_T) -> np.ndarray:
    """Host: the n_T proper times (Simpson nodes of x = 1/(1+T/Tmax)), increasing from a."""
    T = np.empty(int(n_T), dtype=np.float64)
    _check(_lib.wl_proper_time_nodes(float(a), float(Tmax), int(n_T), T.ctypes.data_as(C.POINTER(C.c_double))),
           "wl_proper_time_nodes")
    return T


def wl_action_density(field, group_sums, n_loops, T, rho_cm, m2, a, Tmax, stream=None):
    """Per-group proper-time integral of eq. (12)/(70): density [G][n_rho]; see include/wl.h."""
    gs = _cuda_f64(group_sums, "group_sums")
    T = _cuda_f64(T, "T")
    rho_cm = _cuda_f64(rho_cm, "rho_cm")
    G, n_T, n_rho = gs.shape
    if T.numel() != n_T or rho_cm.numel() != n_rho:
        raise ValueError("group_sums must be [G][n_T][n_rho]")
    out = torch.empty((G, n_rho), dtype=torch.float64, device=gs.device)
    with torch.cuda.device(gs.device):
        _check(_lib.wl_action_density(field._h, _ptr(gs), G, int(n_loops), _ptr(T), n_T, _ptr(rho_cm), n_rho,
                                      float(m2), float(a), float(Tmax), _ptr(out), _stream(stream)),
               "wl_action_density")
    return out


def wl_action_radial(density, rho_cm, stream=None):
    """(1/4 pi) int rho density d rho per group (eq. (12)), Simpson on the uniform grid rho_cm (n_rho odd)."""
    d = _cuda_f64(density, "density")
    rho_cm = _cuda_f64(rho_cm, "rho_cm", d.shape[1])
    out = torch.empty((d.shape[0],), dtype=torch.float64, device=d.device)
    with torch.cuda.device(d.device):
        _check(_lib.wl_action_radial(_ptr(d), d.shape[0], _ptr(rho_cm), d.shape[1], _ptr(out), _stream(stream)),
               "wl_action_radial")
    return out
