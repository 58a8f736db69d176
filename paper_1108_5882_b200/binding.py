"""Thin ctypes binding of include/pwa.h — argument marshalling only.

Every step of the hot path runs inside libpwa.so's CUDA kernels; there is no Python or CPU
fallback: if the shared library is missing, import of this module raises, and if no CUDA
device is present pwa_create raises PwaError(PWA_ERR_CUDA).

Functions carry the same names as the C entry points.  Amplitude arrays are numpy arrays
(host) of shape [N, n, 2] or torch CUDA tensors / raw device pointers (device); V is a
float64 numpy array [n, 2] (or [K, n, 2] for the batched call).
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libpwa.so")

PWA_OK, PWA_ERR_INVALID_ARG, PWA_ERR_STATE, PWA_ERR_OOM, PWA_ERR_CUDA, PWA_ERR_UNSUPPORTED, \
    PWA_WARN_NONFINITE = range(7)
PWA_F64, PWA_F32 = 0, 1
PWA_DATA, PWA_MC = 0, 1
PWA_COPY, PWA_BORROW = 0, 1

SYMBOLS = [
    "pwa_create", "pwa_destroy", "pwa_last_error", "pwa_status_string", "pwa_upload_events",
    "pwa_upload_events_factored", "pwa_set_wave_map", "pwa_set_resonances", "pwa_build_norm",
    "pwa_set_norm", "pwa_nll_grad", "pwa_nll_grad_batch", "pwa_nll_grad_enqueue",
    "pwa_nll_grad_batch_enqueue", "pwa_fetch", "pwa_data_term_enqueue", "pwa_assemble_host",
    "pwa_res_grad", "pwa_minimize_bfgs", "pwa_minimize_bfgs_batch", "pwa_n_waves",
    "pwa_launch_count", "pwa_sync", "pwa_set_option", "pwa_microbench", "pwa_norm_error_bound",
    "pwa_assemble_host_eq2", "pwa_grad_to_polar", "pwa_polar_to_cartesian", "pwa_fix_phase_host", "pwa_fumili_hessian", "pwa_set_weights",
    "pwa_batch_path", "pwa_minimize_bfgs_floating", "pwa_minimize_bfgs_batch_ex", "pwa_minimize_bfgs_floating_ex",
    "pwa_n_res", "pwa_nll_grad_floating", "pwa_get_option", "pwa_storage", "pwa_n_events", "pwa_norm_sums", "pwa_combine_norm_host", "pwa_assemble_host_shards",
    "pwa_data_term_static",
]
PWA_FIT_CONVERGED, PWA_FIT_MAX_ITER, PWA_FIT_LINE_SEARCH = 0, 1, 2


class PwaError(RuntimeError):
    def __init__(self, status, msg=""):
        self.status = int(status)
        super().__init__(f"{_status_name(status)}: {msg}")


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} not found: build it with `python -m paper_1108_5882_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, u32, dp = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.POINTER(C.c_double)
    sig = {
        "pwa_create": (C.c_int, [C.POINTER(vp), i32, C.c_int, i32, vp]),
        "pwa_destroy": (None, [vp]),
        "pwa_last_error": (C.c_char_p, [vp]),
        "pwa_status_string": (C.c_char_p, [C.c_int]),
        "pwa_upload_events": (C.c_int, [vp, C.c_int, vp, i64, i64, u32]),
        "pwa_upload_events_factored": (C.c_int, [vp, C.c_int, vp, vp, i32, i64, i64, u32]),
        "pwa_set_wave_map": (C.c_int, [vp, i32, vp, vp]),
        "pwa_set_resonances": (C.c_int, [vp, vp, vp]),
        "pwa_build_norm": (C.c_int, [vp, vp]),
        "pwa_set_norm": (C.c_int, [vp, vp]),
        "pwa_nll_grad": (C.c_int, [vp, vp, dp, vp, vp]),
        "pwa_nll_grad_batch": (C.c_int, [vp, i32, vp, vp, vp, vp]),
        "pwa_nll_grad_enqueue": (C.c_int, [vp, vp]),
        "pwa_nll_grad_batch_enqueue": (C.c_int, [vp, i32, vp]),
        "pwa_fetch": (C.c_int, [vp, i32, vp, vp, vp]),
        "pwa_data_term_enqueue": (C.c_int, [vp, vp, vp]),
        "pwa_data_term_static": (C.c_int, [i32, vp, C.c_int, i32, vp, C.c_int64, vp, vp, vp, i32]),
        "pwa_assemble_host": (C.c_int, [i32, C.c_double, vp, vp, vp, dp, vp, vp]),
        "pwa_res_grad": (C.c_int, [vp, vp, vp, vp]),
        "pwa_minimize_bfgs": (C.c_int, [vp, vp, i32, C.c_double, dp, C.POINTER(i32), C.POINTER(i32)]),
        "pwa_minimize_bfgs_batch": (C.c_int, [vp, i32, vp, i32, C.c_double, vp, C.POINTER(i32)]),
        "pwa_n_waves": (i32, [vp]),
        "pwa_launch_count": (C.c_uint64, [vp]),
        "pwa_sync": (C.c_int, [vp]),
        "pwa_set_option": (C.c_int, [vp, C.c_char_p, i32]),
        "pwa_microbench": (C.c_int, [vp, i32, i64, dp]),
        "pwa_norm_error_bound": (C.c_int, [vp, dp, C.POINTER(i32)]),
        "pwa_assemble_host_eq2": (C.c_int, [i32, C.c_double, C.c_double, vp, vp, vp, dp, vp, vp]),
        "pwa_grad_to_polar": (C.c_int, [i32, vp, vp, vp]),
        "pwa_fumili_hessian": (C.c_int, [vp, vp, vp, i32]),
        "pwa_set_weights": (C.c_int, [vp, C.c_int, vp, u32]),
        "pwa_polar_to_cartesian": (C.c_int, [i32, vp, vp]),
        "pwa_fix_phase_host": (C.c_int, [i32, i32, vp, vp]),
        "pwa_batch_path": (C.c_int, [vp, C.POINTER(i32), dp]),
        "pwa_minimize_bfgs_floating": (C.c_int, [vp, vp, vp, vp, i32, vp, i32, i32, C.c_double, dp,
                                                 C.POINTER(i32), C.POINTER(i32)]),
        "pwa_minimize_bfgs_floating_ex": (C.c_int, [vp, vp, vp, vp, i32, vp, i32, i32, C.c_double, dp,
                                                    C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]),
        "pwa_minimize_bfgs_batch_ex": (C.c_int, [vp, i32, vp, i32, C.c_double, vp, vp, vp, C.POINTER(i32)]),
        "pwa_n_res": (i32, [vp]),
        "pwa_nll_grad_floating": (C.c_int, [vp, vp, vp, vp, dp, vp, vp, vp, vp]),
        "pwa_get_option": (C.c_int, [vp, C.c_char_p, C.POINTER(i32)]),
        "pwa_storage": (C.c_int, [vp]),
        "pwa_n_events": (i64, [vp, C.c_int]),
        "pwa_norm_sums": (C.c_int, [vp, vp, C.POINTER(i64)]),
        "pwa_combine_norm_host": (C.c_int, [i32, i32, vp, vp, vp, C.POINTER(i64)]),
        "pwa_assemble_host_shards": (C.c_int, [i32, i32, vp, vp, vp, i32, C.c_double, dp, vp, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)          # AttributeError here = header/library mismatch
        fn.restype, fn.argtypes = res, args
    return lib


_lib = _load()


def _status_name(s):
    return _lib.pwa_status_string(int(s)).decode()


def _check(ctx, status, allow_warn=True):
    status = int(status)
    if status == PWA_OK or (allow_warn and status == PWA_WARN_NONFINITE):
        return status
    msg = _lib.pwa_last_error(ctx).decode() if ctx else ""
    raise PwaError(status, msg)


def _ptr_and_keep(x):
    """-> (address, keepalive, dtype_code or None). numpy -> host ptr; torch tensor / int -> device ptr."""
    if x is None:
        return None, None, None
    if isinstance(x, int):
        return x, None, None
    if isinstance(x, np.ndarray):
        x = np.ascontiguousarray(x)
        return x.ctypes.data, x, (PWA_F32 if x.dtype == np.float32 else PWA_F64 if x.dtype == np.float64 else None)
    if hasattr(x, "data_ptr"):   # torch tensor (device or pinned host)
        if not x.is_contiguous():
            raise ValueError("tensor must be contiguous")
        code = {"torch.float32": PWA_F32, "torch.float64": PWA_F64}.get(str(x.dtype))
        return x.data_ptr(), x, code
    raise TypeError(f"unsupported buffer type {type(x)}")


def _f64(x, shape=None):
    a = np.ascontiguousarray(x, dtype=np.float64)
    if shape is not None and tuple(a.shape) != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def pwa_create(n_waves, storage, device=0, cuda_stream=0):
    """storage: PWA_F64 / PWA_F32 or 'f64' / 'f32'.  Returns an opaque context handle."""
    if isinstance(storage, str):
        storage = {"f64": PWA_F64, "f32": PWA_F32}[storage]
    ctx = C.c_void_p()
    st = _lib.pwa_create(C.byref(ctx), int(n_waves), int(storage), int(device), C.c_void_p(int(cuda_stream) or None))
    if st != PWA_OK:
        raise PwaError(st, "pwa_create failed (no CUDA device, bad arguments or out of memory)")
    return ctx


def pwa_destroy(ctx):
    _lib.pwa_destroy(ctx)


def _check_amps(ctx, x, n_events, inner, what):
    """The C side reads n_events * inner * 2 elements of the context's storage type: refuse arrays of another
    dtype or with fewer elements (a raw int address cannot be checked)."""
    ptr, keep, code = _ptr_and_keep(x)
    if isinstance(x, int) or x is None:
        return ptr, keep
    storage = int(_lib.pwa_storage(ctx))
    if code != storage:
        raise TypeError(f"{what}: dtype {getattr(keep, 'dtype', None)} does not match the context's storage "
                        f"({'float32' if storage == PWA_F32 else 'float64'})")
    have = int(np.prod(keep.shape))
    if have < int(n_events) * inner * 2:
        raise ValueError(f"{what}: {have} elements, need n_events * {inner} * 2 = {int(n_events) * inner * 2}")
    return ptr, keep


def pwa_upload_events(ctx, which, amps, n_events=None, n_generated=0, flags=PWA_COPY):
    n = _lib.pwa_n_waves(ctx)
    if n_events is None:
        if tuple(amps.shape[1:]) != (n, 2):
            raise ValueError(f"amps must be [N, {n}, 2], got {tuple(amps.shape)}")
        n_events = amps.shape[0]
    ptr, keep = _check_amps(ctx, amps, n_events, n, "amps")
    _check(ctx, _lib.pwa_upload_events(ctx, int(which), C.c_void_p(ptr), int(n_events), int(n_generated), int(flags)))
    return keep


def pwa_upload_events_factored(ctx, which, mass, ang, n_ang=None, n_events=None, n_generated=0, flags=PWA_COPY):
    if n_events is None:
        n_events = ang.shape[0]
    if n_ang is None:
        n_ang = ang.shape[1]
    if isinstance(mass, np.ndarray):
        mass = np.ascontiguousarray(mass, dtype=np.float64)
    pm, km, cm = _ptr_and_keep(mass)
    if not isinstance(mass, int) and (cm != PWA_F64 or int(np.prod(km.shape)) < int(n_events)):
        raise ValueError("mass must be float64 with >= n_events elements")
    pa, ka = _check_amps(ctx, ang, n_events, int(n_ang), "ang")
    _check(ctx, _lib.pwa_upload_events_factored(ctx, int(which), C.c_void_p(pm), C.c_void_p(pa), int(n_ang),
                                                int(n_events), int(n_generated), int(flags)))
    return km, ka


def pwa_set_weights(ctx, which, w, flags=PWA_COPY):
    """w: float64 numpy [n_events] / torch CUDA tensor / None (remove).  Returns the keep-alive object for BORROW."""
    if w is None:
        _check(ctx, _lib.pwa_set_weights(ctx, int(which), None, int(flags)))
        return None
    if isinstance(w, np.ndarray):
        w = np.ascontiguousarray(w, dtype=np.float64)
    addr, keep, code = _ptr_and_keep(w)
    if not isinstance(w, int):
        if code != PWA_F64 or int(np.prod(keep.shape)) != int(_lib.pwa_n_events(ctx, int(which))):
            raise ValueError("weights must be float64 with one element per event of the uploaded sample")
    _check(ctx, _lib.pwa_set_weights(ctx, int(which), C.c_void_p(addr), int(flags)))
    return keep


def pwa_set_wave_map(ctx, n_res, res_of_wave, ang_of_wave):
    r = np.ascontiguousarray(res_of_wave, dtype=np.int32)
    a = np.ascontiguousarray(ang_of_wave, dtype=np.int32)
    n = _lib.pwa_n_waves(ctx)
    if r.shape != (n,) or a.shape != (n,):
        raise ValueError(f"res_of_wave and ang_of_wave must have n_waves = {n} entries")
    _check(ctx, _lib.pwa_set_wave_map(ctx, int(n_res), r.ctypes.data, a.ctypes.data))


def pwa_set_resonances(ctx, mass0, width0):
    nr = (_lib.pwa_n_res(ctx),)
    m, w = _f64(mass0, nr), _f64(width0, nr)
    _check(ctx, _lib.pwa_set_resonances(ctx, m.ctypes.data, w.ctypes.data))


def pwa_build_norm(ctx, want_M=True):
    n = _lib.pwa_n_waves(ctx)
    if not want_M:
        _check(ctx, _lib.pwa_build_norm(ctx, None))
        return None
    M = np.empty((n, n, 2))
    _check(ctx, _lib.pwa_build_norm(ctx, M.ctypes.data))
    return M


def pwa_norm_error_bound(ctx):
    """-> (bound on max|M_ab - exact|, path) with path 0 = FP64 build, 1 = int8 tcgen05 build."""
    b, w = C.c_double(0.0), C.c_int32(0)
    _check(ctx, _lib.pwa_norm_error_bound(ctx, C.byref(b), C.byref(w)))
    return b.value, int(w.value)


def pwa_batch_path(ctx):
    """-> (path, err_rel) of the most recent batched call: 0 = streaming passes, 1 = FP64 DMMA, 2 = int8 tcgen05."""
    w, e = C.c_int32(0), C.c_double(0.0)
    _check(ctx, _lib.pwa_batch_path(ctx, C.byref(w), C.byref(e)))
    return int(w.value), e.value


def pwa_set_norm(ctx, M):
    n = _lib.pwa_n_waves(ctx)
    M = _f64(M, (n, n, 2))
    _check(ctx, _lib.pwa_set_norm(ctx, M.ctypes.data))


def pwa_nll_grad(ctx, V, want_status=False):
    """-> (nll, grad[n, 2], parts[2]) (+ status when want_status)."""
    n = _lib.pwa_n_waves(ctx)
    V = _f64(V, (n, 2))
    nll = C.c_double(0.0)
    grad, parts = np.empty((n, 2)), np.empty(2)
    st = _check(ctx, _lib.pwa_nll_grad(ctx, V.ctypes.data, C.byref(nll), grad.ctypes.data, parts.ctypes.data))
    return (nll.value, grad, parts, st) if want_status else (nll.value, grad, parts)


def pwa_nll_grad_batch(ctx, V, want_status=False):
    """V [K, n, 2] -> (nll[K], grad[K, n, 2], parts[K, 2])."""
    n = _lib.pwa_n_waves(ctx)
    V = _f64(V)
    K = V.shape[0]
    if V.shape != (K, n, 2):
        raise ValueError("V must be [K, n, 2]")
    nll, grad, parts = np.empty(K), np.empty((K, n, 2)), np.empty((K, 2))
    st = _check(ctx, _lib.pwa_nll_grad_batch(ctx, K, V.ctypes.data, nll.ctypes.data, grad.ctypes.data, parts.ctypes.data))
    return (nll, grad, parts, st) if want_status else (nll, grad, parts)


def pwa_nll_grad_enqueue(ctx, V):
    n = _lib.pwa_n_waves(ctx)
    V = _f64(V, (n, 2))
    _check(ctx, _lib.pwa_nll_grad_enqueue(ctx, V.ctypes.data))


def pwa_nll_grad_batch_enqueue(ctx, V):
    V = _f64(V)
    if V.ndim != 3 or V.shape[1:] != (_lib.pwa_n_waves(ctx), 2):
        raise ValueError("V must be [K, n, 2]")
    _check(ctx, _lib.pwa_nll_grad_batch_enqueue(ctx, V.shape[0], V.ctypes.data))


def pwa_fetch(ctx, K=1):
    n = _lib.pwa_n_waves(ctx)
    nll, grad, parts = np.empty(K), np.empty((K, n, 2)), np.empty((K, 2))
    _check(ctx, _lib.pwa_fetch(ctx, int(K), nll.ctypes.data, grad.ctypes.data, parts.ctypes.data))
    return nll, grad, parts


def pwa_data_term_enqueue(ctx, V, out_dev):
    """out_dev: torch CUDA float64 tensor with >= 2 + 2n elements (or a raw device address)."""
    n = _lib.pwa_n_waves(ctx)
    V = _f64(V, (n, 2))
    ptr, _, _ = _ptr_and_keep(out_dev)
    _check(ctx, _lib.pwa_data_term_enqueue(ctx, V.ctypes.data, C.c_void_p(ptr)))


PWA_STATIC_MAX_WAVES = 64


def pwa_data_term_static(amps_dev, V, out_dev, n_events=None, device=0, cuda_stream=0):
    """Allocation-free data term (no context): amps_dev torch CUDA tensor [N, n, 2] float32 / float64, V [n, 2],
    out_dev torch CUDA float64 tensor with >= 2 + 2n elements.  Asynchronous on cuda_stream."""
    V = _f64(V)
    n = V.shape[0]
    if V.shape != (n, 2):
        raise ValueError(f"V must be [n, 2], got {V.shape}")
    pa, ka, code = _ptr_and_keep(amps_dev)
    if code is None or isinstance(ka, np.ndarray):
        raise TypeError("amps_dev must be a float32 / float64 CUDA tensor")
    if n_events is None:
        if tuple(ka.shape[1:]) != (n, 2):
            raise ValueError(f"amps_dev must be [N, {n}, 2], got {tuple(ka.shape)}")
        n_events = ka.shape[0]
    if int(np.prod(ka.shape)) < int(n_events) * n * 2:
        raise ValueError("amps_dev holds fewer than n_events * n * 2 elements")
    po, ko, co = _ptr_and_keep(out_dev)
    if co != PWA_F64 or int(np.prod(ko.shape)) < 2 + 2 * n:
        raise ValueError("out_dev must be a float64 CUDA tensor with >= 2 + 2n elements")
    err = C.create_string_buffer(256)
    st = int(_lib.pwa_data_term_static(int(device), C.c_void_p(int(cuda_stream) or None), int(code), n, C.c_void_p(pa),
                                       int(n_events), V.ctypes.data, C.c_void_p(po), err, 256))
    if st != PWA_OK:
        raise PwaError(st, err.value.decode())


def pwa_assemble_host(L_data, T, M, V):
    """Host-only step A7 -> (nll, grad[n, 2], parts[2])."""
    V = _f64(V)
    n = V.shape[0]
    T, M = _f64(T, (n, 2)), _f64(M, (n, n, 2))
    nll = C.c_double(0.0)
    grad, parts = np.empty((n, 2)), np.empty(2)
    st = _lib.pwa_assemble_host(n, float(L_data), T.ctypes.data, M.ctypes.data, V.ctypes.data,
                                C.byref(nll), grad.ctypes.data, parts.ctypes.data)
    if st != PWA_OK:
        raise PwaError(st, "pwa_assemble_host")
    return nll.value, grad, parts


def pwa_fumili_hessian(ctx, V, with_norm=True):
    """-> H [2n, 2n] (Fumili-style approximate Hessian of nll, parameter order as in grad)."""
    n = _lib.pwa_n_waves(ctx)
    V = _f64(V, (n, 2))
    H = np.zeros((2 * n, 2 * n))
    _check(ctx, _lib.pwa_fumili_hessian(ctx, V.ctypes.data, H.ctypes.data, 1 if with_norm else 0))
    return H


def pwa_assemble_host_eq2(n_data, L_data, T, M, V):
    """eq. 2 form of step A7 on the host -> (nll2, grad[n,2], parts[2])."""
    V = _f64(V)
    n = V.shape[0]
    T, M = _f64(T, (n, 2)), _f64(M, (n, n, 2))
    nll, g, parts = C.c_double(0.0), np.zeros((n, 2)), np.zeros(2)
    st = _lib.pwa_assemble_host_eq2(n, float(n_data), float(L_data), T.ctypes.data, M.ctypes.data, V.ctypes.data,
                                    C.byref(nll), g.ctypes.data, parts.ctypes.data)
    _check(None, st)
    return nll.value, g, parts


def pwa_grad_to_polar(V, grad):
    V = _f64(V)
    n = V.shape[0]
    grad = _f64(grad, (n, 2))
    out = np.zeros((n, 2))
    _check(None, _lib.pwa_grad_to_polar(n, V.ctypes.data, grad.ctypes.data, out.ctypes.data))
    return out


def pwa_fix_phase_host(V, grad=None, ref_wave=0):
    """-> (V', grad') in the gauge Im V_ref = 0, Re V_ref >= 0 (copies; grad' is None when grad is None)."""
    V = np.array(V, dtype=np.float64, order="C")
    n = V.shape[0]
    if V.shape != (n, 2):
        raise ValueError(f"V must be [n, 2], got {V.shape}")
    g = None
    if grad is not None:
        g = np.array(grad, dtype=np.float64, order="C")
        if g.shape != (n, 2):
            raise ValueError(f"grad must be [{n}, 2], got {g.shape}")
    _check(None, _lib.pwa_fix_phase_host(n, int(ref_wave), V.ctypes.data, None if g is None else g.ctypes.data))
    return V, g


def pwa_polar_to_cartesian(r_phi):
    r_phi = _f64(r_phi)
    n = r_phi.shape[0]
    V = np.zeros((n, 2))
    _check(None, _lib.pwa_polar_to_cartesian(n, r_phi.ctypes.data, V.ctypes.data))
    return V


def pwa_res_grad(ctx, V, n_res=None):
    """-> (d nll / d M_r, d nll / d G_r), [n_res] each; n_res is the wave map's (pwa_n_res), the argument is checked."""
    n = _lib.pwa_n_waves(ctx)
    V = _f64(V, (n, 2))
    have = int(_lib.pwa_n_res(ctx))
    if n_res is not None and int(n_res) != have:
        raise ValueError(f"n_res = {n_res} but the wave map has {have} resonances")
    n_res = have
    dM, dG = np.empty(n_res), np.empty(n_res)
    _check(ctx, _lib.pwa_res_grad(ctx, V.ctypes.data, dM.ctypes.data, dG.ctypes.data))
    return dM, dG


def pwa_nll_grad_floating(ctx, V, mass0, width0, want_status=False):
    """Two-pass floating evaluation -> (nll, grad[n, 2], d nll / d M_r [n_res], d nll / d G_r [n_res], parts[2])."""
    n, nr = _lib.pwa_n_waves(ctx), (_lib.pwa_n_res(ctx),)
    V, m, w = _f64(V, (n, 2)), _f64(mass0, nr), _f64(width0, nr)
    nll = C.c_double(0.0)
    grad, dM, dG, parts = np.empty((n, 2)), np.empty(nr), np.empty(nr), np.empty(2)
    st = _check(ctx, _lib.pwa_nll_grad_floating(ctx, V.ctypes.data, m.ctypes.data, w.ctypes.data, C.byref(nll),
                                                grad.ctypes.data, dM.ctypes.data, dG.ctypes.data, parts.ctypes.data))
    return (nll.value, grad, dM, dG, parts, st) if want_status else (nll.value, grad, dM, dG, parts)


def pwa_minimize_bfgs(ctx, V0, max_iter=200, gtol=1e-6, want_iters=False):
    """-> (V, nll, evaluations, status) (+ iterations when want_iters)."""
    n = _lib.pwa_n_waves(ctx)
    V = _f64(V0, (n, 2)).copy()
    nll = C.c_double(0.0)
    it, ev = C.c_int32(0), C.c_int32(0)
    st = _check(ctx, _lib.pwa_minimize_bfgs(ctx, V.ctypes.data, int(max_iter), float(gtol), C.byref(nll),
                                            C.byref(it), C.byref(ev)))
    return (V, nll.value, ev.value, st, it.value) if want_iters else (V, nll.value, ev.value, st)


def pwa_minimize_bfgs_batch(ctx, V0, max_iter=300, gtol=1e-6):
    V, nll, ev, st, _, _ = pwa_minimize_bfgs_batch_ex(ctx, V0, max_iter, gtol)
    return V, nll, ev, st


def pwa_minimize_bfgs_batch_ex(ctx, V0, max_iter=300, gtol=1e-6):
    """-> (V[K,n,2], nll[K], evaluations, status, iterations[K], why[K] (PWA_FIT_*))."""
    V = _f64(V0).copy()
    K = V.shape[0]
    if V.shape != (K, _lib.pwa_n_waves(ctx), 2):
        raise ValueError("V0 must be [K, n, 2]")
    nll = np.empty(K)
    its, why = np.zeros(K, dtype=np.int32), np.zeros(K, dtype=np.int32)
    ev = C.c_int32(0)
    st = _check(ctx, _lib.pwa_minimize_bfgs_batch_ex(ctx, K, V.ctypes.data, int(max_iter), float(gtol), nll.ctypes.data,
                                                     its.ctypes.data, why.ctypes.data, C.byref(ev)))
    return V, nll, ev.value, st, its, why


def pwa_minimize_bfgs_floating(ctx, V0, mass0, width0, free_res, max_iter=200, gtol=1e-6):
    """-> (V, mass, width, nll, iterations, evaluations, status): BFGS over V and the masses / widths of free_res."""
    n = _lib.pwa_n_waves(ctx)
    return pwa_minimize_bfgs_floating_ex(ctx, V0, mass0, width0, free_res, max_iter, gtol)[:7]


def pwa_minimize_bfgs_floating_ex(ctx, V0, mass0, width0, free_res, max_iter=200, gtol=1e-6):
    """-> (V, mass, width, nll, iterations, evaluations, status, why (PWA_FIT_*))."""
    n = _lib.pwa_n_waves(ctx)
    nr = (_lib.pwa_n_res(ctx),)
    V = _f64(V0, (n, 2)).copy()
    Mr, Gr = _f64(mass0, nr).copy(), _f64(width0, nr).copy()
    fr = np.ascontiguousarray(free_res, dtype=np.int32)
    nll = C.c_double(0.0)
    it, ev, why = C.c_int32(0), C.c_int32(0), C.c_int32(0)
    st = _check(ctx, _lib.pwa_minimize_bfgs_floating_ex(ctx, V.ctypes.data, Mr.ctypes.data, Gr.ctypes.data, len(Mr),
                                                        fr.ctypes.data, len(fr), int(max_iter), float(gtol),
                                                        C.byref(nll), C.byref(it), C.byref(ev), C.byref(why)))
    return V, Mr, Gr, nll.value, it.value, ev.value, st, why.value


def pwa_norm_sums(ctx):
    """-> (G [n, n, 2] = B^H B of this context's MC events, N_gen of this shard)."""
    n = _lib.pwa_n_waves(ctx)
    G, ng = np.empty((n, n, 2)), C.c_int64(0)
    _check(ctx, _lib.pwa_norm_sums(ctx, G.ctypes.data, C.byref(ng)))
    return G, int(ng.value)


def pwa_combine_norm_host(G, n_gen):
    """G [R, n, n, 2], n_gen [R] -> (M [n, n, 2] of all shards, N_gen total); host only."""
    G = _f64(G)
    if G.ndim != 4 or G.shape[1] != G.shape[2] or G.shape[3] != 2:
        raise ValueError("G must be [R, n, n, 2]")
    R, n = G.shape[0], G.shape[1]
    ng = np.ascontiguousarray(n_gen, dtype=np.int64)
    if ng.shape != (R,):
        raise ValueError("n_gen must be [R]")
    M, tot = np.empty((n, n, 2)), C.c_int64(0)
    _check(None, _lib.pwa_combine_norm_host(n, R, G.ctypes.data, ng.ctypes.data, M.ctypes.data, C.byref(tot)))
    return M, int(tot.value)


def pwa_assemble_host_shards(terms, M, V, likelihood=0, n_data=0.0, want_status=False):
    """terms [R, 2 + 2n] (one pwa_data_term_enqueue record per shard) -> (nll, grad[n, 2], parts[2])."""
    V = _f64(V)
    n = V.shape[0]
    terms = _f64(terms)
    R = terms.shape[0]
    if terms.shape != (R, 2 + 2 * n):
        raise ValueError("terms must be [R, 2 + 2n]")
    M = _f64(M, (n, n, 2))
    nll = C.c_double(0.0)
    grad, parts = np.empty((n, 2)), np.empty(2)
    st = _lib.pwa_assemble_host_shards(n, R, terms.ctypes.data, M.ctypes.data, V.ctypes.data, int(likelihood),
                                       float(n_data), C.byref(nll), grad.ctypes.data, parts.ctypes.data)
    _check(None, st)
    return (nll.value, grad, parts, st) if want_status else (nll.value, grad, parts)


def pwa_launch_count(ctx):
    return int(_lib.pwa_launch_count(ctx))


def pwa_sync(ctx):
    _check(ctx, _lib.pwa_sync(ctx))


def pwa_set_option(ctx, key, value):
    _check(ctx, _lib.pwa_set_option(ctx, key.encode(), int(value)))


def pwa_get_option(ctx, key):
    v = C.c_int32(0)
    _check(ctx, _lib.pwa_get_option(ctx, key.encode(), C.byref(v)))
    return int(v.value)


def pwa_microbench(ctx, which, nbytes=0):
    out = C.c_double(0.0)
    _check(ctx, _lib.pwa_microbench(ctx, int(which), int(nbytes), C.byref(out)))
    return out.value


def pwa_n_waves(ctx):
    return int(_lib.pwa_n_waves(ctx))


def pwa_n_res(ctx):
    return int(_lib.pwa_n_res(ctx))


def pwa_storage(ctx):
    return int(_lib.pwa_storage(ctx))


def pwa_n_events(ctx, which):
    return int(_lib.pwa_n_events(ctx, int(which)))


def pwa_last_error(ctx):
    return _lib.pwa_last_error(ctx).decode()


def pwa_status_string(status):
    return _status_name(status)
