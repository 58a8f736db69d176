"""ctypes front-end of the CPU oracle (oracle/pwa_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It imports
nothing from paper_1108_5882_b200 and the CUDA library imports nothing from here.

Array conventions (same as include/pwa.h so both sides get the identical bit patterns):
amplitudes are numpy arrays of shape [N, n, 2] (re, im), dtype float64 or float32;
V is [n, 2] float64; M is [n, n, 2] float64 with M[a, b] = M_ab.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        _lib.pwa_oracle_data_term.restype = C.c_int64
        _lib.pwa_oracle_nll_grad.restype = C.c_int64
        _lib.pwa_oracle_nll_grad_batch.restype = C.c_int64
        _lib.pwa_oracle_intensity_eq1.restype = C.c_double
        _lib.pwa_oracle_threads.restype = C.c_int
    return _lib


def threads() -> int:
    return int(lib().pwa_oracle_threads())


def set_threads(t: int) -> None:
    lib().pwa_oracle_set_threads(C.c_int(int(t)))


def _amp(x):
    x = np.ascontiguousarray(x)
    if x.dtype == np.complex128:
        x = x.view(np.float64).reshape(x.shape + (2,))
    elif x.dtype == np.complex64:
        x = x.view(np.float32).reshape(x.shape + (2,))
    if x.dtype == np.float64:
        dt = 0
    elif x.dtype == np.float32:
        dt = 1
    else:
        raise TypeError("amplitudes must be float64/float32 [N, n, 2]")
    if x.ndim != 3 or x.shape[2] != 2:
        raise ValueError("amplitudes must have shape [N, n, 2]")
    return x, dt


def _f64(x, shape=None):
    x = np.ascontiguousarray(x, dtype=np.float64)
    if shape is not None and tuple(x.shape) != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {x.shape}")
    return x


def _p(x):
    return x.ctypes.data_as(C.c_void_p)


def _i32(x):
    return np.ascontiguousarray(x, dtype=np.int32)


def bw(m, M, G):
    out = np.zeros(2)
    lib().pwa_oracle_bw(C.c_double(m), C.c_double(M), C.c_double(G), _p(out))
    return complex(out[0], out[1])


def bw_deriv(m, M, G):
    dM, dG = np.zeros(2), np.zeros(2)
    lib().pwa_oracle_bw_deriv(C.c_double(m), C.c_double(M), C.c_double(G), _p(dM), _p(dG))
    return complex(dM[0], dM[1]), complex(dG[0], dG[1])


def expand_factored(mass, Z, res_of_wave, ang_of_wave, Mr, Gr):
    """A[i, a] = BW(mass_i; Mr[r(a)], Gr[r(a)]) * Z[i, s(a)]  ->  float64 [N, n, 2]."""
    Z, dtZ = _amp(Z)
    mass = _f64(mass)
    N, n_ang = Z.shape[0], Z.shape[1]
    row, aow = _i32(res_of_wave), _i32(ang_of_wave)
    n = row.shape[0]
    Mr, Gr = _f64(Mr), _f64(Gr)
    out = np.empty((N, n, 2))
    lib().pwa_oracle_expand_factored(_p(mass), _p(Z), C.c_int(dtZ), C.c_int(n_ang),
                                     C.c_int64(N), C.c_int(n), _p(row), _p(aow),
                                     _p(Mr), _p(Gr), _p(out))
    return out


def data_term(A, V):
    """-> (L_data, T[n,2], n_nonfinite)."""
    A, dt = _amp(A)
    N, n = A.shape[0], A.shape[1]
    V = _f64(V, (n, 2))
    L = C.c_double(0.0)
    T = np.zeros((n, 2))
    bad = lib().pwa_oracle_data_term(_p(A), C.c_int(dt), C.c_int64(N), C.c_int(n), _p(V),
                                     C.byref(L), _p(T))
    return L.value, T, int(bad)


def data_term_w(A, V, w):
    """Weighted data term: L = sum_i w_i ln I_i, T_a = sum_i w_i A_ia / S_i -> (L, T[n,2], n_nonfinite)."""
    A, dt = _amp(A)
    N, n = A.shape[0], A.shape[1]
    V, w = _f64(V, (n, 2)), _f64(w, (N,))
    L = C.c_double(0.0)
    T = np.zeros((n, 2))
    lib().pwa_oracle_data_term_w.restype = C.c_int64
    bad = lib().pwa_oracle_data_term_w(_p(A), C.c_int(dt), C.c_int64(N), C.c_int(n), _p(V), _p(w), C.byref(L), _p(T))
    return L.value, T, int(bad)


def norm_matrix_w(B, n_gen, w):
    """Weighted normalisation matrix M_ab = (1/N_gen) sum_j w_j conj(B_ja) B_jb."""
    B, dt = _amp(B)
    N, n = B.shape[0], B.shape[1]
    w = _f64(w, (N,))
    M = np.zeros((n, n, 2))
    lib().pwa_oracle_norm_block_w(_p(B), C.c_int(dt), C.c_int64(N), C.c_int(n), C.c_int64(int(n_gen)), _p(w),
                                  C.c_int(0), C.c_int(n), C.c_int(0), C.c_int(n), _p(M))
    return M


def norm_matrix(B, n_gen):
    B, dt = _amp(B)
    N, n = B.shape[0], B.shape[1]
    M = np.zeros((n, n, 2))
    lib().pwa_oracle_norm_matrix(_p(B), C.c_int(dt), C.c_int64(N), C.c_int(n),
                                 C.c_int64(int(n_gen)), _p(M))
    return M


def norm_block(B, n_gen, a0, a1, b0, b1):
    """Entries M[a0:a1, b0:b1] only (others zero); for sampled checks at full size."""
    B, dt = _amp(B)
    N, n = B.shape[0], B.shape[1]
    M = np.zeros((n, n, 2))
    lib().pwa_oracle_norm_block(_p(B), C.c_int(dt), C.c_int64(N), C.c_int(n),
                                C.c_int64(int(n_gen)), C.c_int(a0), C.c_int(a1),
                                C.c_int(b0), C.c_int(b1), _p(M))
    return M


def norm_explicit(B, n_gen, V):
    """-> (Norm' = (1/N_gen) sum_j |S_j|^2,  gN'[n,2] = (2/N_gen) sum_j conj(B_ja) S_j)."""
    B, dt = _amp(B)
    N, n = B.shape[0], B.shape[1]
    V = _f64(V, (n, 2))
    nv = C.c_double(0.0)
    g = np.zeros((n, 2))
    lib().pwa_oracle_norm_explicit(_p(B), C.c_int(dt), C.c_int64(N), C.c_int(n),
                                   C.c_int64(int(n_gen)), _p(V), C.byref(nv), _p(g))
    return nv.value, g


def assemble(L, T, M, V):
    """-> (nll, grad[n,2], parts[2])."""
    n = np.asarray(V).shape[0]
    T, M, V = _f64(T, (n, 2)), _f64(M, (n, n, 2)), _f64(V, (n, 2))
    nll = C.c_double(0.0)
    g = np.zeros((n, 2))
    parts = np.zeros(2)
    lib().pwa_oracle_assemble(C.c_int(n), C.c_double(L), _p(T), _p(M), _p(V),
                              C.byref(nll), _p(g), _p(parts))
    return nll.value, g, parts


def assemble_eq2(n_data, L, T, M, V):
    """eq. 2 (normalised) form -> (nll2, grad[n,2], parts[2])."""
    n = np.asarray(V).shape[0]
    T, M, V = _f64(T, (n, 2)), _f64(M, (n, n, 2)), _f64(V, (n, 2))
    nll = C.c_double(0.0)
    g = np.zeros((n, 2))
    parts = np.zeros(2)
    lib().pwa_oracle_assemble_eq2(C.c_int(n), C.c_double(float(n_data)), C.c_double(L), _p(T), _p(M), _p(V),
                                  C.byref(nll), _p(g), _p(parts))
    return nll.value, g, parts


def nll_grad_eq2(A, M, V):
    """eq. 2 form from the data term + M -> (nll2, grad[n,2], parts[2])."""
    L, T, bad = data_term(A, V)
    return assemble_eq2(np.asarray(A).shape[0], L, T, M, V)


def grad_polar(V, grad):
    """Cartesian gradient [n,2] -> (d/dr, d/dphi) [n,2] at V = r exp(i phi)."""
    n = np.asarray(V).shape[0]
    V, grad = _f64(V, (n, 2)), _f64(grad, (n, 2))
    out = np.zeros((n, 2))
    lib().pwa_oracle_grad_polar(C.c_int(n), _p(V), _p(grad), _p(out))
    return out


def fix_phase(V, grad=None, ref=0):
    """Fixed-phase gauge: -> (V', grad') with wave `ref` real and non-negative, the gradient turned by the same angle and its
    d/d Im V_ref component dropped (0).  grad=None -> (V', None)."""
    n = np.asarray(V).shape[0]
    V2 = _f64(V, (n, 2)).copy()
    g2 = None if grad is None else _f64(grad, (n, 2)).copy()
    lib().pwa_oracle_fix_phase(C.c_int(n), C.c_int(int(ref)), _p(V2), None if g2 is None else _p(g2))
    return V2, g2


def fumili(A, V, M=None):
    """Fumili-style approximate Hessian [2n, 2n] in the (x_0, y_0, x_1, ...) order; M=None -> data part only."""
    A, dt = _amp(A)
    N, n = A.shape[0], A.shape[1]
    V = _f64(V, (n, 2))
    H = np.zeros((2 * n, 2 * n))
    Mp = _p(_f64(M, (n, n, 2))) if M is not None else None
    lib().pwa_oracle_fumili(_p(A), C.c_int(dt), C.c_int64(N), C.c_int(n), _p(V), Mp, _p(H))
    return H


def fumili_rows(A, V, p0, p1):
    """Rows p0:p1 of the data part of the Fumili matrix (other rows zero); for sampled checks at full size."""
    A, dt = _amp(A)
    N, n = A.shape[0], A.shape[1]
    V = _f64(V, (n, 2))
    H = np.zeros((2 * n, 2 * n))
    lib().pwa_oracle_fumili_rows(_p(A), C.c_int(dt), C.c_int64(N), C.c_int(n), _p(V), C.c_int(p0), C.c_int(p1), _p(H))
    return H


def nll_grad(A, M, V):
    """-> (nll, grad[n,2], parts[2], n_nonfinite)."""
    A, dt = _amp(A)
    N, n = A.shape[0], A.shape[1]
    M, V = _f64(M, (n, n, 2)), _f64(V, (n, 2))
    nll = C.c_double(0.0)
    g = np.zeros((n, 2))
    parts = np.zeros(2)
    bad = lib().pwa_oracle_nll_grad(_p(A), C.c_int(dt), C.c_int64(N), C.c_int(n), _p(M), _p(V),
                                    C.byref(nll), _p(g), _p(parts))
    return nll.value, g, parts, int(bad)


def nll_grad_batch(A, M, Vk):
    """Vk [K, n, 2] -> (nll[K], grad[K,n,2], parts[K,2], n_nonfinite)."""
    A, dt = _amp(A)
    N, n = A.shape[0], A.shape[1]
    Vk = _f64(Vk)
    K = Vk.shape[0]
    M = _f64(M, (n, n, 2))
    nll = np.zeros(K)
    g = np.zeros((K, n, 2))
    parts = np.zeros((K, 2))
    bad = lib().pwa_oracle_nll_grad_batch(_p(A), C.c_int(dt), C.c_int64(N), C.c_int(n), _p(M),
                                          C.c_int(K), _p(Vk), _p(nll), _p(g), _p(parts))
    return nll, g, parts, int(bad)


def intensity_eq1(Arow, V):
    Arow, V = _f64(Arow), _f64(V)
    return float(lib().pwa_oracle_intensity_eq1(_p(Arow), C.c_int(V.shape[0]), _p(V)))


def intensity_eq3(Arow, V):
    Arow, V = _f64(Arow), _f64(V)
    out = np.zeros(2)
    lib().pwa_oracle_intensity_eq3(_p(Arow), C.c_int(V.shape[0]), _p(V), _p(out))
    return complex(out[0], out[1])


def res_grad(mass, Z, res_of_wave, ang_of_wave, Mr, Gr, V, mode, n_gen=1):
    """Gradient w.r.t. (M_r, G_r): mode 0 -> d L_data, mode 1 -> d Norm.  -> (dM[n_res], dG[n_res])."""
    Z, dtZ = _amp(Z)
    mass = _f64(mass)
    N, n_ang = Z.shape[0], Z.shape[1]
    row, aow = _i32(res_of_wave), _i32(ang_of_wave)
    n = row.shape[0]
    Mr, Gr = _f64(Mr), _f64(Gr)
    n_res = Mr.shape[0]
    V = _f64(V, (n, 2))
    dM, dG = np.zeros(n_res), np.zeros(n_res)
    lib().pwa_oracle_res_grad(_p(mass), _p(Z), C.c_int(dtZ), C.c_int(n_ang), C.c_int64(N),
                              C.c_int(n), C.c_int(n_res), _p(row), _p(aow), _p(Mr), _p(Gr),
                              _p(V), C.c_int(mode), C.c_int64(int(n_gen)), _p(dM), _p(dG))
    return dM, dG
