"""Thin Python binding of libcc_b200.so (include/cc_b200.h): argument marshalling only.

Every function has the name and argument order of its C entry point; tensors are passed as
`data_ptr()`s.  PyTorch is used for device memory and streams, nothing else.  There is no CPU
fallback: importing this module fails loudly when the library has not been built
(`python -m paper_1409_2065_b200.build`), and every compute call fails with CC_ECUDA without a GPU.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcc_b200.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1409_2065_b200.build` "
                      "(there is no CPU fallback)")
_lib = ctypes.CDLL(LIB_PATH)

CC_OK, CC_EINVAL, CC_EGRAPH, CC_EMASK, CC_ENOMEM, CC_ECUDA, CC_ESTATE, CC_ENOCONV = 0, -1, -2, -3, -4, -5, -6, -7

SYMBOLS = ("cc_default_params", "cc_knn_weights", "cc_knn_weights_composite", "cc_knn_weights_geodesic", "cc_dense_weights", "cc_dense_weights_noalloc", "cc_graph_components",
           "cc_smallest_connected_k", "cc_free_graph", "cc_create", "cc_solve", "cc_solve_continuation", "cc_path", "cc_path_continuation",
           "cc_get_U", "cc_get_projection", "cc_principal_components", "cc_clusters", "cc_get_history", "cc_get_stats", "cc_get_profile", "cc_reset_profile",
           "cc_reset", "cc_get_counts",
           "cc_last_error", "cc_destroy")


class cc_params(ctypes.Structure):
    _fields_ = [("rho_scale", ctypes.c_double), ("rho_abs", ctypes.c_double), ("kappa", ctypes.c_double),
                ("eps_abs", ctypes.c_double), ("proj_tol", ctypes.c_double), ("proj_maxit", ctypes.c_int32),
                ("min_it", ctypes.c_int32), ("dense", ctypes.c_int32), ("use_graph", ctypes.c_int32),
                ("hist_cap", ctypes.c_int32), ("max_snapshots", ctypes.c_int32), ("reserved", ctypes.c_int32)]


_vp, _i64, _i32, _dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
_P = ctypes.POINTER
_lib.cc_default_params.argtypes = [_P(cc_params)]
_lib.cc_knn_weights.argtypes = [_i64, _i64, _vp, _vp, _i32, ctypes.c_float, _i32, _P(_vp), _P(_vp), _P(_vp),
                                _P(_i64), _vp]
_lib.cc_knn_weights_composite.argtypes = [_i64, _i64, _vp, _vp, _i32, _vp, _P(ctypes.c_float), ctypes.c_float, _i32,
                                          ctypes.c_float, _i32, _P(_vp), _P(_vp), _P(_vp), _P(_i64), _vp]
_lib.cc_knn_weights_geodesic.argtypes = [_i64, _i64, _vp, _vp, _vp, ctypes.c_float, ctypes.c_float, _i32,
                                         ctypes.c_float, _i32, _P(_vp), _P(_vp), _P(_vp), _P(_i64), _vp]
_lib.cc_dense_weights.argtypes = [_i64, _i64, _vp, _vp, ctypes.c_float, _i32, _vp, _vp]
_lib.cc_dense_weights_noalloc.argtypes = [_i64, _i64, _vp, _vp, ctypes.c_float, _vp, _vp]
_lib.cc_graph_components.argtypes = [_i64, _vp, _vp, _vp, _P(_i32), _vp]
_lib.cc_smallest_connected_k.argtypes = [_i64, _i64, _vp, _vp, _i32, _P(_i32), _vp]
_lib.cc_free_graph.argtypes = [_vp, _vp, _vp]
_lib.cc_free_graph.restype = None
_lib.cc_create.argtypes = [_P(_vp), _i64, _i64, _vp, _vp, _vp, _vp, _vp, _P(cc_params), _vp]
_lib.cc_solve.argtypes = [_vp, _dbl, _dbl, _i32, _P(_i32), _P(_dbl)]
_lib.cc_solve_continuation.argtypes = [_vp, _dbl, _dbl, _dbl, _i32, _dbl, _i32, _P(_i32), _i32, _P(_i32), _P(_dbl)]
_lib.cc_path.argtypes = [_vp, _P(_dbl), _i32, _dbl, _i32, _P(_i32), _P(_dbl)]
_lib.cc_path_continuation.argtypes = [_vp, _P(_dbl), _i32, _dbl, _dbl, _i32, _dbl, _i32, _P(_i32), _P(_dbl)]
_lib.cc_get_U.argtypes = [_vp, _i32, _vp, _i32]
_lib.cc_clusters.argtypes = [_vp, _i32, _vp, _i32, _P(_i32)]
_lib.cc_get_projection.argtypes = [_vp, _i32, _vp, _i32, _vp, _i32]
_lib.cc_principal_components.argtypes = [_vp, _i32, _i32, _dbl, _vp, _i32, _vp, _vp, _P(_i32)]
_lib.cc_get_history.argtypes = [_vp, _vp, _vp, _i32, _P(_i32)]
_lib.cc_get_stats.argtypes = [_vp, _P(_dbl), _P(_dbl), _P(_i64), _P(_dbl), _P(_dbl)]
_lib.cc_reset.argtypes = [_vp]
_lib.cc_get_profile.argtypes = [_vp, _vp, _vp]
_lib.cc_reset_profile.argtypes = [_vp]
_lib.cc_get_counts.argtypes = [_vp, _P(_i64), _P(_i64), _P(_i64)]
_lib.cc_last_error.argtypes = [_vp]
_lib.cc_last_error.restype = ctypes.c_char_p
_lib.cc_destroy.argtypes = [_vp]
_lib.cc_destroy.restype = None


class CCError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libcc_b200 error {code}: {msg}")
        self.code = code


def _check(rc, h=None, allow=()):
    if rc != CC_OK and rc not in allow:
        raise CCError(rc, _lib.cc_last_error(h).decode())
    return rc


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream():
    if not torch.cuda.is_available():   # let the library report CC_ECUDA itself
        return None
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def cc_default_params(**overrides) -> cc_params:
    prm = cc_params()
    _check(_lib.cc_default_params(ctypes.byref(prm)))
    for k, v in overrides.items():
        if not hasattr(prm, k):
            raise AttributeError(k)
        setattr(prm, k, v)
    return prm


def cc_create(n, p, X, mask, rowptr, col, w, prm=None):
    """Device tensors: X fp32 (n,p), mask uint8 (n,p) or None, rowptr int64, col int32, w fp32
    (or the (n,n) matrix when prm.dense = 1).  Returns the opaque handle."""
    h = ctypes.c_void_p()
    rc = _lib.cc_create(ctypes.byref(h), n, p, _ptr(X), _ptr(mask), _ptr(rowptr), _ptr(col), _ptr(w),
                        ctypes.byref(prm) if prm is not None else None, _stream())
    _check(rc)
    return h


def cc_solve(h, gamma, tol, maxit, allow_noconv=False):
    it, phi = _i32(0), _dbl(0.0)
    rc = _check(_lib.cc_solve(h, gamma, tol, maxit, ctypes.byref(it), ctypes.byref(phi)), h,
                allow=(CC_ENOCONV,) if allow_noconv else ())
    return it.value, phi.value, rc


def cc_path(h, gammas, tol, maxit):
    g = (ctypes.c_double * len(gammas))(*[float(x) for x in gammas])
    its = (ctypes.c_int32 * len(gammas))()
    phis = (ctypes.c_double * len(gammas))()
    _check(_lib.cc_path(h, g, len(gammas), tol, maxit, its, phis), h)
    return list(its), list(phis)


def cc_path_continuation(h, gammas, kappa_start, factor, stage_maxit, tol, maxit):
    g = (ctypes.c_double * len(gammas))(*[float(x) for x in gammas])
    its = (ctypes.c_int32 * len(gammas))()
    phis = (ctypes.c_double * len(gammas))()
    _check(_lib.cc_path_continuation(h, g, len(gammas), kappa_start, factor, stage_maxit, tol, maxit, its, phis), h,
           allow=(CC_ENOCONV,))
    return list(its), list(phis)


def cc_solve_continuation(h, gamma, kappa_start, factor, stage_maxit, tol, maxit):
    """Returns (stage_iters list, phi of the last stage, return code CC_OK / CC_ENOCONV)."""
    cap = 64
    its, ns, phi = (_i32 * cap)(), _i32(0), _dbl(0.0)
    rc = _lib.cc_solve_continuation(h, gamma, kappa_start, factor, stage_maxit, tol, maxit, its, cap, ctypes.byref(ns),
                                    ctypes.byref(phi))
    if rc != CC_ENOCONV:
        _check(rc, h)
    return list(its[:min(ns.value, cap)]), phi.value, rc


def cc_get_U(h, gamma_index, U_out):
    """U_out: fp32 (n,p) contiguous torch tensor, on the device or on the host."""
    _check(_lib.cc_get_U(h, gamma_index, _ptr(U_out), 1 if U_out.is_cuda else 0), h)
    return U_out


def cc_get_projection(h, gamma_index, P, out):
    """P: fp32 (p,q) device tensor; out: fp32 (n,q) tensor on the device or the host."""
    _check(_lib.cc_get_projection(h, gamma_index, _ptr(P), P.shape[1], _ptr(out), 1 if out.is_cuda else 0), h)
    return out


def cc_principal_components(h, P_out, maxit=300, tol=1e-6):
    """P_out: fp32 (p,q) contiguous torch tensor (device or host).  Returns (P_out, variances[q], residuals[q], steps)."""
    q = P_out.shape[1]
    var, res, its = (_dbl * q)(), (_dbl * q)(), _i32(0)
    _check(_lib.cc_principal_components(h, q, maxit, tol, _ptr(P_out), 1 if P_out.is_cuda else 0, var, res,
                                        ctypes.byref(its)), h)
    return P_out, list(var), list(res), its.value


def cc_clusters(h, gamma_index, labels_out):
    k = _i32(0)
    _check(_lib.cc_clusters(h, gamma_index, _ptr(labels_out), 1 if labels_out.is_cuda else 0, ctypes.byref(k)), h)
    return labels_out, k.value


def cc_get_history(h, cap=4096):
    phi = np.zeros(cap)
    d = np.zeros(cap)
    cnt = _i32(0)
    _check(_lib.cc_get_history(h, phi.ctypes.data_as(_vp), d.ctypes.data_as(_vp), cap, ctypes.byref(cnt)), h)
    return phi[:cnt.value].copy(), d[:cnt.value].copy()


def cc_get_stats(h, f_gamma=False, min_margin=False):
    rho, eps, fg, mm = _dbl(0), _dbl(0), _dbl(0), _dbl(0)
    pi = _i64(0)
    _check(_lib.cc_get_stats(h, ctypes.byref(rho), ctypes.byref(eps), ctypes.byref(pi),
                             ctypes.byref(fg) if f_gamma else None, ctypes.byref(mm) if min_margin else None), h)
    return {"rho": rho.value, "eps": eps.value, "proj_iters": pi.value,
            "f_gamma": fg.value if f_gamma else None, "min_margin": mm.value if min_margin else None}


KERNEL_NAMES = ("k_rhs", "k_cg_spmv", "k_cg_update", "k_norm", "k_update", "kd_proj", "kd_pairs", "kd_edges")


def cc_get_profile(h):
    ns = np.zeros(8)
    calls = np.zeros(8, dtype=np.int64)
    _check(_lib.cc_get_profile(h, ns.ctypes.data_as(_vp), calls.ctypes.data_as(_vp)), h)
    return {k: {"ns": float(ns[i]), "calls": int(calls[i])} for i, k in enumerate(KERNEL_NAMES)}


def cc_reset_profile(h):
    _check(_lib.cc_reset_profile(h), h)


def cc_reset(h):
    _check(_lib.cc_reset(h), h)


def cc_get_counts(h):
    a, b, c = _i64(0), _i64(0), _i64(0)
    _check(_lib.cc_get_counts(h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), h)
    return {"n_pairs": a.value, "nnz": b.value, "launches": c.value}


def cc_last_error(h=None) -> str:
    return _lib.cc_last_error(h).decode()


def cc_destroy(h):
    _lib.cc_destroy(h)


def cc_dense_weights(n, p, X, mask, phi, normalize=False):
    """All-pairs Gaussian weights as an (n, n) fp32 device tensor (for prm.dense = 1)."""
    W = torch.empty(n, n, dtype=torch.float32, device=X.device)
    _check(_lib.cc_dense_weights(n, p, _ptr(X), _ptr(mask), phi, 1 if normalize else 0, _ptr(W), _stream()))
    return W


def cc_dense_weights_noalloc(n, p, X, mask, phi, W_out):
    """cc_dense_weights without any allocation: W_out is a caller-made (n, n) fp32 device tensor (see cc_b200.h)."""
    _check(_lib.cc_dense_weights_noalloc(n, p, _ptr(X), _ptr(mask), phi, _ptr(W_out), _stream()))
    return W_out


def cc_graph_components(n, rowptr, col, labels_out):
    k = _i32(0)
    _check(_lib.cc_graph_components(n, _ptr(rowptr), _ptr(col), _ptr(labels_out), ctypes.byref(k), _stream()))
    return labels_out, k.value


def cc_smallest_connected_k(n, p, X, mask, kmax):
    k = _i32(0)
    _check(_lib.cc_smallest_connected_k(n, p, _ptr(X), _ptr(mask), kmax, ctypes.byref(k), _stream()))
    return k.value


class _DevArray:
    """Zero-copy view of a library-owned device array (CUDA array interface) for torch.as_tensor."""

    def __init__(self, ptr, count, typestr):
        self.__cuda_array_interface__ = {"shape": (count,), "typestr": typestr, "data": (ptr, False), "version": 3}


def _wrap(ptr, count, typestr, dev):
    if count == 0:
        return torch.empty(0, dtype={"<i8": torch.int64, "<i4": torch.int32, "<f4": torch.float32}[typestr], device=dev)
    return torch.as_tensor(_DevArray(ptr, count, typestr), device=dev)


def cc_knn_weights(n, p, X, mask, k, phi, normalize=False, Y=None, period=None, alpha=1.0, geodesic_radius=None):
    """Returns (rowptr int64, col int32, w fp32) as torch device tensors (copies; the library's
    arrays are released with cc_free_graph before returning).  With Y (n,q device tensor): the composite
    distance of eq. 9 (cc_knn_weights_composite), period = q floats or None; with geodesic_radius, Y is
    (longitude, latitude) in degrees and the side distance is the great circle (cc_knn_weights_geodesic)."""
    rp, cl, ww = _vp(), _vp(), _vp()
    nnz = _i64(0)
    if Y is None:
        _check(_lib.cc_knn_weights(n, p, _ptr(X), _ptr(mask), k, phi, 1 if normalize else 0, ctypes.byref(rp),
                                   ctypes.byref(cl), ctypes.byref(ww), ctypes.byref(nnz), _stream()))
    elif geodesic_radius is not None:
        if Y.dim() != 2 or Y.shape[1] != 2:
            raise CCError(CC_EINVAL, "cc_knn_weights: geodesic side coordinates must be (n, 2) = (longitude, latitude)")
        _check(_lib.cc_knn_weights_geodesic(n, p, _ptr(X), _ptr(mask), _ptr(Y), float(geodesic_radius), alpha, k, phi,
                                            1 if normalize else 0, ctypes.byref(rp), ctypes.byref(cl), ctypes.byref(ww),
                                            ctypes.byref(nnz), _stream()))
    else:
        q = Y.shape[1]
        per = None if period is None else (ctypes.c_float * q)(*[float(x) for x in period])
        _check(_lib.cc_knn_weights_composite(n, p, _ptr(X), _ptr(mask), q, _ptr(Y), per, alpha, k, phi,
                                             1 if normalize else 0, ctypes.byref(rp), ctypes.byref(cl), ctypes.byref(ww),
                                             ctypes.byref(nnz), _stream()))
    dev = X.device
    rowptr = _wrap(rp.value, n + 1, "<i8", dev).clone()
    col = _wrap(cl.value, nnz.value, "<i4", dev).clone()
    w = _wrap(ww.value, nnz.value, "<f4", dev).clone()
    torch.cuda.synchronize(dev)
    _lib.cc_free_graph(rp, cl, ww)
    return rowptr, col, w
