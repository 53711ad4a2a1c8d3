"""Python face of the fp64 CPU oracle (oracle/cc_oracle.c) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  Nothing here imports or is imported by paper_1409_2065_b200 (the CUDA path).

Everything is fp64.  Each function cites the PAPER.md passage (or DESIGN.md reading Sx) it follows.
The numpy parts are plain definitions (weights eq. 8, default constants, objective eq. 1/6).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cc_oracle.c")
_LIB = os.path.join(_HERE, "libcc_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile cc_oracle.c with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _L():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        i64, i32, dbl, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        L.orc_num_threads.restype = i32
        L.orc_set_threads.argtypes = [i32]
        L.orc_row_dist2.argtypes = [i64, i64, vp, vp, i64, vp]
        L.orc_knn.argtypes = [i64, i64, vp, vp, i32, i64, vp, vp, vp]
        L.orc_knn.restype = i32
        L.orc_project.argtypes = [i64, i64, i64, vp, vp, vp, vp, i32, dbl, i64, vp]
        L.orc_project.restype = i64
        L.orc_mm.argtypes = [i64, i64, vp, vp, i64, vp, vp, vp, dbl, dbl, dbl, i32, dbl, i32, i32, dbl, i64,
                             vp, vp, vp, vp, vp, vp]
        L.orc_mm.restype = i32
        L.orc_labels.argtypes = [i64, i64, i64, vp, vp, vp, vp]
        L.orc_labels.restype = i64
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def num_threads() -> int:
    return int(_L().orc_num_threads())


def set_threads(t: int) -> None:
    _L().orc_set_threads(int(t))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _u8(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.uint8)


# ----------------------------------------------------------------------------- weights (a0)
def row_dist2(X, mask, i: int) -> np.ndarray:
    """Squared distances from row i to all rows (masked rule: reading S11)."""
    X = _f64(X)
    mask = _u8(mask)
    n, p = X.shape
    out = np.empty(n)
    _L().orc_row_dist2(n, p, _p(X), _p(mask), int(i), _p(out))
    return out


def knn(X, mask, k: int, rows=None):
    """k nearest neighbours by brute force (S9: self excluded, ties -> smaller index)."""
    X = _f64(X)
    mask = _u8(mask)
    n, p = X.shape
    rows_a = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    nr = n if rows_a is None else rows_a.size
    nbr = np.empty((nr, k), dtype=np.int32)
    d2 = np.empty((nr, k))
    rc = _L().orc_knn(n, p, _p(X), _p(mask), int(k), nr, _p(rows_a), _p(nbr), _p(d2))
    if rc:
        raise ValueError("orc_knn: need 1 <= k <= n-1")
    return nbr, d2


def pair_dist2(X, mask, i, j) -> np.ndarray:
    """Squared distances of the listed pairs, same rule as the C code (plain definition in numpy)."""
    X = _f64(X)
    out = np.empty(len(i))
    step = max(1, (1 << 22) // max(1, X.shape[1]))
    for s in range(0, len(i), step):
        ii, jj = i[s:s + step], j[s:s + step]
        df = X[ii] - X[jj]
        if mask is None:
            out[s:s + step] = np.einsum("ij,ij->i", df, df)
        else:
            co = (mask[ii] != 0) & (mask[jj] != 0)
            cnt = co.sum(axis=1)
            ss = np.einsum("ij,ij->i", df * co, df * co)
            with np.errstate(divide="ignore", invalid="ignore"):
                out[s:s + step] = np.where(cnt > 0, ss * X.shape[1] / np.maximum(cnt, 1), np.inf)
    return out


def knn_graph(X, mask, k: int, phi: float, normalize: bool = False):
    """Weights of eq. 8: i~j iff j among the k nearest of i OR vice versa;
    w_ij = exp(-phi d_ij^2); optional normalisation to sum 1 over pairs i<j (S8).
    Returns (ei, ej, w, d2) with ei<ej, sorted by (ei, ej)."""
    n = X.shape[0]
    nbr, d2 = knn(X, mask, k)
    i = np.repeat(np.arange(n, dtype=np.int64), k)
    j = nbr.reshape(-1).astype(np.int64)
    lo, hi = np.minimum(i, j), np.maximum(i, j)
    key = lo * n + hi
    key_u, first = np.unique(key, return_index=True)
    ei = (key_u // n).astype(np.int32)
    ej = (key_u % n).astype(np.int32)
    dd = d2.reshape(-1)[first]
    w = np.exp(-phi * dd)
    if normalize:
        w = w / w.sum()
    return ei, ej, w, dd


def side_dist(Y, period, i: int) -> np.ndarray:
    """||y_i - y_j|| for all j, the components of the difference "computed in modulo arithmetic" (PAPER.md L137,
    below eq. 9): with a period P_c > 0 coordinate c's difference is wrapped to [-P_c/2, P_c/2] [reading S27]."""
    Y = _f64(Y)
    df = Y[i][None, :] - Y
    if period is not None:
        P = np.asarray(period, dtype=np.float64)
        wrap = P > 0
        df[:, wrap] = df[:, wrap] - P[wrap] * np.round(df[:, wrap] / P[wrap])
    return np.sqrt((df * df).sum(axis=1))


def geodesic_dist(LL, radius: float, i: int) -> np.ndarray:
    """"An even better alternative replaces ||y_i - y_j|| by the geodesic distance between i and j"
    [reading S28]: y = (longitude, latitude) in degrees, the geodesic is the great circle on a sphere of the given
    radius, d_ij = radius * theta_ij with the central angle from the haversine formula
        hav(theta) = sin^2(dlat/2) + cos(lat_i) cos(lat_j) sin^2(dlon/2),   theta = 2 atan2(sqrt(hav), sqrt(1 - hav)).
    Returns d_ij for all j."""
    LL = _f64(LL)
    lon, lat = np.deg2rad(LL[:, 0]), np.deg2rad(LL[:, 1])
    sl = np.sin((lat - lat[i]) / 2.0)
    so = np.sin((lon - lon[i]) / 2.0)
    hav = sl * sl + np.cos(lat[i]) * np.cos(lat) * so * so
    hav = np.clip(hav, 0.0, 1.0)
    return radius * 2.0 * np.arctan2(np.sqrt(hav), np.sqrt(1.0 - hav))


def composite_knn_graph(X, mask, Y, period, alpha: float, k: int, phi: float, normalize: bool = False,
                        geodesic_radius=None):
    """Eq. 9: d_ij = alpha ||x_i - x_j|| + (1 - alpha) ||y_i - y_j||, then eq. 8 with this d:
    i~j iff j is among the k nearest of i by d OR vice versa (S9: self excluded, ties -> smaller index),
    w_ij = exp(-phi d_ij^2), optional normalisation (S8).  ||x_i - x_j|| is the square root of row_dist2 (masked
    rule S11).  With geodesic_radius, ||y_i - y_j|| is replaced by geodesic_dist (L137, S28; `period` is unused).
    Returns (ei, ej, w, d) with ei<ej sorted by (ei, ej)."""
    n = X.shape[0]
    pairs = {}
    for i in range(n):
        dx = np.sqrt(row_dist2(X, mask, i))
        dx[i] = 0.0                      # row_dist2 marks the row itself with inf; it is excluded below
        dy = side_dist(Y, period, i) if geodesic_radius is None else geodesic_dist(Y, geodesic_radius, i)
        d = alpha * dx + (1.0 - alpha) * dy
        d[i] = np.inf
        order = np.lexsort((np.arange(n), d))[:k]
        for j in order:
            pairs[(min(i, int(j)), max(i, int(j)))] = d[j]
    keys = sorted(pairs)
    ei = np.array([a for a, _ in keys], dtype=np.int32)
    ej = np.array([b for _, b in keys], dtype=np.int32)
    dd = np.array([pairs[key] for key in keys])
    w = np.exp(-phi * dd * dd)
    if normalize:
        w = w / w.sum()
    return ei, ej, w, dd


def complete_graph(X, mask, phi: float, normalize: bool = False):
    """All pairs i<j with Gaussian weights (eq. 8 with k = n-1)."""
    n = X.shape[0]
    ei, ej = np.triu_indices(n, k=1)
    dd = pair_dist2(X, mask, ei, ej)
    w = np.exp(-phi * dd)
    if normalize:
        w = w / w.sum()
    return ei.astype(np.int32), ej.astype(np.int32), w, dd


def to_csr(n: int, ei, ej, w):
    """Symmetric CSR (both directions) of the pair list: rowptr int64, col int32 (sorted), w."""
    r = np.concatenate([ei, ej]).astype(np.int64)
    c = np.concatenate([ej, ei]).astype(np.int64)
    ww = np.concatenate([w, w])
    order = np.lexsort((c, r))
    r, c, ww = r[order], c[order], ww[order]
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.add.at(rowptr, r + 1, 1)
    rowptr = np.cumsum(rowptr)
    return rowptr, c.astype(np.int32), ww


# ----------------------------------------------------------------------------- constants
def column_means(X, mask):
    """Observed column means (used by the cold start S4 and by G_bound S1)."""
    X = _f64(X)
    if mask is None:
        return X.mean(axis=0)
    mk = mask != 0
    cnt = mk.sum(axis=0)
    return (X * mk).sum(axis=0) / np.maximum(cnt, 1)


def g_bound(X, mask, w, gamma: float) -> float:
    """[reading S1] G_bound(gamma) = sqrt(sum_Gamma (x - xbar_j)^2 + gamma^2 sum_E w^2)."""
    X = _f64(X)
    xc = X - column_means(X, mask)[None, :]
    if mask is not None:
        xc = xc * (mask != 0)
    return float(np.sqrt((xc * xc).sum() + gamma * gamma * float((np.asarray(w, dtype=np.float64) ** 2).sum())))


def default_rho_eps(X, mask, w, gamma: float, rho_scale: float = 1.1, kappa: float = 1e-2):
    """[readings S1, S2] rho = rho_scale * G_bound(gamma), eps = (kappa rho)^2."""
    rho = rho_scale * g_bound(X, mask, w, gamma)
    return rho, (kappa * rho) ** 2


def cold_start(X, mask, ei, ej):
    """[reading S4] U0 = X with missing entries set to the observed column mean; V0 = D U0."""
    U = _f64(X).copy()
    if mask is not None:
        cm = column_means(X, mask)
        miss = mask == 0
        U[miss] = np.broadcast_to(cm, U.shape)[miss]
    V = U[ei] - U[ej]
    return U, np.ascontiguousarray(V)


# ----------------------------------------------------------------------------- MM iteration
def project(U, V, ei, ej, method: int = 0, tol: float = 1e-13, maxcycles: int = 100000):
    """Projection of (U~,V~) onto C.  Returns (A, cycles); B = A[ei]-A[ej]."""
    U = _f64(U)
    V = _f64(V)
    ei = np.ascontiguousarray(ei, dtype=np.int32)
    ej = np.ascontiguousarray(ej, dtype=np.int32)
    n, p = U.shape
    A = np.empty_like(U)
    cyc = _L().orc_project(n, p, ei.size, _p(ei), _p(ej), _p(U), _p(V), int(method), float(tol),
                           int(maxcycles), _p(A))
    if cyc < 0:
        raise RuntimeError(f"oracle projection failed to converge (code {cyc})")
    return A, int(cyc)


def mm(X, mask, ei, ej, w, gamma, rho, eps, U, V, maxit, tol=0.0, min_it=10, proj_method=0,
       proj_tol=1e-13, proj_maxcycles=100000):
    """Run the MM iteration from state (U,V); returns a dict with the new
    state, the Phi_m / d_m sequences and the iteration count.  Fails loudly on non-convergence of the
    projection or on an increase of Phi (MM descent property)."""
    X = _f64(X)
    mask = _u8(mask)
    ei = np.ascontiguousarray(ei, dtype=np.int32)
    ej = np.ascontiguousarray(ej, dtype=np.int32)
    w = _f64(w)
    n, p = X.shape
    U = _f64(U).copy()
    V = _f64(V).copy()
    phi_h = np.zeros(max(1, maxit))
    d_h = np.zeros(max(1, maxit))
    it = ctypes.c_int(0)
    cyc = ctypes.c_int64(0)
    rc = _L().orc_mm(n, p, _p(X), _p(mask), ei.size, _p(ei), _p(ej), _p(w), float(gamma), float(rho),
                     float(eps), int(maxit), float(tol), int(min_it), int(proj_method), float(proj_tol),
                     int(proj_maxcycles), _p(U), _p(V), _p(phi_h), _p(d_h), ctypes.byref(it),
                     ctypes.byref(cyc))
    if rc:
        raise RuntimeError({-1: "projection did not converge", -2: "out of memory",
                            -3: "Phi increased: MM descent property violated"}.get(rc, str(rc)))
    k = it.value
    return {"U": U, "V": V, "phi": phi_h[:k].copy(), "d": d_h[:k].copy(), "iters": k,
            "proj_cycles": int(cyc.value)}


def labels(V, ei, ej, n: int):
    """[reading S16] components over pairs with v_ij == 0 exactly, canonical numbering."""
    V = _f64(V)
    ei = np.ascontiguousarray(ei, dtype=np.int32)
    ej = np.ascontiguousarray(ej, dtype=np.int32)
    lab = np.empty(n, dtype=np.int32)
    k = _L().orc_labels(n, V.shape[1], ei.size, _p(ei), _p(ej), _p(V), _p(lab))
    return lab, int(k)


def objective(X, mask, ei, ej, w, gamma, U) -> float:
    """f_gamma(U) of eq. 1 / eq. 6."""
    X = _f64(X)
    U = _f64(U)
    r = X - U
    if mask is not None:
        r = r * (mask != 0)
    df = U[ei] - U[ej]
    return float(0.5 * (r * r).sum() + gamma * (np.asarray(w) * np.sqrt(np.einsum("ij,ij->i", df, df))).sum())


# ----------------------------------------------------------------------------- f2: principal components
def principal_components(X, mask, q: int):
    """[reading S25; "project the cluster path onto any two principal components of the
    original data"]  The q leading principal directions of the original data: X with its missing
    entries set to the observed column mean (the cold start U0 of S4), columns centred, then the
    textbook definition by the singular value decomposition  Xc = W diag(sigma) P^T:  direction k is
    row k of P^T, its variance sigma_k^2 / (n - 1)  (the eigenpairs of the sample covariance
    Xc^T Xc / (n - 1)).  Signs: the entry of largest magnitude of each direction is made positive.
    Returns (P  p x q,  variances  q)."""
    U0, _ = cold_start(X, mask, np.zeros(0, dtype=np.int64), np.zeros(0, dtype=np.int64))
    n = U0.shape[0]
    Xc = U0 - U0.mean(axis=0)[None, :]
    _, sig, Pt = np.linalg.svd(Xc, full_matrices=False)
    P = Pt[:q].T.copy()
    for k in range(P.shape[1]):
        if P[np.argmax(np.abs(P[:, k])), k] < 0:
            P[:, k] = -P[:, k]
    return P, (sig[:q] ** 2) / max(n - 1, 1)


def project_on_components(X, mask, U, P):
    """[PAPER.md L144, L210] coordinates of the rows of U on the directions P (p x q), measured from
    the observed column means of X:  (U - 1 xbar^T) P."""
    return (_f64(U) - column_means(X, mask)[None, :]) @ _f64(P)


# ----------------------------------------------------------------------------- f1: kappa continuation
def kappa_schedule(kappa_start: float, factor: float, kappa_final: float):
    """[reading S26] kappa_start, kappa_start*factor, ... while larger than kappa_final, then kappa_final."""
    ks = []
    k = float(kappa_start)
    while k > kappa_final * (1.0 + 1e-12):
        ks.append(k)
        k *= factor
    ks.append(float(kappa_final))
    return ks


def mm_continuation(X, mask, ei, ej, w, gamma, U, V, kappa_start, factor, stage_maxit, maxit, tol=0.0, min_it=10,
                    rho_scale=1.1, kappa=1e-2, proj_method=0, proj_tol=1e-13):
    """[reading S26; not in the paper, SURVEY 8(f) f1]  The MM iteration of L57-L88 run in stages at one gamma:
    rho stays at S1's value, eps_s = (kappa_s rho)^2 follows kappa_schedule; every stage starts from the state the
    previous one left, runs until the stop rule S3 or `stage_maxit` iterations (`maxit` for the last stage, whose
    kappa is the contract value).  Returns the last stage's dict plus the per-stage iteration counts."""
    rho, _ = default_rho_eps(X, mask, w, gamma, rho_scale, kappa)
    ks = kappa_schedule(kappa_start, factor, kappa)
    its = []
    r = None
    for s, k in enumerate(ks):
        last = s == len(ks) - 1
        r = mm(X, mask, ei, ej, w, gamma, rho, (k * rho) ** 2, U, V, maxit if last else stage_maxit, tol, min_it,
               proj_method, proj_tol)
        U, V = r["U"], r["V"]
        its.append(r["iters"])
    r.update(stage_iters=its, kappas=ks, rho=rho)
    return r


def path(X, mask, ei, ej, w, gammas, maxit, tol=0.0, min_it=10, rho_scale=1.1, kappa=1e-2, proj_method=0,
         proj_tol=1e-13):
    """gamma path with warm starts (warm start: reading S4).  rho, eps per gamma by
    S1/S2.  Returns a list of per-gamma dicts (U, labels, nclusters, iters, phi, d, rho, eps)."""
    U, V = cold_start(X, mask, ei, ej)
    out = []
    n = X.shape[0]
    for g in gammas:
        rho, eps = default_rho_eps(X, mask, w, g, rho_scale, kappa)
        r = mm(X, mask, ei, ej, w, g, rho, eps, U, V, maxit, tol, min_it, proj_method, proj_tol)
        U, V = r["U"], r["V"]
        lab, k = labels(V, ei, ej, n)
        r.update(labels=lab, nclusters=k, rho=rho, eps=eps, gamma=float(g))
        out.append(r)
    return out
