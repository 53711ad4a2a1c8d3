"""Shared test plumbing: builds one problem instance for BOTH sides.  The graph and weights come from
the oracle's eq.-8 code (weights are an *input* of the hot path); they are cast to fp32 once and the
same fp32 values (widened to fp64) go to the oracle."""
from __future__ import annotations

import numpy as np

from paper_1409_2065_b200 import synth


def build_problem(O, wl, n_pairs_phi=200_000):
    """Returns dict(X64, mask, ei, ej, w64, rowptr, col, wcsr32, phi)."""
    X64 = wl.X.astype(np.float64)
    n = wl.n
    if wl.phi_rule == "fixed":
        phi = wl.phi
    else:
        si, sj = synth.sample_pairs(n, n_pairs_phi, wl.seed)
        d2 = O.pair_dist2(X64, wl.mask, si, sj)
        phi = 1.0 / float(np.median(d2[np.isfinite(d2)]))
    if wl.graph == "knn":
        ei, ej, w, _ = O.knn_graph(X64, wl.mask, wl.k, phi)
    else:
        ei, ej, w, _ = O.complete_graph(X64, wl.mask, phi)
    w32 = w.astype(np.float32)
    keep = w32 > 0            # a weight that underflows in fp32 is a zero weight: the pair is absent (L40)
    ei, ej, w32 = ei[keep], ej[keep], w32[keep]
    w64 = w32.astype(np.float64)
    rowptr, col, wcsr = O.to_csr(n, ei, ej, w64)
    return {"X64": X64, "mask": wl.mask, "ei": ei, "ej": ej, "w64": w64, "rowptr": rowptr, "col": col,
            "wcsr32": wcsr.astype(np.float32), "phi": phi, "n": n, "p": wl.p}


def gpu_create(B, torch, prob, **prm_over):
    dev = torch.device("cuda:0")
    X = torch.from_numpy(prob["X64"].astype(np.float32)).to(dev)
    mask = None if prob["mask"] is None else torch.from_numpy(prob["mask"]).to(dev)
    rowptr = torch.from_numpy(prob["rowptr"].astype(np.int64)).to(dev)
    col = torch.from_numpy(prob["col"].astype(np.int32)).to(dev)
    w = torch.from_numpy(prob["wcsr32"]).to(dev)
    prm = B.cc_default_params(**prm_over)
    return B.cc_create(prob["n"], prob["p"], X, mask, rowptr, col, w, prm)


def oracle_path(O, prob, gammas, iters, proj_method=0, rho_scale=1.1, kappa=1e-2):
    return O.path(prob["X64"], prob["mask"], prob["ei"], prob["ej"], prob["w64"], gammas, iters,
                  rho_scale=rho_scale, kappa=kappa, proj_method=proj_method)


def relerr(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))
