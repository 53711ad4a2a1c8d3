"""Pins P1-P13: the fp64 oracle checked against what the paper and the mathematics fix,
never against itself.  CPU only (-m "not gpu")."""
import json
import os

import numpy as np
import pytest

from paper_1409_2065_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _tiny(O, seed=0, n=24, p=3, miss=0.0, connected=True, deg=4.0):
    rng = np.random.default_rng(seed)
    X = rng.normal(size=(n, p)) + 3.0 * rng.integers(0, 3, size=(n, 1))
    ei, ej, w = synth.random_graph(n, deg, seed + 1, connected=connected)
    mask = None
    if miss > 0:
        mask = (rng.random(size=(n, p)) >= miss).astype(np.uint8)
        mask[0, :] = 1
    return X, mask, ei, ej, w


def _incidence(n, ei, ej):
    D = np.zeros((len(ei), n))
    D[np.arange(len(ei)), ei] = 1.0
    D[np.arange(len(ei)), ej] = -1.0
    return D


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("miss", [0.0, 0.2])
def test_P1_gamma_zero_gives_X(oracle, miss):
    O = oracle
    X, mask, ei, ej, w = _tiny(O, 1, miss=miss)
    U, V = O.cold_start(X, mask, ei, ej)
    rho, eps = O.default_rho_eps(X, mask, w, 0.0)
    r = O.mm(X, mask, ei, ej, w, 0.0, rho, eps, U, V, 25)
    obs = np.ones_like(X, bool) if mask is None else mask != 0
    assert np.abs(r["U"] - X)[obs].max() < 1e-11
    # from the cold start the iterate is feasible at every iteration: d = sqrt(eps)
    assert np.allclose(r["d"], np.sqrt(eps), rtol=1e-9)


# ---------------------------------------------------------------- P2  n = 2 closed forms
def test_P2_two_points_unfused_and_fused(oracle):
    O = oracle
    x = np.array([[0.0, 0.0, 1.0], [3.0, 4.0, 1.0]])
    delta = 5.0
    ei, ej = np.array([0], np.int32), np.array([1], np.int32)
    w = np.array([0.7])
    U, V = O.cold_start(x, None, ei, ej)
    # unfused: exact solution of (1): each point moves gamma*w along the unit difference (north_star)
    g = 1.0
    rho, kappa = 40.0, 1e-2
    eps = (kappa * rho) ** 2
    r = O.mm(x, None, ei, ej, w, g, rho, eps, U, V, 60000, tol=0.0)
    u = r["U"]
    e = (x[0] - x[1]) / delta
    assert np.abs(u[0] - (x[0] - g * w[0] * e)).max() < 1e-9
    assert np.abs(u[1] - (x[1] + g * w[0] * e)).max() < 1e-9
    assert np.abs((u[0] + u[1]) / 2 - (x[0] + x[1]) / 2).max() < 1e-10
    d_fix = np.sqrt(eps / (1.0 - 3.0 * (g * w[0]) ** 2 / rho ** 2))
    assert abs(r["d"][-1] - d_fix) < 1e-9 * d_fix
    kap = d_fix / rho
    assert abs(np.linalg.norm(r["V"][0]) - (delta - 2 * g * w[0] - 3 * kap * g * w[0])) < 1e-8
    # fused: delta <= 2 gamma w  =>  v = 0, residual gap 3 kappa delta / (2 + 3 kappa), mean preserved
    g = 5.0
    r = O.mm(x, None, ei, ej, w, g, rho, eps, U, V, 60000, tol=0.0)
    u = r["U"]
    assert np.all(r["V"] == 0.0)
    kap = r["d"][-1] / rho
    gap = np.linalg.norm(u[0] - u[1])
    assert abs(gap - 3 * kap * delta / (2 + 3 * kap)) < 1e-9
    assert abs(r["d"][-1] ** 2 - (gap ** 2 / 3 + eps)) < 1e-9
    assert np.abs((u[0] + u[1]) / 2 - x.mean(axis=0)).max() < 1e-10
    lab, k = O.labels(r["V"], ei, ej, 2)
    assert k == 1 and list(lab) == [0, 0]


def test_P2_projection_formula_n2(oracle):
    O = oracle
    rng = np.random.default_rng(3)
    U = rng.normal(size=(2, 4))
    V = rng.normal(size=(1, 4))
    ei, ej = np.array([0], np.int32), np.array([1], np.int32)
    A, _ = O.project(U, V, ei, ej)
    assert np.abs((A[0] - A[1]) - (U[0] - U[1] + 2 * V[0]) / 3).max() < 1e-12
    dist2 = ((U - A) ** 2).sum() + ((V[0] - (A[0] - A[1])) ** 2).sum()
    assert abs(dist2 - ((U[0] - U[1] - V[0]) ** 2).sum() / 3) < 1e-12


# ---------------------------------------------------------------- P3 / P4  projection
def test_P3_complete_graph_closed_form(oracle):
    O = oracle
    rng = np.random.default_rng(4)
    n, p = 9, 5
    U = rng.normal(size=(n, p))
    ei, ej = np.triu_indices(n, 1)
    V = rng.normal(size=(len(ei), p))
    A, _ = O.project(U, V, ei, ej)
    D = _incidence(n, ei, ej)
    R = U + D.T @ V
    assert np.abs(A - (R + U.sum(axis=0)[None, :]) / (n + 1)).max() < 1e-12


@pytest.mark.parametrize("method", [0, 1])
def test_P4_projection_is_the_dense_solve(oracle, method):
    O = oracle
    rng = np.random.default_rng(5)
    n, p = 30, 4
    ei, ej, _ = synth.random_graph(n, 5.0, 11)
    U = rng.normal(size=(n, p))
    V = rng.normal(size=(len(ei), p))
    A, cyc = O.project(U, V, ei, ej, method=method)
    D = _incidence(n, ei, ej)
    Lap = D.T @ D
    A_ref = np.linalg.solve(np.eye(n) + Lap, U + D.T @ V)
    assert np.abs(A - A_ref).max() < 1e-11
    B = D @ A
    # normal equation and Pythagoras for the orthogonal projection onto the subspace C
    assert np.abs((U - A) + D.T @ (V - B)).max() < 1e-11
    lhs = ((U - A) ** 2).sum() + ((V - B) ** 2).sum()
    rhs = (U ** 2).sum() + (V ** 2).sum() - (A ** 2).sum() - (B ** 2).sum()
    assert abs(lhs - rhs) < 1e-10
    # it is the closest point of C: random feasible competitors are farther
    for _ in range(5):
        A2 = A + 0.1 * rng.normal(size=A.shape)
        assert ((U - A2) ** 2).sum() + ((V - D @ A2) ** 2).sum() > lhs


# ---------------------------------------------------------------- P5
@pytest.mark.parametrize("miss", [0.0, 0.15])
def test_P5_phi_monotone_and_matches_definition(oracle, miss):
    O = oracle
    X, mask, ei, ej, w = _tiny(O, 6, miss=miss)
    U, V = O.cold_start(X, mask, ei, ej)
    g = 0.8
    rho, eps = O.default_rho_eps(X, mask, w, g)
    r = O.mm(X, mask, ei, ej, w, g, rho, eps, U, V, 400)
    assert np.all(np.diff(r["phi"]) <= 1e-12 * np.abs(r["phi"][:-1]))
    # Phi_0 retyped from the definition at the cold start: feasible => dist = 0
    obs = np.ones_like(X, bool) if mask is None else mask != 0
    phi0 = 0.5 * ((X - U) ** 2)[obs].sum() + g * (w * np.linalg.norm(V, axis=1)).sum() + rho * np.sqrt(eps)
    assert abs(r["phi"][0] - phi0) < 1e-10 * abs(phi0)
    # Phi_1 from an independent dense evaluation of one iteration
    r1 = O.mm(X, mask, ei, ej, w, g, rho, eps, U, V, 1)
    D = _incidence(len(X), ei, ej)
    U1, V1 = r1["U"], r1["V"]
    A1 = np.linalg.solve(np.eye(len(X)) + D.T @ D, U1 + D.T @ V1)
    d1 = np.sqrt(((U1 - A1) ** 2).sum() + ((V1 - D @ A1) ** 2).sum() + eps)
    phi1 = 0.5 * ((X - U1) ** 2)[obs].sum() + g * (w * np.linalg.norm(V1, axis=1)).sum() + rho * d1
    assert abs(r["phi"][1] - phi1) < 1e-10 * abs(phi1)
    assert abs(r["d"][1] - d1) < 1e-9 * d1


# ---------------------------------------------------------------- P6  column sums per component
def test_P6_column_sums_conserved_per_component(oracle):
    O = oracle
    X, _, ei, ej, w = _tiny(O, 7, n=30, connected=False, deg=1.6)
    n = len(X)
    U, V = O.cold_start(X, None, ei, ej)
    g = 1.3
    rho, eps = O.default_rho_eps(X, None, w, g)
    comp, ncomp = O.labels(np.zeros((len(ei), 1)), ei, ej, n)   # all edges "fused" => graph components
    assert ncomp > 1
    for iters in (1, 7, 60):
        r = O.mm(X, None, ei, ej, w, g, rho, eps, U, V, iters)
        for c in range(ncomp):
            assert np.abs(r["U"][comp == c].sum(0) - X[comp == c].sum(0)).max() < 5e-9


# ---------------------------------------------------------------- P7  subgradient certificate
def test_P7_converged_certificate(oracle):
    O = oracle
    X, mask, ei, ej, w = _tiny(O, 8, n=12, p=2, miss=0.1, deg=3.0)
    n = len(X)
    U, V = O.cold_start(X, mask, ei, ej)
    g = 0.6
    rho, eps = O.default_rho_eps(X, mask, w, g, kappa=5e-2)
    r = O.mm(X, mask, ei, ej, w, g, rho, eps, U, V, 30000)
    U, V = r["U"], r["V"]
    A, _ = O.project(U, V, ei, ej)
    B = A[ei] - A[ej]
    d = np.sqrt(((U - A) ** 2).sum() + ((V - B) ** 2).sum() + eps)
    kap = d / rho
    G = (B - V) / (kap * g * w[:, None])
    gn = np.linalg.norm(G, axis=1)
    assert gn.max() <= 1.0 + 1e-7
    nz = np.linalg.norm(V, axis=1) > 0
    assert nz.any() and (~nz).any()          # both regimes present in this instance
    assert np.abs(G[nz] - V[nz] / np.linalg.norm(V[nz], axis=1, keepdims=True)).max() < 1e-6
    D = _incidence(n, ei, ej)
    res = (X - U) - g * D.T @ (w[:, None] * G)
    obs = mask != 0
    assert np.abs(res[obs]).max() < 1e-6
    # missing entries carry no loss gradient: the penalty subgradient alone vanishes there
    assert np.abs((g * D.T @ (w[:, None] * G))[~obs]).max() < 1e-6


# ---------------------------------------------------------------- P8
def test_P8_large_gamma_fuses_to_masked_component_means(oracle):
    O = oracle
    X, mask, ei, ej, w = _tiny(O, 9, n=30, miss=0.15, connected=True)
    n = len(X)
    obs = mask != 0
    mean = (X * obs).sum(0) / obs.sum(0)
    devs = []
    for kappa in (1e-1, 1e-2, 1e-3):
        U, V = O.cold_start(X, mask, ei, ej)
        g = 1e4
        rho, eps = O.default_rho_eps(X, mask, w, g, kappa=kappa)
        r = O.mm(X, mask, ei, ej, w, g, rho, eps, U, V, int(40 / kappa))
        assert np.all(r["V"] == 0.0)
        lab, k = O.labels(r["V"], ei, ej, n)
        assert k == 1
        devs.append(np.abs(r["U"] - mean[None, :]).max())
    # residual is O(kappa), not zero, and shrinks linearly in kappa
    assert devs[1] < 0.2 * devs[0] and devs[2] < 0.2 * devs[1]
    assert devs[2] < 2e-3 * 2 * np.abs(X - mean).max() * 10


def test_P8_disconnected_components_fuse_separately(oracle):
    O = oracle
    rng = np.random.default_rng(10)
    X = rng.normal(size=(10, 3))
    ei = np.array([0, 1, 2, 3, 5, 6, 7, 8], np.int32)
    ej = np.array([1, 2, 3, 4, 6, 7, 8, 9], np.int32)    # two chains: 0-4 and 5-9
    w = np.ones(8)
    U, V = O.cold_start(X, None, ei, ej)
    g = 1e3
    rho, eps = O.default_rho_eps(X, None, w, g, kappa=1e-3)
    r = O.mm(X, None, ei, ej, w, g, rho, eps, U, V, 40000)
    lab, k = O.labels(r["V"], ei, ej, 10)
    assert k == 2 and list(lab) == [0] * 5 + [1] * 5
    assert np.abs(r["U"][:5] - X[:5].mean(0)).max() < 1e-2
    assert np.abs(r["U"][5:] - X[5:].mean(0)).max() < 1e-2


# ---------------------------------------------------------------- P9  independent exact solver
def _admm_exact(X, ei, ej, w, g, iters=20000, nu=1.0):
    """Independent solver of (1): ADMM on the split problem (not the paper's algorithm)."""
    n, p = X.shape
    D = _incidence(n, ei, ej)
    M = np.linalg.inv(np.eye(n) + nu * D.T @ D)
    V = D @ X
    Lm = np.zeros_like(V)
    U = X.copy()
    for _ in range(iters):
        U = M @ (X + nu * D.T @ (V - Lm))
        Z = D @ U + Lm
        nz = np.linalg.norm(Z, axis=1, keepdims=True)
        V = np.maximum(1.0 - (g * w[:, None] / nu) / np.maximum(nz, 1e-300), 0.0) * Z
        Lm = Z - V
    return U


def test_P9_matches_independent_solver_within_c_kappa(oracle):
    O = oracle
    X, _, ei, ej, w = _tiny(O, 12, n=8, p=2, deg=3.0)
    g = 0.5
    U_star = _admm_exact(X, ei, ej, w, g)
    # U_star is optimal for (1): objective not larger than at perturbed points
    f_star = O.objective(X, None, ei, ej, w, g, U_star)
    rng = np.random.default_rng(0)
    for _ in range(10):
        assert O.objective(X, None, ei, ej, w, g, U_star + 1e-3 * rng.normal(size=X.shape)) >= f_star
    errs = []
    for kappa in (1e-1, 1e-2, 1e-3):
        U, V = O.cold_start(X, None, ei, ej)
        rho, eps = O.default_rho_eps(X, None, w, g, kappa=kappa)
        r = O.mm(X, None, ei, ej, w, g, rho, eps, U, V, int(60 / kappa))
        errs.append(np.linalg.norm(r["U"] - U_star) / np.linalg.norm(U_star))
    assert errs[0] < 0.2 and errs[1] < 0.2 * errs[0] + 1e-6 and errs[2] < 0.2 * errs[1] + 1e-6


# ---------------------------------------------------------------- P10
def test_P10_zero_b_gives_zero_v(oracle):
    O = oracle
    X = np.array([[1.0, 2.0], [1.0, 2.0], [4.0, 0.0]])       # points 0 and 1 coincide
    ei, ej = np.array([0, 1], np.int32), np.array([1, 2], np.int32)
    w = np.array([0.5, 0.5])
    U, V = O.cold_start(X, None, ei, ej)
    rho, eps = O.default_rho_eps(X, None, w, 0.1)
    r = O.mm(X, None, ei, ej, w, 0.1, rho, eps, U, V, 50)
    assert np.all(r["V"][0] == 0.0) and np.all(np.isfinite(r["U"]))
    lab, k = O.labels(r["V"], ei, ej, 3)
    assert list(lab) == [0, 0, 1] and k == 2


# ---------------------------------------------------------------- P12 / P13 invariances
def test_P12_equivariances(oracle):
    O = oracle
    X, _, ei, ej, w = _tiny(O, 13, n=16, p=3)
    g, c = 0.7, 3.5
    def run(Xa, ga, ei_, ej_, w_):
        U, V = O.cold_start(Xa, None, ei_, ej_)
        rho, eps = O.default_rho_eps(Xa, None, w_, ga)
        return O.mm(Xa, None, ei_, ej_, w_, ga, rho, eps, U, V, 300)["U"]
    U0 = run(X, g, ei, ej, w)
    assert np.abs(run(c * X, c * g, ei, ej, w) - c * U0).max() < 1e-10
    t = np.array([[5.0, -2.0, 0.5]])
    assert np.abs(run(X + t, g, ei, ej, w) - (U0 + t)).max() < 1e-10
    perm = np.random.default_rng(1).permutation(len(X))
    inv = np.argsort(perm)                     # new index of old node i is inv[i]
    a, b = inv[ei], inv[ej]
    lo, hi = np.minimum(a, b).astype(np.int32), np.maximum(a, b).astype(np.int32)
    Up = run(X[perm], g, lo, hi, w)
    # a pair stored as (j,i) instead of (i,j) carries -v: same problem, rows permuted
    assert np.abs(Up - U0[perm]).max() < 1e-9


def test_P13_weight_normalisation_is_gamma_rescaling(oracle):
    O = oracle
    X, mask, ei, ej, w = _tiny(O, 14, miss=0.1)
    g, c = 0.9, w.sum()
    U, V = O.cold_start(X, mask, ei, ej)
    rho, eps = O.default_rho_eps(X, mask, w, g)
    r1 = O.mm(X, mask, ei, ej, w, g, rho, eps, U, V, 100)
    r2 = O.mm(X, mask, ei, ej, w / c, c * g, rho, eps, U, V, 100)
    assert np.abs(r1["U"] - r2["U"]).max() < 1e-12


# ---------------------------------------------------------------- a0 weights (eq. 8)
def test_knn_graph_against_numpy_brute_force(oracle):
    O = oracle
    rng = np.random.default_rng(15)
    X = rng.normal(size=(40, 6))
    k, phi = 4, 0.3
    ei, ej, w, dd = O.knn_graph(X, None, k, phi)
    D2 = ((X[:, None, :] - X[None, :, :]) ** 2).sum(-1)
    np.fill_diagonal(D2, np.inf)
    nn = np.argsort(D2, axis=1, kind="stable")[:, :k]
    adj = np.zeros((40, 40), bool)
    adj[np.repeat(np.arange(40), k), nn.reshape(-1)] = True
    adj = adj | adj.T                                     # "or vice versa"
    ii, jj = np.nonzero(np.triu(adj, 1))
    assert np.array_equal(ii, ei) and np.array_equal(jj, ej)
    assert np.allclose(w, np.exp(-phi * D2[ii, jj]), rtol=1e-13)
    # phi = 0: uniform weights (L131); normalisation sums to one (L133)
    assert np.all(O.knn_graph(X, None, k, 0.0)[2] == 1.0)
    assert abs(O.knn_graph(X, None, k, phi, normalize=True)[2].sum() - 1.0) < 1e-14
    rp, col, ww = O.to_csr(40, ei, ej, w)
    assert rp[-1] == 2 * len(ei) and np.all(np.diff(rp) >= k)


def test_knn_masked_distance_rule(oracle):
    O = oracle
    X = np.array([[0.0, 0.0, 9.0, 1.0], [1.0, 1.0, 0.0, 1.0], [5.0, 5.0, 5.0, 5.0]])
    mask = np.array([[1, 1, 0, 1], [1, 1, 1, 0], [1, 1, 1, 1]], np.uint8)
    d = O.row_dist2(X, mask, 0)
    assert d[0] == np.inf and abs(d[1] - 2.0 * 4 / 2) < 1e-15 and abs(d[2] - (25 + 25 + 16) * 4 / 3) < 1e-13


def _brute_knn(X, mask, k):
    """k nearest by the definition: all squared distances (masked rule S11 by explicit loops), stable argsort
    (equal distances keep the smaller index first, S9), self excluded."""
    n, p = X.shape
    D2 = np.full((n, n), np.inf)
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            if mask is None:
                D2[i, j] = float(((X[i] - X[j]) ** 2).sum())
            else:
                co = [c for c in range(p) if mask[i, c] and mask[j, c]]
                if co:
                    D2[i, j] = float(sum((X[i, c] - X[j, c]) ** 2 for c in co)) * p / len(co)
    return np.argsort(D2, axis=1, kind="stable")[:, :k], D2


def test_knn_tie_rule_smaller_index_first(oracle):
    """Reading S9 (PAPER.md L127 does not say how ties are broken): equal distances go to the smaller index.
    Lattice points and duplicated rows have many exact ties; turning the oracle's strict '<' into '<=' (or
    scanning candidates in another order) changes these neighbour lists."""
    O = oracle
    n_ties = 0
    for name, X32, mask, k in synth.tie_cases():
        X = X32.astype(np.float64)
        nn, D2 = _brute_knn(X, mask, k)
        nbr, d2 = O.knn(X, mask, k)
        assert np.array_equal(nbr, nn), name
        assert np.array_equal(d2, np.take_along_axis(D2, nn, axis=1)), name
        # the cases really have ties AT the cut: the k-th and (k+1)-th distances coincide for some rows
        srt = np.sort(D2, axis=1)
        n_ties += int((srt[:, k - 1] == srt[:, k]).sum())
        # numpy restatement of the masked rule (used for the phi rule) agrees with the C rule
        ii, jj = np.triu_indices(X.shape[0], 1)
        d_np = O.pair_dist2(X, mask, ii, jj)
        assert np.array_equal(d_np, D2[ii, jj]) or np.allclose(d_np, D2[ii, jj], rtol=1e-15), name
    assert n_ties > 50


def test_pair_dist2_masked_branch_matches_the_c_rule(oracle):
    """oracle.pair_dist2 (numpy, used for the phi rule S10) restates orc_row_dist2's masked rule S11."""
    O = oracle
    rng = np.random.default_rng(3)
    X = rng.normal(size=(25, 9))
    mask = (rng.random(size=X.shape) >= 0.4).astype(np.uint8)
    mask[3, :] = 0
    mask[3, 0] = 1
    mask[4, :] = 0
    mask[4, 5] = 1                                   # rows 3 and 4 share no observed coordinate
    for i in (0, 3, 4, 11):
        d_c = O.row_dist2(X, mask, i)
        jj = np.array([j for j in range(25) if j != i])
        d_np = O.pair_dist2(X, mask, np.full(jj.size, i), jj)
        assert np.allclose(d_np[np.isfinite(d_np)], d_c[jj][np.isfinite(d_c[jj])], rtol=1e-14)
        assert np.array_equal(np.isinf(d_np), np.isinf(d_c[jj]))
    assert np.isinf(O.row_dist2(X, mask, 3)[4])


def test_S3_stop_rule_iteration_count(oracle):
    """Reading S3: stop after iteration m (0-based) as soon as m + 1 >= min_it, m >= 1 and
    Phi_{m-1} - Phi_m <= tol (1 + |Phi_{m-1}|).  The count is re-derived here from the Phi history of a
    fixed-length run (tol = 0), so an off-by-one in either index of the rule fails."""
    O = oracle
    X, mask, ei, ej, w = _tiny(O, seed=21, n=18, p=3)
    g = 1.5
    rho, eps = O.default_rho_eps(X, mask, w, g)
    U0, V0 = O.cold_start(X, mask, ei, ej)
    full = O.mm(X, mask, ei, ej, w, g, rho, eps, U0, V0, 400)
    phi = full["phi"]
    dec = (phi[:-1] - phi[1:]) / (1.0 + np.abs(phi[:-1]))        # dec[m-1] belongs to iteration m
    assert np.all(np.diff(dec[5:]) < 0)                           # decreasing: the first crossing is well defined

    def expected(tol, min_it):
        for m in range(1, len(phi)):
            if m + 1 >= min_it and dec[m - 1] <= tol:
                return m + 1
        return len(phi)

    for min_it in (0, 1, 2, 7, 10, 40):
        for m_star in (12, 30):
            tol = float(np.sqrt(dec[m_star - 1] * dec[m_star - 2]))   # between the decreases of iterations m*-1 and m*
            r = O.mm(X, mask, ei, ej, w, g, rho, eps, U0, V0, 400, tol=tol, min_it=min_it)
            want = expected(tol, min_it)
            assert r["iters"] == want == max(m_star + 1, min_it, 2), (min_it, m_star, r["iters"], want)
            assert np.array_equal(r["phi"], phi[:want])
    # a tolerance that every decrease satisfies: min_it alone decides, but never before two iterations (m >= 1)
    for min_it, want in ((0, 2), (1, 2), (2, 2), (3, 3), (9, 9)):
        assert O.mm(X, mask, ei, ej, w, g, rho, eps, U0, V0, 400, tol=1e9, min_it=min_it)["iters"] == want


# ---------------------------------------------------------------- golden fixture (oracle-written)
def test_golden_tiny_path_is_reproducible(oracle):
    """tests/golden/tiny_path.json is written by tests/golden/make_golden.py, which calls only
    oracle/.  It guards the oracle against silent drift; the values are pinned by P1-P13 above."""
    O = oracle
    with open(os.path.join(GOLD, "tiny_path.json")) as f:
        gold = json.load(f)
    wl = synth.make("tiny")
    X = wl.X.astype(np.float64)
    ei, ej, w, _ = O.knn_graph(X, None, wl.k, wl.phi)
    assert len(ei) == gold["n_pairs"]
    res = O.path(X, None, ei, ej, w, gold["gammas"], gold["iters"])
    for r, g in zip(res, gold["per_gamma"]):
        assert abs(r["phi"][-1] - g["phi_last"]) < 1e-9 * abs(g["phi_last"])
        assert abs(np.linalg.norm(r["U"]) - g["U_fro"]) < 1e-9 * g["U_fro"]
        assert r["nclusters"] == g["nclusters"]


# ----------------------------------------------------------------------------- f2: principal components (S25, L144)
def _householder(p, seed):
    """An explicit orthogonal matrix I - 2 h h^T / (h^T h) (its columns are the planted directions)."""
    h = np.random.default_rng(seed).standard_normal(p)
    return np.eye(p) - 2.0 * np.outer(h, h) / float(h @ h)


def test_P14_principal_components_of_a_planted_cross(oracle):
    """Closed form: the 2p points  c +/- s_k r_k  (r_k the columns of a reflector R) have the sample
    covariance  R diag(2 s_k^2 / (n-1)) R^T,  so direction k is r_k and its variance 2 s_k^2/(n-1)."""
    p = 6
    R = _householder(p, 3)
    s = np.array([5.0, 3.5, 2.0, 1.0, 0.5, 0.25])
    c = np.linspace(-1.0, 2.0, p)
    X = np.concatenate([c[None, :] + s[:, None] * R.T, c[None, :] - s[:, None] * R.T])
    X = X[np.random.default_rng(0).permutation(2 * p)]
    P, var = oracle.principal_components(X, None, 3)
    assert np.allclose(var, 2.0 * s[:3] ** 2 / (2 * p - 1), rtol=1e-12)
    for k in range(3):
        r = R[:, k] * np.sign(R[np.argmax(np.abs(R[:, k])), k])
        assert np.allclose(P[:, k], r, atol=1e-12)


def test_P14_principal_components_satisfy_the_eigen_equation_of_a_loop_built_covariance(oracle):
    """Brute force on a tiny masked input: the covariance is accumulated entry by entry with Python loops
    from the imputed data; C v = lambda v, orthonormality, the trace identity with q = p, decreasing order,
    and the variance of the projected coordinates equals lambda."""
    rng = np.random.default_rng(5)
    n, p = 9, 4
    X = rng.standard_normal((n, p)) * np.array([3.0, 1.0, 0.3, 2.0]) + 1.5
    mask = (rng.random((n, p)) > 0.25).astype(np.uint8)
    mask[0, :] = 1
    mean = [sum(X[i, c] for i in range(n) if mask[i, c]) / sum(int(mask[i, c]) for i in range(n)) for c in range(p)]
    Y = [[X[i, c] if mask[i, c] else mean[c] for c in range(p)] for i in range(n)]
    cm = [sum(Y[i][c] for i in range(n)) / n for c in range(p)]
    C = np.zeros((p, p))
    for a in range(p):
        for b in range(p):
            C[a, b] = sum((Y[i][a] - cm[a]) * (Y[i][b] - cm[b]) for i in range(n)) / (n - 1)
    P, var = oracle.principal_components(X, mask, p)
    assert np.all(np.diff(var) <= 1e-15)
    assert np.isclose(var.sum(), np.trace(C), rtol=1e-12)
    assert np.allclose(P.T @ P, np.eye(p), atol=1e-12)
    for k in range(p):
        assert np.allclose(C @ P[:, k], var[k] * P[:, k], atol=1e-12)
    # imputed entries sit at the column mean, so the centring of project_on_components is the same mean
    coords = oracle.project_on_components(X, mask, np.array(Y), P)
    assert np.allclose(coords.mean(axis=0), 0.0, atol=1e-12)
    assert np.allclose(coords.var(axis=0, ddof=1), var, rtol=1e-12)


def test_P14_rank_one_data_has_one_direction(oracle):
    """x_i = c + t_i g: one direction g/||g|| with variance var(t) ||g||^2, every other variance 0."""
    rng = np.random.default_rng(8)
    g = np.array([1.0, -2.0, 0.5, 4.0, 0.0])
    t = rng.standard_normal(40)
    X = 0.7 + t[:, None] * g[None, :]
    P, var = oracle.principal_components(X, None, 2)
    assert np.allclose(P[:, 0], g / np.linalg.norm(g), atol=1e-12)
    assert np.isclose(var[0], t.var(ddof=1) * float(g @ g), rtol=1e-12)
    assert var[1] <= 1e-25 * var[0]


# ----------------------------------------------------------------------------- f1: kappa continuation (S26)
def test_P15_kappa_schedule_and_single_stage_is_the_plain_iteration(oracle):
    assert oracle.kappa_schedule(1.0, 0.1, 1e-2) == pytest.approx([1.0, 0.1, 1e-2])
    assert oracle.kappa_schedule(1e-2, 0.1, 1e-2) == [1e-2]
    assert oracle.kappa_schedule(0.5, 0.5, 0.1) == pytest.approx([0.5, 0.25, 0.125, 0.1])
    X, mask, ei, ej, w = _tiny(oracle, seed=3)
    U0, V0 = oracle.cold_start(X, mask, ei, ej)
    rho, eps = oracle.default_rho_eps(X, mask, w, 0.8)
    a = oracle.mm(X, mask, ei, ej, w, 0.8, rho, eps, U0, V0, 25)
    b = oracle.mm_continuation(X, mask, ei, ej, w, 0.8, U0, V0, 1e-2, 0.1, 7, 25)
    assert b["stage_iters"] == [25] and np.array_equal(a["U"], b["U"]) and np.array_equal(a["phi"], b["phi"])


def test_P15_continuation_reaches_the_fixed_point_of_the_last_stage(oracle):
    """The surrogate-free objective of the last stage (eps = (kappa rho)^2) is convex with a unique minimiser in U,
    so staged and plain runs, both converged, meet: the stages change the road, not the destination.  Also: every
    stage by itself is the monotone MM iteration (oracle.mm raises if Phi increases)."""
    X, mask, ei, ej, w = _tiny(oracle, seed=5, n=20, miss=0.15)
    U0, V0 = oracle.cold_start(X, mask, ei, ej)
    g = 0.6
    rho, eps = oracle.default_rho_eps(X, mask, w, g)
    plain = oracle.mm(X, mask, ei, ej, w, g, rho, eps, U0, V0, 60000, tol=1e-15, min_it=10)
    cont = oracle.mm_continuation(X, mask, ei, ej, w, g, U0, V0, 1.0, 0.1, 2000, 60000, tol=1e-15)
    assert len(cont["stage_iters"]) == 3
    scale = np.linalg.norm(plain["U"])
    assert np.linalg.norm(plain["U"] - cont["U"]) <= 1e-5 * scale
    assert abs(oracle.objective(X, mask, ei, ej, w, g, plain["U"]) -
               oracle.objective(X, mask, ei, ej, w, g, cont["U"])) <= 1e-6 * abs(oracle.objective(X, mask, ei, ej, w, g, plain["U"]))
    print("iterations plain", plain["iters"], "staged", cont["stage_iters"])


# ----------------------------------------------------------------------------- f4: composite distance, eq. 9 (L135-L137)
def test_P16_composite_distance_limits_and_wrap(oracle):
    rng = np.random.default_rng(2)
    n, p = 40, 5
    X = rng.standard_normal((n, p))
    Y = np.stack([rng.uniform(-180, 180, n), rng.uniform(-60, 60, n)], axis=1)
    # alpha = 1: eq. 9 is ||x_i - x_j||, so the graph is eq. 8's and the weight exp(-phi d^2) is the same number
    e8 = oracle.knn_graph(X, None, 4, 0.3)
    e9 = oracle.composite_knn_graph(X, None, Y, None, 1.0, 4, 0.3)
    assert np.array_equal(e8[0], e9[0]) and np.array_equal(e8[1], e9[1]) and np.allclose(e8[2], e9[2], rtol=1e-12)
    # alpha = 0: the graph of the side coordinates alone
    e8y = oracle.knn_graph(Y, None, 4, 0.3)
    e9y = oracle.composite_knn_graph(X, None, Y, None, 0.0, 4, 0.3)
    assert np.array_equal(e8y[0], e9y[0]) and np.array_equal(e8y[1], e9y[1]) and np.allclose(e8y[2], e9y[2], rtol=1e-12)
    # modulo arithmetic: longitudes 179 and -179 are 2 apart, not 358; latitude (period 0) is not wrapped
    Yw = np.array([[179.0, 10.0], [-179.0, 10.0], [0.0, 10.0], [90.0, -50.0]])
    d = oracle.side_dist(Yw, [360.0, 0.0], 0)
    assert np.allclose(d, [0.0, 2.0, 179.0, np.hypot(89.0, 60.0)])
    assert np.allclose(oracle.side_dist(Yw, None, 0)[1], 358.0)
    # brute force of eq. 9 entry by entry on the small case, and the OR rule
    al = 0.35
    D = np.zeros((n, n))
    for i in range(n):
        for j in range(n):
            dy0 = Y[i, 0] - Y[j, 0]
            dy0 -= 360.0 * round(dy0 / 360.0)
            D[i, j] = al * np.sqrt(sum((X[i, c] - X[j, c]) ** 2 for c in range(p))) + (1 - al) * np.hypot(dy0, Y[i, 1] - Y[j, 1])
        D[i, i] = np.inf
    near = [set(np.argsort(D[i], kind="stable")[:3].tolist()) for i in range(n)]
    want = sorted({(min(i, j), max(i, j)) for i in range(n) for j in near[i]})
    ei, ej, w, dd = oracle.composite_knn_graph(X, None, Y, [360.0, 0.0], al, 3, 0.01)
    assert list(zip(ei.tolist(), ej.tolist())) == want
    assert np.allclose(dd, [D[a, b] for a, b in want], rtol=1e-12)
    assert np.allclose(w, np.exp(-0.01 * dd ** 2), rtol=1e-12)
    wn = oracle.composite_knn_graph(X, None, Y, [360.0, 0.0], al, 3, 0.01, normalize=True)[2]
    assert np.isclose(wn.sum(), 1.0) and np.allclose(wn * w.sum(), w)


# ----------------------------------------------------------------------------- f4: geodesic alternative of eq. 9 (L137, S28)
def test_P17_geodesic_distance(oracle):
    R = 6371.0
    # closed forms on the sphere: pole to equator is a quarter circle, antipodes half a circle, along a meridian
    # R |dlat|, along the equator R |dlon| taken the short way round (179 E to 179 W is 2 degrees, not 358)
    LL = np.array([[0.0, 0.0], [0.0, 90.0], [180.0, 0.0], [37.0, -90.0], [0.0, 33.0], [179.0, 0.0], [-179.0, 0.0],
                   [90.0, 0.0]])
    d0 = oracle.geodesic_dist(LL, R, 0)
    assert np.allclose(d0, R * np.array([0.0, np.pi / 2, np.pi, np.pi / 2, np.deg2rad(33.0), np.deg2rad(179.0),
                                         np.deg2rad(179.0), np.pi / 2]), rtol=1e-12)
    assert np.isclose(oracle.geodesic_dist(LL, R, 5)[6], R * np.deg2rad(2.0), rtol=1e-9)
    assert np.isclose(oracle.geodesic_dist(LL, R, 1)[3], R * np.pi, rtol=1e-12)        # pole to pole, any longitudes
    # a different definition of the same angle: unit vectors in 3-D, theta = atan2(|a x b|, a.b)
    rng = np.random.default_rng(5)
    n = 60
    LLr = np.stack([rng.uniform(-180, 180, n), rng.uniform(-90, 90, n)], axis=1)
    lon, lat = np.deg2rad(LLr[:, 0]), np.deg2rad(LLr[:, 1])
    V = np.stack([np.cos(lat) * np.cos(lon), np.cos(lat) * np.sin(lon), np.sin(lat)], axis=1)
    D = np.zeros((n, n))
    for i in range(n):
        D[i] = oracle.geodesic_dist(LLr, 1.0, i)
        for j in range(n):
            th = np.arctan2(np.linalg.norm(np.cross(V[i], V[j])), float(V[i] @ V[j]))
            assert abs(D[i, j] - th) <= 1e-12, (i, j)
    # a metric: symmetric, zero diagonal, triangle inequality
    assert np.allclose(D, D.T, atol=1e-14) and np.all(np.diag(D) == 0.0)
    for i in range(0, n, 7):
        for j in range(n):
            assert np.all(D[i, j] <= D[i, :] + D[:, j] + 1e-12)
    # small separations: the sphere is flat, d ~ R sqrt(dlat^2 + (cos(lat) dlon)^2)
    base = np.array([[12.0, 48.0]])
    near = base + 1e-3 * rng.standard_normal((20, 2))
    LLs = np.concatenate([base, near])
    ds = oracle.geodesic_dist(LLs, R, 0)[1:]
    flat = R * np.hypot(np.deg2rad(near[:, 1] - 48.0), np.cos(np.deg2rad(48.0)) * np.deg2rad(near[:, 0] - 12.0))
    assert np.allclose(ds, flat, rtol=1e-4)
    # inside eq. 9: alpha = 0 gives the k-NN graph of the geodesic distances alone (brute force), alpha = 1 is eq. 8
    X = rng.standard_normal((n, 4))
    e8 = oracle.knn_graph(X, None, 3, 0.2)
    e9 = oracle.composite_knn_graph(X, None, LLr, None, 1.0, 3, 0.2, geodesic_radius=R)
    assert np.array_equal(e8[0], e9[0]) and np.array_equal(e8[1], e9[1]) and np.allclose(e8[2], e9[2], rtol=1e-12)
    Dn = D.copy()
    np.fill_diagonal(Dn, np.inf)
    near3 = [set(np.argsort(Dn[i], kind="stable")[:3].tolist()) for i in range(n)]
    want = sorted({(min(i, j), max(i, j)) for i in range(n) for j in near3[i]})
    ei, ej, w, dd = oracle.composite_knn_graph(X, None, LLr, None, 0.0, 3, 0.5, geodesic_radius=1.0)
    assert list(zip(ei.tolist(), ej.tolist())) == want
    assert np.allclose(dd, [D[a, b] for a, b in want], rtol=1e-12) and np.allclose(w, np.exp(-0.5 * dd ** 2), rtol=1e-12)
    # mixed: entry by entry
    al = 0.6
    ei, ej, w, dd = oracle.composite_knn_graph(X, None, LLr, None, al, 3, 0.5, geodesic_radius=2.0)
    for a, b, dv in zip(ei.tolist(), ej.tolist(), dd.tolist()):
        assert np.isclose(dv, al * np.linalg.norm(X[a] - X[b]) + (1 - al) * 2.0 * D[a, b], rtol=1e-12)
