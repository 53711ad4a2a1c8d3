"""GPU tests of the boundary (-m gpu): input validation / error codes of include/cc_b200.h, and the
a0 weight build against the oracle's brute-force eq. 8."""
import numpy as np
import pytest

import helpers as H
from paper_1409_2065_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_2065_b200 import binding
    return binding


def _dev(torch, a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def _create(B, torch, n, p, X, mask, rowptr, col, w, **prm):
    return B.cc_create(n, p, _dev(torch, X), _dev(torch, mask), _dev(torch, rowptr), _dev(torch, col), _dev(torch, w),
                       B.cc_default_params(**prm))


def test_validation_error_codes(B):
    import torch
    n, p = 4, 3
    X = np.arange(12, dtype=np.float32).reshape(n, p)
    # path 0-1, 1-2, 2-3
    rowptr = np.array([0, 1, 3, 5, 6], np.int64)
    col = np.array([1, 0, 2, 1, 3, 2], np.int32)
    w = np.ones(6, np.float32)
    h = _create(B, torch, n, p, X, None, rowptr, col, w)
    assert B.cc_get_counts(h)["n_pairs"] == 3
    with pytest.raises(B.CCError) as e:
        B.cc_solve(h, -1.0, 0.0, 5)
    assert e.value.code == B.CC_EINVAL
    with pytest.raises(B.CCError) as e:
        B.cc_solve(h, float("nan"), 0.0, 5)
    assert e.value.code == B.CC_EINVAL
    assert B.cc_solve(h, 1.0, 0.0, 0)[0] == 0
    B.cc_destroy(h)

    def fails(code, X=X, mask=None, rowptr=rowptr, col=col, w=w, n=n, p=p):
        with pytest.raises(B.CCError) as e:
            _create(B, torch, n, p, X, mask, rowptr, col, w)
        assert e.value.code == code, (e.value.code, str(e.value))

    w2 = w.copy(); w2[0] = 2.0
    fails(B.CC_EGRAPH, w=w2)                                                   # w_ij != w_ji
    fails(B.CC_EGRAPH, col=np.array([1, 0, 2, 1, 3, 3], np.int32))             # self loop / asymmetric
    fails(B.CC_EGRAPH, col=np.array([1, 2, 0, 1, 3, 2], np.int32))             # unsorted row
    fails(B.CC_EGRAPH, col=np.array([1, 0, 2, 1, 9, 2], np.int32))             # out of range
    w3 = w.copy(); w3[0] = w3[1] = 0.0
    fails(B.CC_EGRAPH, w=w3)                                                   # w <= 0
    fails(B.CC_EGRAPH, rowptr=np.array([0, 2, 1, 5, 6], np.int64))             # rowptr not monotone
    Xn = X.copy(); Xn[1, 1] = np.nan
    fails(B.CC_EINVAL, X=Xn)
    mk = np.ones((n, p), np.uint8); mk[:, 2] = 0
    fails(B.CC_EMASK, mask=mk)                                                 # a column never observed
    mk2 = np.ones((n, p), np.uint8); mk2[1, 1] = 0                             # NaN at a missing entry is ignored
    h = _create(B, torch, n, p, Xn, mk2, rowptr, col, w)
    B.cc_solve(h, 0.5, 0.0, 10)
    U = torch.empty(n, p, device="cuda:0")
    B.cc_get_U(h, -1, U)
    assert torch.isfinite(U).all()
    B.cc_destroy(h)
    fails(B.CC_EINVAL, n=0)
    with pytest.raises(B.CCError) as e:
        B.cc_knn_weights(5, 2, _dev(torch, X[:, :2].copy()), None, 7, 1.0)
    assert e.value.code == B.CC_EINVAL


@pytest.mark.parametrize("name,kw,k,phi,norm", [("tiny", {}, 5, 0.5, False),
                                                ("large_sparse", dict(n=3000, p=64, n_clusters=10), 10, 0.01, False),
                                                ("large_sparse", dict(n=1000, p=21, n_clusters=5), 3, 0.02, True),
                                                ("expression", dict(n=60, p=333), 10, 0.002, False)])
def test_knn_weights_match_oracle(B, oracle, name, kw, k, phi, norm):
    """a0 against brute-force eq. 8: same neighbour sets (the data are continuous: no exact ties), same
    CSR, weights to fp32 rounding; includes the masked distance rule S11 and normalisation S8."""
    import torch
    wl = synth.make(name, **kw)
    X64 = wl.X.astype(np.float64)
    ei, ej, w, _ = oracle.knn_graph(X64, wl.mask, k, phi, normalize=norm)
    rp, cl, ww = oracle.to_csr(wl.n, ei, ej, w)
    rowptr, col, wg = B.cc_knn_weights(wl.n, wl.p, _dev(torch, wl.X), _dev(torch, wl.mask), k, phi, normalize=norm)
    assert np.array_equal(rowptr.cpu().numpy(), rp)
    assert np.array_equal(col.cpu().numpy(), cl)
    assert np.abs(wg.cpu().numpy() - ww).max() <= 2e-5 * ww.max()
    # feeds cc_create unchanged (symmetric, sorted, w_ij == w_ji bitwise)
    h = B.cc_create(wl.n, wl.p, _dev(torch, wl.X), _dev(torch, wl.mask), rowptr, col, wg, None)
    assert B.cc_get_counts(h)["n_pairs"] == len(ei)
    B.cc_destroy(h)


def _oracle_csr(oracle, X32, mask, k, phi):
    """The oracle's eq.-8 graph as the CSR the library must return: weights cast to fp32 once, pairs whose weight
    is 0 in fp32 absent (S24)."""
    n = X32.shape[0]
    ei, ej, w, _ = oracle.knn_graph(X32.astype(np.float64), mask, k, phi)
    w32 = w.astype(np.float32)
    keep = w32 > 0
    rp, cl, ww = oracle.to_csr(n, ei[keep], ej[keep], w32[keep].astype(np.float64))
    return rp, cl, ww.astype(np.float32), int((~keep).sum())


def test_knn_tie_rule_and_rows_with_few_candidates(B, oracle):
    """Index output is held to identity.  (1) Exact ties (lattice points, duplicated rows): the smaller index wins on
    both sides (S9) -- the fp32 pass cannot settle these rows and hands them to the exact pass.  (2) Masked rows with
    fewer than k candidates at finite distance (disjoint observed sets): the row holds only those (advisor finding:
    the fill used to write past the row)."""
    import torch
    for name, X32, mask, k in synth.tie_cases():
        rp, cl, ww, _ = _oracle_csr(oracle, X32, mask, k, 0.25)
        rowptr, col, wg = B.cc_knn_weights(X32.shape[0], X32.shape[1], _dev(torch, X32), _dev(torch, mask), k, 0.25)
        assert np.array_equal(rowptr.cpu().numpy(), rp), name
        assert np.array_equal(col.cpu().numpy(), cl), name
        assert np.array_equal(wg.cpu().numpy(), ww), name          # same fp64 distance, same exp, one rounding to fp32
    # two groups of rows that observe disjoint coordinates: 2 candidates at finite distance, k = 4
    rng = np.random.default_rng(8)
    X32 = rng.normal(size=(6, 4)).astype(np.float32)
    mask = np.array([[1, 1, 0, 0]] * 3 + [[0, 0, 1, 1]] * 3, np.uint8)
    rp, cl, ww, dropped = _oracle_csr(oracle, X32, mask, 4, 0.5)
    assert dropped > 0 and rp[-1] == 12                             # the oracle lists infinite-distance pairs; weight 0
    rowptr, col, wg = B.cc_knn_weights(6, 4, _dev(torch, X32), _dev(torch, mask), 4, 0.5)
    assert np.array_equal(rowptr.cpu().numpy(), rp) and np.array_equal(col.cpu().numpy(), cl)
    assert np.allclose(wg.cpu().numpy(), ww, rtol=1e-6)
    # larger: random masks at 70 % missing leave many pairs without a common coordinate
    X32 = rng.normal(size=(300, 5)).astype(np.float32)
    mask = (rng.random(size=X32.shape) >= 0.7).astype(np.uint8)
    mask[:, 0] |= (mask.sum(1) == 0).astype(np.uint8)
    rp, cl, ww, _ = _oracle_csr(oracle, X32, mask, 12, 0.125)
    rowptr, col, wg = B.cc_knn_weights(300, 5, _dev(torch, X32), _dev(torch, mask), 12, 0.125)
    assert np.array_equal(rowptr.cpu().numpy(), rp) and np.array_equal(col.cpu().numpy(), cl)
    assert np.allclose(wg.cpu().numpy(), ww, rtol=1e-6)


def test_large_phi_underflowing_weights_end_to_end(B, oracle):
    """raising phi sends most k-NN weights to 0.  A weight that is 0 in fp32 is an absent pair (S24):
    cc_knn_weights drops those entries in both directions, so what it returns is what cc_create accepts, and the
    solve on it follows the oracle's on the same graph."""
    import torch
    wl = synth.make("popres", n=500, phi=512.0)
    rp, cl, ww, dropped = _oracle_csr(oracle, wl.X, None, wl.k, wl.phi)
    assert dropped > 500 and rp[-1] > 1000                          # a real mix of underflowed and live pairs
    X = _dev(torch, wl.X)
    rowptr, col, wg = B.cc_knn_weights(wl.n, wl.p, X, None, wl.k, wl.phi)
    assert np.array_equal(rowptr.cpu().numpy(), rp) and np.array_equal(col.cpu().numpy(), cl)
    assert np.allclose(wg.cpu().numpy(), ww, rtol=1e-6, atol=0) and float(wg.min()) > 0.0
    h = B.cc_create(wl.n, wl.p, X, None, rowptr, col, wg, None)     # used to fail with CC_EGRAPH (w <= 0)
    up = cl > np.repeat(np.arange(wl.n), np.diff(rp))
    ei, ej = np.repeat(np.arange(wl.n), np.diff(rp))[up].astype(np.int32), cl[up].astype(np.int32)
    w64 = wg.cpu().numpy()[up].astype(np.float64)
    ref = oracle.path(wl.X.astype(np.float64), None, ei, ej, w64, [0.5, 20.0], 60, proj_method=1)
    U = torch.empty(wl.n, wl.p, device="cuda:0")
    lab = torch.empty(wl.n, dtype=torch.int32, device="cuda:0")
    for g, r in zip([0.5, 20.0], ref):
        B.cc_solve(h, g, 0.0, 60)
        B.cc_get_U(h, -1, U)
        _, kc = B.cc_clusters(h, -1, lab)
        assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= 1e-4
        assert kc == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"])
    B.cc_destroy(h)


@pytest.mark.parametrize("name,kw,phi,norm", [("genotype", dict(n=52, p=3001), 0.01, False),
                                              ("dense_weight", dict(n=200, p=64, n_clusters=4), 0.005, True),
                                              ("expression", dict(n=70, p=333), 0.002, False),
                                              # few pair tiles, many columns: the column-sliced path (plain and masked)
                                              ("genotype", dict(n=52, p=40000), 0.002, True),
                                              ("expression", dict(n=30, p=5000), 0.0002, False)])
def test_dense_weights_match_oracle(B, oracle, name, kw, phi, norm):
    """a0 for complete graphs against the oracle's eq. 8 with all pairs (incl. masked rule S11, S8)."""
    import torch
    wl = synth.make(name, **kw)
    ei, ej, w, _ = oracle.complete_graph(wl.X.astype(np.float64), wl.mask, phi, normalize=norm)
    Wref = np.zeros((wl.n, wl.n))
    Wref[ei, ej] = w
    Wref = Wref + Wref.T
    W = B.cc_dense_weights(wl.n, wl.p, _dev(torch, wl.X), _dev(torch, wl.mask), phi, normalize=norm).cpu().numpy()
    assert np.array_equal(W, W.T) and np.all(np.diag(W) == 0)
    assert np.abs(W - Wref).max() <= 2e-5 * Wref.max()


def test_graph_utilities(B, oracle):
    """f4: components of the k-NN graph and the smallest connected k, against a plain
    union-find over the oracle's brute-force graphs."""
    import torch

    def components(n, ei, ej):
        par = list(range(n))

        def find(x):
            while par[x] != x:
                par[x] = par[par[x]]
                x = par[x]
            return x
        for a, b in zip(ei, ej):
            ra, rb = find(int(a)), find(int(b))
            if ra != rb:
                par[max(ra, rb)] = min(ra, rb)
        roots = [find(i) for i in range(n)]
        order = {r: k for k, r in enumerate(sorted(set(roots)))}
        return np.array([order[r] for r in roots], np.int32)

    wl = synth.make("tiny")
    X64 = wl.X.astype(np.float64)
    ei, ej, w, _ = oracle.knn_graph(X64, None, wl.k, 0.5)
    ref = components(wl.n, ei, ej)
    rp, cl, _w = oracle.to_csr(wl.n, ei, ej, w)
    lab = torch.empty(wl.n, dtype=torch.int32, device="cuda:0")
    _, k = B.cc_graph_components(wl.n, _dev(torch, rp.astype(np.int64)), _dev(torch, cl.astype(np.int32)), lab)
    assert k == ref.max() + 1 and np.array_equal(lab.cpu().numpy(), ref)
    assert k > 1                                   # the tiny config's 5-NN graph is disconnected
    kref = -1
    for kk in range(1, 41):
        e1, e2, _a, _b = oracle.knn_graph(X64, None, kk, 0.0)
        if components(wl.n, e1, e2).max() == 0:
            kref = kk
            break
    assert B.cc_smallest_connected_k(wl.n, wl.p, _dev(torch, wl.X), None, 40) == kref
    assert B.cc_smallest_connected_k(wl.n, wl.p, _dev(torch, wl.X), None, max(1, kref - 1)) == -1


def test_projection_of_the_path_on_given_directions(B, oracle):
    """f2 (part): (U - xbar) P on the device against the plain fp64 product, masked data (xbar = observed means)."""
    import torch
    wl = synth.make("expression", n=30, p=203)
    X64 = wl.X.astype(np.float64)
    ei, ej, w, _ = oracle.knn_graph(X64, wl.mask, 4, 0.002)
    rp, cl, ww = oracle.to_csr(wl.n, ei, ej, w)
    h = B.cc_create(wl.n, wl.p, _dev(torch, wl.X), _dev(torch, wl.mask), _dev(torch, rp.astype(np.int64)),
                    _dev(torch, cl.astype(np.int32)), _dev(torch, ww.astype(np.float32)), None)
    B.cc_path(h, [1.0, 10.0], 0.0, 20)
    rng = np.random.default_rng(0)
    P = rng.normal(size=(wl.p, 2)).astype(np.float32)
    xbar = oracle.column_means(X64, wl.mask)
    U = torch.empty(wl.n, wl.p)
    for gi in (0, 1, -1):
        B.cc_get_U(h, gi, U)
        ref = (U.numpy().astype(np.float64) - xbar[None, :]) @ P.astype(np.float64)
        out_h = torch.empty(wl.n, 2)
        out_d = torch.empty(wl.n, 2, device="cuda:0")
        B.cc_get_projection(h, gi, _dev(torch, P), out_h)
        B.cc_get_projection(h, gi, _dev(torch, P), out_d)
        assert np.array_equal(out_h.numpy(), out_d.cpu().numpy())
        assert np.abs(out_h.numpy() - ref).max() <= 1e-4 * max(1.0, np.abs(ref).max())
    B.cc_destroy(h)


def test_full_size_large_sparse_properties(B):
    """configs[3] at full size, in the launch configuration bench.py times: properties that hold at
    any size -- Phi non-increasing, column sums of U equal those of X when nothing
    is missing (pin P6: 1'L = 0), shrink factors in [0,1], and U rows of fused pairs O(kappa)-close."""
    import torch
    wl = synth.make("large_sparse")
    X = _dev(torch, wl.X)
    rowptr, col, w = B.cc_knn_weights(wl.n, wl.p, X, None, wl.k, 0.01)
    h = B.cc_create(wl.n, wl.p, X, None, rowptr, col, w, None)
    for g in (3.0, 30.0):
        it, phi, _ = B.cc_solve(h, g, 0.0, 30)
        ph, dd = B.cc_get_history(h)
        assert it == 30 and np.all(np.diff(ph) <= 1e-6 * np.abs(ph[:-1]))
        assert np.all(dd > 0)
    U = torch.empty(wl.n, wl.p, device="cuda:0")
    B.cc_get_U(h, -1, U)
    cs_u, cs_x = U.double().sum(0).cpu().numpy(), X.double().sum(0).cpu().numpy()
    # exact for an exact projection; the CG stop rule (proj_tol) leaves a column-sum residual of this order
    rel = np.abs(cs_u - cs_x).max() / X.double().abs().sum(0).max().item()
    assert rel <= 1e-4, rel
    lab = torch.empty(wl.n, dtype=torch.int32, device="cuda:0")
    _, k = B.cc_clusters(h, -1, lab)
    assert 1 <= k <= wl.n
    # labels are canonical: label of a node <= its index rank, first node has label 0, labels are dense
    l = lab.cpu().numpy()
    assert l[0] == 0 and l.max() == k - 1 and np.array_equal(np.unique(l), np.arange(k))
    B.cc_destroy(h)


@pytest.mark.parametrize("name,kw,k,phi,alpha,scale,norm", [
    ("genotype", dict(n=52, p=4682), 4, 1e-3, 0.5, 1.0, False),      # HGDP-like (L166-L178): k = 4, alpha = 0.5
    ("popres", dict(n=1500), 40, 0.0, 0.5, 0.01, True),              # POPRES-like (L182-L186), uniform weights
    ("expression", dict(n=70, p=333), 5, 1e-3, 0.3, 0.2, False),     # masked x-distance (S11) inside eq. 9
    ("large_sparse", dict(n=3000), 10, 1e-3, 0.8, 0.05, False),
])
def test_composite_distance_weights_match_oracle(B, oracle, name, kw, k, phi, alpha, scale, norm):
    """f4: eq. 9 with modulo longitude differences (S27), then eq. 8 on the composite distance."""
    import torch
    wl = synth.make(name, **kw)
    Y = synth.side_coordinates(wl.n, 1, scale)
    period = [360.0 * scale, 0.0]
    ei, ej, w, _ = oracle.composite_knn_graph(wl.X.astype(np.float64), wl.mask, Y.astype(np.float64), period, alpha, k, phi,
                                              normalize=norm)
    rp, cl, ww = oracle.to_csr(wl.n, ei, ej, w)
    rowptr, col, wg = B.cc_knn_weights(wl.n, wl.p, _dev(torch, wl.X), _dev(torch, wl.mask), k, phi, normalize=norm,
                                       Y=_dev(torch, Y), period=period, alpha=alpha)
    assert np.array_equal(rowptr.cpu().numpy(), rp)
    assert np.array_equal(col.cpu().numpy(), cl)
    assert np.abs(wg.cpu().numpy() - ww).max() <= 2e-5 * ww.max()
    # the wrap matters on this recipe: without it the graph is a different one
    ei2, ej2, _, _ = oracle.composite_knn_graph(wl.X.astype(np.float64), wl.mask, Y.astype(np.float64), None, alpha, k, phi)
    assert len(ei2) != len(ei) or not (np.array_equal(ei2, ei) and np.array_equal(ej2, ej))
    h = B.cc_create(wl.n, wl.p, _dev(torch, wl.X), _dev(torch, wl.mask), rowptr, col, wg, None)
    assert B.cc_get_counts(h)["n_pairs"] == len(ei)
    B.cc_destroy(h)


@pytest.mark.parametrize("name,kw,k,phi,alpha,radius,norm", [
    ("genotype", dict(n=52, p=4682), 4, 1e-3, 0.5, 57.29578, False),   # HGDP-like, geodesic in degrees of arc
    ("popres", dict(n=1500), 40, 0.0, 0.5, 0.5, True),                 # POPRES-like, uniform weights
    ("expression", dict(n=70, p=333), 5, 1e-7, 0.3, 6371.0, False),    # masked x-distance, geodesic in km
    ("large_sparse", dict(n=3000), 10, 1e-3, 0.8, 3.0, False),
])
def test_geodesic_distance_weights_match_oracle(B, oracle, name, kw, k, phi, alpha, radius, norm):
    """f4: eq. 9 with the geodesic alternative of L137 (S28), then eq. 8 on the composite distance."""
    import torch
    wl = synth.make(name, **kw)
    Y = synth.side_coordinates(wl.n, 3, 1.0)             # (longitude, latitude) in degrees, groups across +-180
    ei, ej, w, dd = oracle.composite_knn_graph(wl.X.astype(np.float64), wl.mask, Y.astype(np.float64), None, alpha, k, phi,
                                               normalize=norm, geodesic_radius=radius)
    rp, cl, ww = oracle.to_csr(wl.n, ei, ej, w)
    rowptr, col, wg = B.cc_knn_weights(wl.n, wl.p, _dev(torch, wl.X), _dev(torch, wl.mask), k, phi, normalize=norm,
                                       Y=_dev(torch, Y), alpha=alpha, geodesic_radius=radius)
    assert np.array_equal(rowptr.cpu().numpy(), rp)
    assert np.array_equal(col.cpu().numpy(), cl)
    assert np.abs(wg.cpu().numpy() - ww).max() <= 2e-5 * ww.max()
    # it is not the wrapped Euclidean distance in degrees: that graph differs (cos(lat) shrinks the longitude term)
    ei2, ej2, _, _ = oracle.composite_knn_graph(wl.X.astype(np.float64), wl.mask, Y.astype(np.float64), [360.0, 0.0], alpha, k, phi)
    if radius == 57.29578:
        assert len(ei2) != len(ei) or not (np.array_equal(ei2, ei) and np.array_equal(ej2, ej))


def test_geodesic_distance_limits_and_errors(B, oracle):
    import torch
    wl = synth.make("large_sparse", n=2000)
    X = _dev(torch, wl.X)
    Y = _dev(torch, synth.side_coordinates(wl.n, 2))
    r0, c0, w0 = B.cc_knn_weights(wl.n, wl.p, X, None, 8, 0.01)
    r1, c1, w1 = B.cc_knn_weights(wl.n, wl.p, X, None, 8, 0.01, Y=Y, alpha=1.0, geodesic_radius=6371.0)   # eq. 9 -> eq. 8
    assert torch.equal(r0, r1) and torch.equal(c0, c1) and float((w0 - w1).abs().max()) <= 1e-5 * float(w0.max())
    # alpha = 0 with positions on the equator / a meridian: distances are R |dlon| (short way round) and R |dlat|
    ll = np.array([[179.0, 0.0], [-179.0, 0.0], [-170.0, 0.0], [120.0, 0.0], [0.0, 80.0], [0.0, 70.0], [0.0, -10.0]], dtype=np.float32)
    Xs = np.zeros((7, 3), dtype=np.float32)
    rp, cl, ww = B.cc_knn_weights(7, 3, _dev(torch, Xs), None, 1, 1.0, Y=_dev(torch, ll), alpha=0.0, geodesic_radius=1.0)
    ei, ej, w, dd = oracle.composite_knn_graph(Xs.astype(np.float64), None, ll.astype(np.float64), None, 0.0, 1, 1.0,
                                               geodesic_radius=1.0)
    rpo, clo, wwo = oracle.to_csr(7, ei, ej, w)
    assert np.array_equal(rp.cpu().numpy(), rpo) and np.array_equal(cl.cpu().numpy(), clo)
    assert (0, 1) in set(zip(ei.tolist(), ej.tolist()))                       # 179 E and 179 W are neighbours
    assert np.abs(ww.cpu().numpy() - wwo).max() <= 1e-6
    for bad in (dict(alpha=1.5), dict(geodesic_radius=0.0), dict(geodesic_radius=-1.0), dict(geodesic_radius=float("inf"))):
        args = dict(Y=Y, alpha=0.5, geodesic_radius=1.0)
        args.update(bad)
        with pytest.raises(B.CCError) as e:
            B.cc_knn_weights(wl.n, wl.p, X, None, 8, 0.01, **args)
        assert e.value.code == B.CC_EINVAL
    with pytest.raises(B.CCError) as e:
        B.cc_knn_weights(wl.n, wl.p, X, None, 8, 0.01, Y=torch.zeros(wl.n, 3, device="cuda:0"), alpha=0.5, geodesic_radius=1.0)
    assert e.value.code == B.CC_EINVAL


def test_composite_distance_limits_and_errors(B, oracle):
    import torch
    wl = synth.make("large_sparse", n=2000)
    X = _dev(torch, wl.X)
    Y = _dev(torch, synth.side_coordinates(wl.n, 2))
    r0, c0, w0 = B.cc_knn_weights(wl.n, wl.p, X, None, 8, 0.01)
    r1, c1, w1 = B.cc_knn_weights(wl.n, wl.p, X, None, 8, 0.01, Y=Y, period=[360.0, 0.0], alpha=1.0)   # eq. 9 -> eq. 8
    assert torch.equal(r0, r1) and torch.equal(c0, c1) and float((w0 - w1).abs().max()) <= 1e-5 * float(w0.max())
    for bad in (dict(alpha=1.5), dict(alpha=-0.1), dict(period=[-1.0, 0.0])):
        args = dict(Y=Y, period=[360.0, 0.0], alpha=0.5)
        args.update(bad)
        with pytest.raises(B.CCError) as e:
            B.cc_knn_weights(wl.n, wl.p, X, None, 8, 0.01, **args)
        assert e.value.code == B.CC_EINVAL
    with pytest.raises(B.CCError) as e:
        B.cc_knn_weights(wl.n, wl.p, X, None, 8, 0.01, Y=torch.zeros(wl.n, 5, device="cuda:0"), alpha=0.5)
    assert e.value.code == B.CC_EINVAL
