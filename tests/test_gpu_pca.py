"""GPU tests of f2 (-m gpu): cc_principal_components (reading S25) against the oracle's SVD
definition, and the path read back as coordinates on those directions (cc_get_projection).

An eigenvector is unique up to sign only when its eigenvalue is separated from its neighbours, so each direction
is compared as the sine of its angle to the oracle's, scaled by the relative gap; what is always unique
(variances, orthonormality, the span) is compared directly."""
import numpy as np
import pytest

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


def _chain_handle(B, torch, X, mask, **prm):
    """A handle on a path graph 0-1-...-(n-1): the directions do not depend on the graph."""
    n, p = X.shape
    rowptr = np.zeros(n + 1, np.int64)
    col = []
    for i in range(n):
        nb = [j for j in (i - 1, i + 1) if 0 <= j < n]
        col += nb
        rowptr[i + 1] = rowptr[i] + len(nb)
    col = np.array(col, np.int32)
    w = np.ones(len(col), np.float32)
    return B.cc_create(n, p, _dev(torch, X), _dev(torch, mask), _dev(torch, rowptr), _dev(torch, col), _dev(torch, w),
                       B.cc_default_params(**prm) if prm else None)


def _check_against_oracle(oracle, X, mask, Pg, var, q, tol_sin=2e-5):
    Pr, vr = oracle.principal_components(X.astype(np.float64), mask, min(q + 1, X.shape[1]))
    Pg = Pg.astype(np.float64)
    assert np.allclose(var, vr[:q], rtol=0, atol=1e-6 * vr[0])
    assert np.abs(Pg.T @ Pg - np.eye(q)).max() <= 1e-5
    for k in range(q):
        # separation of eigenvalue k from its neighbours, relative to the largest
        nb = [abs(vr[k] - vr[j]) for j in (k - 1, k + 1) if 0 <= j < len(vr)]
        gap = min(nb) / vr[0] if nb else 1.0
        sin = np.linalg.norm(Pg[:, k] - (Pr[:, k] @ Pg[:, k]) * Pr[:, k])
        assert sin <= tol_sin / max(gap, 1e-3), (k, sin, gap)
        # sign convention: the entry of largest magnitude is positive
        assert Pg[np.argmax(np.abs(Pg[:, k])), k] > 0
        big = np.sort(np.abs(Pr[:, k]))
        if gap > 1e-2 and big[-1] - big[-2] > 1e-3:
            assert np.abs(Pg[:, k] - Pr[:, k]).max() <= 10 * tol_sin / gap
    return Pr, vr


@pytest.mark.parametrize("name,kw,q", [
    ("tiny", {}, 2),
    ("large_sparse", {"n": 5000}, 3),
    ("expression", {"n": 60, "p": 500}, 2),        # masked
    ("popres", {}, 2),                             # p = 10 < 16: the block is the whole space
    ("genotype", {"n": 200, "p": 3000}, 3),        # few rows, many columns: the column-sliced product
    ("dense_weight", {"n": 700, "p": 33}, 8),      # p not a multiple of 4, q at its maximum
])
def test_principal_components_against_oracle(B, oracle, name, kw, q):
    import torch
    wl = synth.make(name, **kw)
    h = _chain_handle(B, torch, wl.X, wl.mask)
    P = torch.empty(wl.p, q, device="cuda:0")
    _, var, res, its = B.cc_principal_components(h, P, maxit=400, tol=1e-6)
    assert max(res) <= 1e-6 and 1 <= its <= 400
    _check_against_oracle(oracle, wl.X, wl.mask, P.cpu().numpy(), np.array(var), q)
    # host output is the same bytes; a second call repeats them (fixed start block, fixed reduction orders)
    Ph = torch.empty(wl.p, q)
    _, var2, _, its2 = B.cc_principal_components(h, Ph, maxit=400, tol=1e-6)
    assert np.array_equal(Ph.numpy(), P.cpu().numpy()) and var2 == var and its2 == its
    B.cc_destroy(h)


def test_path_coordinates_on_the_principal_components(B, oracle):
    """L144/L210 end to end: the gamma path read back as n x 2 coordinates on the first two principal components of
    the original data, against the oracle's path projected on the oracle's components (up to the sign convention,
    which both sides state the same way)."""
    import torch
    import helpers as H
    wl = synth.make("expression", n=80, p=300)
    prob = H.build_problem(oracle, wl)
    h = H.gpu_create(B, torch, prob)
    gammas = [float(g) for g in synth.gamma_grid(0.5, 50.0, 4)]
    B.cc_path(h, gammas, 0.0, 40)
    ref = H.oracle_path(oracle, prob, gammas, 40)
    P = torch.empty(wl.p, 2, device="cuda:0")
    _, var, res, _ = B.cc_principal_components(h, P)
    Pr, vr = oracle.principal_components(prob["X64"], prob["mask"], 2)
    assert min(abs(vr[0] - vr[1]) / vr[0], 1.0) > 1e-2      # the recipe separates the first two directions
    out = torch.empty(wl.n, 2)
    for gi, r in enumerate(ref):
        B.cc_get_projection(h, gi, P, out)
        want = oracle.project_on_components(prob["X64"], prob["mask"], r["U"], Pr)
        assert np.linalg.norm(out.numpy() - want) <= 1e-4 * max(np.linalg.norm(want), 1e-30)
    B.cc_destroy(h)


def test_principal_components_edge_cases(B, oracle):
    import torch
    # rank-one data: one direction, the second comes back as a zero vector with variance 0 (header contract)
    rng = np.random.default_rng(4)
    g = np.array([1.0, -2.0, 0.5, 4.0, 0.0], np.float32)
    t = rng.standard_normal(40).astype(np.float32)
    X = (0.75 + t[:, None] * g[None, :]).astype(np.float32)
    h = _chain_handle(B, torch, X, None)
    P = torch.empty(5, 2)
    _, var, res, its = B.cc_principal_components(h, P)
    Pr, vr = oracle.principal_components(X.astype(np.float64), None, 1)
    assert np.isclose(var[0], vr[0], rtol=1e-6) and var[1] <= 1e-6 * var[0]
    assert np.abs(P[:, 0].numpy() - Pr[:, 0]).max() <= 1e-6
    assert np.abs(P[:, 1].numpy()).max() <= 1e-6
    with pytest.raises(B.CCError) as e:
        B.cc_principal_components(h, torch.empty(5, 6))          # q > p
    assert e.value.code == B.CC_EINVAL
    with pytest.raises(B.CCError) as e:
        B.cc_principal_components(h, torch.empty(5, 2), maxit=0)
    assert e.value.code == B.CC_EINVAL
    B.cc_destroy(h)
    # p = 2, n = 3; q = p
    X = np.array([[0.0, 0.0], [2.0, 1.0], [4.0, 2.5]], np.float32)
    h = _chain_handle(B, torch, X, None)
    P = torch.empty(2, 2)
    _, var, _, _ = B.cc_principal_components(h, P)
    _check_against_oracle(oracle, X, None, P.numpy(), np.array(var), 2)
    # the MM state is untouched: a solve after the call equals a solve on a fresh handle
    U1, U2 = torch.empty(3, 2), torch.empty(3, 2)
    B.cc_solve(h, 0.3, 0.0, 15)
    B.cc_get_U(h, -1, U1)
    h2 = _chain_handle(B, torch, X, None)
    B.cc_solve(h2, 0.3, 0.0, 15)
    B.cc_get_U(h2, -1, U2)
    assert np.array_equal(U1.numpy(), U2.numpy())
    B.cc_destroy(h)
    B.cc_destroy(h2)


def test_principal_components_full_size(B, oracle):
    """The bench shapes at full size: large-sparse (100,000 x 64), expression-like (100 x 5,000, masked) and
    genotype-like (52 x 200,000: the column-sliced product)."""
    import torch
    for name, q in (("large_sparse", 2), ("expression", 2), ("genotype", 2)):
        wl = synth.make(name)
        h = _chain_handle(B, torch, wl.X, wl.mask)
        P = torch.empty(wl.p, q, device="cuda:0")
        _, var, res, its = B.cc_principal_components(h, P, maxit=400, tol=1e-6)
        assert max(res) <= 1e-6
        _check_against_oracle(oracle, wl.X, wl.mask, P.cpu().numpy(), np.array(var), q)
        B.cc_destroy(h)
