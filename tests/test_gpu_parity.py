"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI (paper_1409_2065_b200.binding),
against the fp64 oracle on the same seeded inputs.  Bar (BASELINE.json north_star): relative
Frobenius error <= 1e-4 after a fixed iteration count, identical cluster labels at every gamma."""
import json
import os

import numpy as np
import pytest

import helpers as H
from paper_1409_2065_b200 import synth

pytestmark = pytest.mark.gpu
TOL = 1e-4   # north_star: "relative Frobenius error <= 1e-4 (fp32)"


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_2065_b200 import binding
    return binding


@pytest.fixture(scope="module")
def torch_():
    import torch
    return torch


def _run_path(B, torch, prob, gammas, iters, ref, **prm):
    h = H.gpu_create(B, torch, prob, **prm)
    n, p = prob["n"], prob["p"]
    U = torch.empty(n, p, device="cuda:0")
    lab = torch.empty(n, dtype=torch.int32, device="cuda:0")
    out = []
    try:
        for g, r in zip(gammas, ref):
            it, phi, _ = B.cc_solve(h, g, 0.0, iters)
            assert it == iters
            B.cc_get_U(h, -1, U)
            _, k = B.cc_clusters(h, -1, lab)
            ph, dd = B.cc_get_history(h)
            err = H.relerr(U.cpu().numpy().astype(np.float64), r["U"])
            assert err <= TOL, (g, err)
            assert k == r["nclusters"], (g, k, r["nclusters"])
            assert np.array_equal(lab.cpu().numpy(), r["labels"]), g
            # Phi and d histories: d_m^2 - eps is a sum of squares of O(kappa) differences of O(1) fp32 numbers,
            # so d carries ~1e-4 relative fp32 noise; U itself is held to 1e-4
            assert np.allclose(ph, r["phi"][:len(ph)], rtol=1e-4), g
            assert np.allclose(dd, r["d"][:len(dd)], rtol=5e-4), g
            # MM descent property up to fp32 noise in the state
            assert np.all(np.diff(ph) <= 1e-6 * np.abs(ph[:-1])), g
            out.append((err, k))
    finally:
        B.cc_destroy(h)
    return out


def test_tiny_path_matches_oracle_and_golden(B, torch_, oracle):
    wl = synth.make("tiny")
    prob = H.build_problem(oracle, wl)
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "tiny_path.json")))
    gammas, iters = gold["gammas"], gold["iters"]
    assert len(prob["ei"]) == gold["n_pairs"]
    ref = H.oracle_path(oracle, prob, gammas, iters)
    out = _run_path(B, torch_, prob, gammas, iters, ref)
    assert [k for _, k in out] == [g["nclusters"] for g in gold["per_gamma"]]


def test_tiny_long_run(B, torch_, oracle):
    """One long run (fp32 drift grows with the iteration count)."""
    wl = synth.make("tiny")
    prob = H.build_problem(oracle, wl)
    ref = H.oracle_path(oracle, prob, [300.0], 3000)
    _run_path(B, torch_, prob, [300.0], 3000, ref)


def test_expression_like_masked(B, torch_, oracle):
    """Missing data, rows wider than one 128-column chunk with a ragged tail."""
    wl = synth.make("expression", n=40, p=301)
    prob = H.build_problem(oracle, wl)
    gammas = [0.5, 5.0, 50.0]
    ref = H.oracle_path(oracle, prob, gammas, 100)
    _run_path(B, torch_, prob, gammas, 100, ref)


def test_large_sparse_reduced(B, torch_, oracle):
    """Same generator as configs[3] at n=3000: several row blocks, hubs, CG-projection oracle."""
    wl = synth.make("large_sparse", n=3000, p=64, n_clusters=10)
    prob = H.build_problem(oracle, wl)
    gammas = [1.0, 30.0, 300.0]
    ref = H.oracle_path(oracle, prob, gammas, 100, proj_method=1)
    out = _run_path(B, torch_, prob, gammas, 100, ref)
    assert out[-1][1] < 100   # the path really fuses


def test_large_sparse_20k_end_to_end(B, torch_, oracle):
    """configs[3]'s generator at n = 20,000 (hundreds of row blocks, hubs): graph built on the GPU by
    cc_knn_weights and required to equal the oracle's brute-force graph, then the MM iteration on it."""
    torch = torch_
    wl = synth.make("large_sparse", n=20000, p=64, n_clusters=20)
    prob = H.build_problem(oracle, wl)
    dev = torch.device("cuda:0")
    X = torch.from_numpy(wl.X).to(dev)
    rowptr, col, w = B.cc_knn_weights(wl.n, wl.p, X, None, wl.k, prob["phi"])
    assert np.array_equal(rowptr.cpu().numpy(), prob["rowptr"])
    assert np.array_equal(col.cpu().numpy(), prob["col"])
    assert np.abs(w.cpu().numpy() - prob["wcsr32"]).max() <= 1e-5 * prob["wcsr32"].max()
    gammas = [3.0, 60.0]
    ref = H.oracle_path(oracle, prob, gammas, 15, proj_method=1)
    _run_path(B, torch, prob, gammas, 15, ref)


@pytest.mark.parametrize("phi", [0.0, 10.0])
def test_popres_like_low_p_large_k(B, torch_, oracle, phi):
    """low p (row groups of 4 lanes), k = 40, uniform weights (phi = 0) and phi = 10."""
    wl = synth.make("popres", n=400, phi=phi)
    prob = H.build_problem(oracle, wl)
    gammas = [0.05, 0.5, 5.0]     # oracle: 400 -> 22 -> 1 clusters (phi = 0), 400 -> 344 -> 20 (phi = 10)
    ref = H.oracle_path(oracle, prob, gammas, 150, proj_method=1)
    out = _run_path(B, torch_, prob, gammas, 150, ref)
    print("popres phi", phi, "clusters", [k for _, k in out])


def test_popres_full_size_dense_inverse_from_l2(B, torch_, oracle):
    """The POPRES-like configuration at its full size (3000 x 10, k = 40): a2 is the dense inverse formed once by the blocked
    Gauss-Jordan and applied from L2 (k_apply_inv_wide); 94 pivot blocks, the last one ragged (3000 = 93 x 32 + 24)."""
    wl = synth.make("popres")
    assert wl.n == 3000 and wl.p == 10
    prob = H.build_problem(oracle, wl)
    gammas = [0.05, 1.0]
    ref = H.oracle_path(oracle, prob, gammas, 40, proj_method=1)
    _run_path(B, torch_, prob, gammas, 40, ref)


@pytest.mark.parametrize("p,k", [(3, 12), (5, 20), (14, 16), (17, 10), (21, 10), (26, 10), (30, 8)])
def test_dense_inverse_from_l2_every_width(B, torch_, oracle, p, k):
    """k_apply_inv_wide has one instantiation per ld / 4 (ld = p rounded up to 4: 4, 8, 16, 20, 24, 28, 32 here; 12 is the
    POPRES shape above): n = 450 > 384 points, so a2 is the blocked Gauss-Jordan inverse applied from L2 (15 pivot blocks,
    the last of 2 rows)."""
    wl = synth.make("popres", n=450, p=p, k=k, phi=2.0)
    prob = H.build_problem(oracle, wl)
    gammas = [0.05, 0.8]
    ref = H.oracle_path(oracle, prob, gammas, 30, proj_method=1)
    _run_path(B, torch_, prob, gammas, 30, ref)


def test_path_with_stop_rule_expression_masked(B, torch_, oracle):
    """cc_path with tol > 0 on a masked instance: per-gamma iteration counts (S3), labels and U follow the oracle."""
    torch = torch_
    wl = synth.make("expression", n=60, p=400)
    prob = H.build_problem(oracle, wl)
    gammas = [float(g) for g in synth.gamma_grid(1.0, 60.0, 5)]
    tol = 1e-4
    ref = oracle.path(prob["X64"], prob["mask"], prob["ei"], prob["ej"], prob["w64"], gammas, 3000, tol=tol, min_it=10)
    h = H.gpu_create(B, torch, prob)
    its, phis = B.cc_path(h, gammas, tol, 3000)
    U = torch.empty(wl.n, wl.p)
    lab = torch.empty(wl.n, dtype=torch.int32)
    for gi, r in enumerate(ref):
        assert abs(its[gi] - r["iters"]) <= max(3, r["iters"] // 20), (gi, its[gi], r["iters"])
        B.cc_get_U(h, gi, U)
        # the two runs may stop a few iterations apart, each iteration moves U by O(kappa * step): compare loosely
        assert H.relerr(U.numpy().astype(np.float64), r["U"]) <= 2e-3, gi
        _, k = B.cc_clusters(h, gi, lab)
        assert abs(k - r["nclusters"]) <= max(1, r["nclusters"] // 20), (gi, k, r["nclusters"])
    B.cc_destroy(h)


@pytest.mark.parametrize("n,p,deg,miss", [(50, 7, 3.0, 0.0), (33, 130, 4.0, 0.15), (200, 2, 6.0, 0.0),
                                          (17, 1, 2.0, 0.0)])
def test_ragged_shapes_random_graphs(B, torch_, oracle, n, p, deg, miss):
    """p not a multiple of 4, p < 4, p spanning two chunks; disconnected graphs with isolated nodes."""
    rng = np.random.default_rng(n * 1000 + p)
    X = (rng.normal(size=(n, p)) + 2.0 * rng.integers(0, 3, size=(n, 1))).astype(np.float32)
    ei, ej, w = synth.random_graph(n, deg, seed=n + p)
    mask = None
    if miss > 0:
        mask = (rng.random(size=(n, p)) >= miss).astype(np.uint8)
        mask[0, :] = 1
    w32 = w.astype(np.float32)
    rowptr, col, wc = oracle.to_csr(n, ei, ej, w32.astype(np.float64))
    prob = {"X64": X.astype(np.float64), "mask": mask, "ei": ei, "ej": ej, "w64": w32.astype(np.float64),
            "rowptr": rowptr, "col": col, "wcsr32": wc.astype(np.float32), "n": n, "p": p}
    gammas = [0.3, 3.0, 30.0]
    ref = H.oracle_path(oracle, prob, gammas, 120)
    _run_path(B, torch_, prob, gammas, 120, ref)


def test_empty_graph_and_gamma_zero(B, torch_, oracle):
    """No pairs at all: U = X after any number of iterations (gamma irrelevant);
    gamma = 0 on a real graph: U = X (pin P1)."""
    torch = torch_
    n, p = 20, 5
    rng = np.random.default_rng(1)
    X = rng.normal(size=(n, p)).astype(np.float32)
    prob = {"X64": X.astype(np.float64), "mask": None, "n": n, "p": p, "rowptr": np.zeros(n + 1, np.int64),
            "col": np.zeros(0, np.int32), "wcsr32": np.zeros(0, np.float32)}
    h = H.gpu_create(B, torch, prob)
    B.cc_solve(h, 5.0, 0.0, 30)
    U = torch.empty(n, p, device="cuda:0")
    B.cc_get_U(h, -1, U)
    assert np.abs(U.cpu().numpy() - X).max() <= 1e-6
    lab = torch.empty(n, dtype=torch.int32, device="cuda:0")
    _, k = B.cc_clusters(h, -1, lab)
    assert k == n and np.array_equal(lab.cpu().numpy(), np.arange(n))
    B.cc_destroy(h)
    wl = synth.make("tiny")
    prob = H.build_problem(oracle, wl)
    h = H.gpu_create(B, torch, prob)
    B.cc_solve(h, 0.0, 0.0, 25)
    U = torch.empty(wl.n, wl.p, device="cuda:0")
    B.cc_get_U(h, -1, U)
    assert np.abs(U.cpu().numpy() - wl.X).max() <= 1e-5
    B.cc_destroy(h)


def test_graph_and_eager_launch_modes_are_bit_identical_and_deterministic(B, torch_, oracle):
    torch = torch_
    wl = synth.make("large_sparse", n=2000, p=64, n_clusters=8)
    prob = H.build_problem(oracle, wl)
    outs = []
    for use_graph in (1, 0, 1):
        h = H.gpu_create(B, torch, prob, use_graph=use_graph)
        for g in (5.0, 80.0):
            B.cc_solve(h, g, 0.0, 40)
        U = torch.empty(wl.n, wl.p, device="cuda:0")
        B.cc_get_U(h, -1, U)
        outs.append(U.cpu().numpy().copy())
        B.cc_destroy(h)
    assert np.array_equal(outs[0], outs[1])
    assert np.array_equal(outs[0], outs[2])


@pytest.mark.parametrize("name,kw", [("tiny", {}), ("expression", dict(n=40, p=301)), ("expression", dict(n=100, p=2000)),
                                     ("expression", dict(n=128, p=900)),     # the largest n of the tensor-core projection: K = M = 128
                                     ("expression", dict(n=97, p=37)),       # one slab, ragged K (97 = 12 x 8 + 1) and N (40 -> 48)
                                     ("expression", dict(n=129, p=600)),     # just above: the FFMA register tiles
                                     ("expression", dict(n=12, p=5000))])    # K = 16 of which 12, wide slabs
def test_persistent_kernel_and_stream_kernels_agree(B, torch_, oracle, name, kw):
    """Small n: cc_solve runs the whole MM loop as one persistent kernel (column slabs in shared memory, two grid
    barriers per iteration; for n <= 128 the projection by the inverse is one tcgen05 tile per slab, the inverse resident in
    tensor memory); prm.use_graph = 0 drives the separate stream kernels from the host.  Different summation
    orders, same iteration: both within the tolerance of the oracle, and within 1e-5 of each other, labels equal."""
    torch = torch_
    wl = synth.make(name, **kw)
    prob = H.build_problem(oracle, wl)
    gammas, iters = ([1.0, 100.0, 1000.0], 120) if name == "tiny" else ([0.5, 5.0, 50.0], 60)
    ref = H.oracle_path(oracle, prob, gammas, iters)
    outs, labs = [], []
    for use_graph in (1, 0):
        h = H.gpu_create(B, torch, prob, use_graph=use_graph)
        U = torch.empty(wl.n, wl.p, device="cuda:0")
        lab = torch.empty(wl.n, dtype=torch.int32, device="cuda:0")
        for g, r in zip(gammas, ref):
            it, _, _ = B.cc_solve(h, g, 0.0, iters)
            assert it == iters
            B.cc_get_U(h, -1, U)
            _, k = B.cc_clusters(h, -1, lab)
            assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= TOL, (use_graph, g)
            assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"]), (use_graph, g)
        outs.append(U.cpu().numpy().astype(np.float64))
        B.cc_destroy(h)
    assert H.relerr(outs[0], outs[1]) <= 1e-5


def test_stop_rule_matches_oracle(B, torch_, oracle):
    """tol > 0 (reading S3): the GPU stops at (nearly) the oracle's iteration."""
    torch = torch_
    wl = synth.make("tiny")
    prob = H.build_problem(oracle, wl)
    X, m = prob["X64"], prob["mask"]
    U0, V0 = oracle.cold_start(X, m, prob["ei"], prob["ej"])
    g, tol = 200.0, 1e-4
    rho, eps = oracle.default_rho_eps(X, m, prob["w64"], g)
    r = oracle.mm(X, m, prob["ei"], prob["ej"], prob["w64"], g, rho, eps, U0, V0, 5000, tol=tol, min_it=10)
    h = H.gpu_create(B, torch, prob)
    it, phi, _ = B.cc_solve(h, g, tol, 5000)
    st = B.cc_get_stats(h)
    B.cc_destroy(h)
    assert abs(st["rho"] - rho) <= 1e-6 * rho and abs(st["eps"] - eps) <= 1e-6 * eps
    assert 10 <= it < 5000 and abs(it - r["iters"]) <= max(2, r["iters"] // 50), (it, r["iters"])
    assert abs(phi - r["phi"][-1]) <= 1e-4 * abs(phi)


def test_cc_path_snapshots(B, torch_, oracle):
    torch = torch_
    wl = synth.make("tiny")
    prob = H.build_problem(oracle, wl)
    gammas = [float(g) for g in synth.gamma_grid(1.0, 1e3, 6)]
    ref = H.oracle_path(oracle, prob, gammas, 80)
    h = H.gpu_create(B, torch, prob)
    its, phis = B.cc_path(h, gammas, 0.0, 80)
    assert its == [80] * 6
    U = torch.empty(wl.n, wl.p, device="cuda:0")
    Uh = torch.empty(wl.n, wl.p)
    lab = torch.empty(wl.n, dtype=torch.int32)
    for gi, r in enumerate(ref):
        B.cc_get_U(h, gi, U)
        B.cc_get_U(h, gi, Uh)
        assert np.array_equal(U.cpu().numpy(), Uh.numpy())
        assert H.relerr(Uh.numpy().astype(np.float64), r["U"]) <= TOL
        _, k = B.cc_clusters(h, gi, lab)
        assert k == r["nclusters"] and np.array_equal(lab.numpy(), r["labels"])
        assert abs(phis[gi] - r["phi"][-1]) <= 1e-5 * abs(phis[gi])
    with pytest.raises(B.CCError) as e:
        B.cc_get_U(h, 6, U)
    assert e.value.code == B.CC_ESTATE
    # f_gamma of eq. 1 at the last U against the oracle's plain definition
    st = B.cc_get_stats(h, f_gamma=True, min_margin=True)
    f_ref = oracle.objective(prob["X64"], None, prob["ei"], prob["ej"], prob["w64"], gammas[-1], ref[-1]["U"])
    assert abs(st["f_gamma"] - f_ref) <= 1e-4 * abs(f_ref)
    assert st["min_margin"] >= 0.0
    B.cc_reset(h)
    B.cc_get_U(h, -1, U)
    assert np.array_equal(U.cpu().numpy(), wl.X)
    B.cc_destroy(h)


@pytest.mark.parametrize("name,kw,miss", [("genotype", dict(n=52, p=5001), 0.0), ("dense_weight", dict(n=37, p=130, n_clusters=3), 0.15),
                                          ("genotype", dict(n=64, p=1200), 0.0),       # the largest n: K = N = 64, 272 pair tiles, one column phase
                                          ("genotype", dict(n=5, p=700), 0.0),         # one K step, 6 pair tiles
                                          ("dense_weight", dict(n=61, p=333, n_clusters=4), 0.1),   # masked, ragged rows and columns
                                          ("genotype", dict(n=20, p=40001), 0.0)])     # 313 chunks: every CTA walks 2-3, both buffers reused
def test_dense_small_n_fused_kernel(B, torch_, oracle, name, kw, miss):
    """n <= 64: the warp-specialised fused kernel kd_small_tc (contraction on tcgen05 in the centred form, operand and
    accumulator in tensor memory, TMA tensor copies, pairs by direct differences in packed fp32) against the oracle, labels
    included, with and without missing entries."""
    torch = torch_
    wl = synth.make(name, **kw)
    if miss > 0:
        rng = np.random.default_rng(11)
        wl.mask = (rng.random(size=wl.X.shape) >= miss).astype(np.uint8)
        wl.mask[0, :] = 1
    prob = H.build_problem(oracle, wl)
    n = wl.n
    W = np.zeros((n, n), np.float32)
    W[prob["ei"], prob["ej"]] = prob["w64"].astype(np.float32)
    W = W + W.T
    gammas = [float(g) for g in synth.gamma_grid(4.0, 40.0, 4)]
    ref = H.oracle_path(oracle, prob, gammas, 60, proj_method=1)
    dev = torch.device("cuda:0")
    mask = None if wl.mask is None else torch.from_numpy(wl.mask).to(dev)
    h = B.cc_create(n, wl.p, torch.from_numpy(wl.X).to(dev), mask, None, None, torch.from_numpy(W).to(dev),
                    B.cc_default_params(dense=1))
    U = torch.empty(n, wl.p, device=dev)
    lab = torch.empty(n, dtype=torch.int32, device=dev)
    for g, r in zip(gammas, ref):
        it, _, _ = B.cc_solve(h, g, 0.0, 60)
        assert it == 60
        B.cc_get_U(h, -1, U)
        _, k = B.cc_clusters(h, -1, lab)
        assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= TOL, g
        assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"]), g
    B.cc_destroy(h)


@pytest.mark.parametrize("name,kw,miss", [("genotype", dict(n=20, p=1000), 0.0),      # 4x4 tiles, one row block, ksplit > 1
                                          ("genotype", dict(n=52, p=5001), 0.0),      # the genotype shape, ragged p
                                          ("dense_weight", dict(n=150, p=200, n_clusters=4), 0.0),   # 8x8 tiles, ragged rows
                                          ("dense_weight", dict(n=70, p=40, n_clusters=3), 0.2),     # masked
                                          ("dense_weight", dict(n=256, p=200, n_clusters=4), 0.0),   # tcgen05 path, ragged N tile
                                          ("dense_weight", dict(n=132, p=64, n_clusters=3), 0.1),    # tcgen05, ragged M and K
                                          ("dense_weight", dict(n=200, p=6, n_clusters=3), 0.0)])    # tcgen05, p far below one tile
def test_dense_mode_complete_graph(B, torch_, oracle, name, kw, miss):
    """prm.dense = 1 (row a9): w is the n x n matrix; closed-form projection, pair tiles."""
    torch = torch_
    wl = synth.make(name, **kw)
    if miss > 0:
        rng = np.random.default_rng(5)
        wl.mask = (rng.random(size=wl.X.shape) >= miss).astype(np.uint8)
        wl.mask[0, :] = 1
    prob = H.build_problem(oracle, wl)
    n = wl.n
    assert len(prob["ei"]) == n * (n - 1) // 2          # no weight underflowed: the graph is complete
    W = np.zeros((n, n), np.float32)
    W[prob["ei"], prob["ej"]] = prob["w64"].astype(np.float32)
    W = W + W.T
    gammas = [float(g) for g in synth.gamma_grid(4.0, 40.0, 6)]   # from no fusion to one cluster
    ref = H.oracle_path(oracle, prob, gammas, 80, proj_method=1)
    assert ref[0]["nclusters"] == n and ref[-1]["nclusters"] == 1
    dev = torch.device("cuda:0")
    mask = None if wl.mask is None else torch.from_numpy(wl.mask).to(dev)
    outs = []
    for use_graph in (1, 0):
        h = B.cc_create(n, wl.p, torch.from_numpy(wl.X).to(dev), mask, None, None, torch.from_numpy(W).to(dev),
                        B.cc_default_params(dense=1, use_graph=use_graph))
        assert B.cc_get_counts(h)["n_pairs"] == n * (n - 1) // 2
        U = torch.empty(n, wl.p, device=dev)
        lab = torch.empty(n, dtype=torch.int32, device=dev)
        ks = []
        for g, r in zip(gammas, ref):
            it, phi, _ = B.cc_solve(h, g, 0.0, 80)
            assert it == 80
            B.cc_get_U(h, -1, U)
            _, k = B.cc_clusters(h, -1, lab)
            ph, dd = B.cc_get_history(h)
            assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= TOL, g
            assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"]), (g, k, r["nclusters"])
            assert np.allclose(ph, r["phi"], rtol=1e-4) and np.allclose(dd, r["d"], rtol=5e-4)
            ks.append(k)
        outs.append(U.cpu().numpy().copy())
        B.cc_destroy(h)
    assert np.array_equal(outs[0], outs[1])
    print(name, kw, "clusters along the path:", ks)


def test_dense_tensor_core_path_through_partial_fusion(B, torch_, oracle):
    """Sharper weights (phi = 6 / median d^2) make the complete graph fuse cluster by cluster: 256 -> 47 -> 4 -> 3.
    With whole clusters fused, most within-cluster pairs go through kd_pairs_tc's direct recompute, the others
    through the Gram blocks; U and the labels must follow the oracle at every gamma."""
    torch = torch_
    wl = synth.make("dense_weight", n=256, p=64, n_clusters=4)
    X64 = wl.X.astype(np.float64)
    si, sj = synth.sample_pairs(wl.n, 200000, 0)
    wl.phi_rule, wl.phi = "fixed", 6.0 / float(np.median(oracle.pair_dist2(X64, None, si, sj)))
    prob = H.build_problem(oracle, wl)
    n = wl.n
    assert len(prob["ei"]) == n * (n - 1) // 2
    W = np.zeros((n, n), np.float32)
    W[prob["ei"], prob["ej"]] = prob["w64"].astype(np.float32)
    W = W + W.T
    gammas = [float(g) for g in synth.gamma_grid(30.0, 3000.0, 6)]
    ref = H.oracle_path(oracle, prob, gammas, 80, proj_method=1)
    ks_ref = [r["nclusters"] for r in ref]
    assert ks_ref[0] == n and 1 < ks_ref[3] < n and ks_ref[-1] <= 4, ks_ref
    dev = torch.device("cuda:0")
    h = B.cc_create(n, wl.p, torch.from_numpy(wl.X).to(dev), None, None, None, torch.from_numpy(W).to(dev),
                    B.cc_default_params(dense=1))
    U = torch.empty(n, wl.p, device=dev)
    lab = torch.empty(n, dtype=torch.int32, device=dev)
    for g, r in zip(gammas, ref):
        B.cc_solve(h, g, 0.0, 80)
        B.cc_get_U(h, -1, U)
        _, k = B.cc_clusters(h, -1, lab)
        ph, dd = B.cc_get_history(h)
        assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= TOL, g
        assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"]), (g, k, r["nclusters"])
        assert np.allclose(ph, r["phi"], rtol=1e-4) and np.allclose(dd, r["d"], rtol=5e-4), g
    B.cc_destroy(h)


def test_dense_mode_rejects_bad_weights(B, torch_):
    torch = torch_
    n, p = 6, 4
    X = torch.randn(n, p, device="cuda:0")
    W = torch.ones(n, n, device="cuda:0")
    W[1, 2] = 2.0
    with pytest.raises(B.CCError) as e:
        B.cc_create(n, p, X, None, None, None, W, B.cc_default_params(dense=1))
    assert e.value.code == B.CC_EGRAPH
    W = torch.ones(n, n, device="cuda:0")
    W[1, 2] = W[2, 1] = -0.5
    with pytest.raises(B.CCError) as e:
        B.cc_create(n, p, X, None, None, None, W, B.cc_default_params(dense=1))
    assert e.value.code == B.CC_EGRAPH


def test_dense_mode_zero_weights_are_unpenalised_pairs(B, torch_, oracle):
    """Dense mode keeps the complete graph as the constraint set; a zero entry of W is a pair of E with no penalty
    (threshold 0, v = b).  cc_dense_weights at a large phi produces such entries; the iteration with them must be
    the oracle's iteration on the complete pair list with those zero weights."""
    torch = torch_
    wl = synth.make("dense_weight", n=90, p=24, n_clusters=3)
    X64 = wl.X.astype(np.float64)
    n = wl.n
    ei, ej, w, d2 = oracle.complete_graph(X64, None, 3.0)
    w32 = w.astype(np.float32)
    assert 100 < int((w32 == 0).sum()) < len(ei) - 100              # a real mix
    dev = torch.device("cuda:0")
    X = torch.from_numpy(wl.X).to(dev)
    W = B.cc_dense_weights(n, wl.p, X, None, 3.0)
    Wref = np.zeros((n, n), np.float32); Wref[ei, ej] = w32; Wref = Wref + Wref.T
    assert np.array_equal(W.cpu().numpy() == 0, Wref == 0)
    W = torch.from_numpy(Wref).to(dev)
    rp, cl, wc = oracle.to_csr(n, ei, ej, w32.astype(np.float64))
    prob = {"X64": X64, "mask": None, "ei": ei, "ej": ej, "w64": w32.astype(np.float64), "n": n, "p": wl.p}
    gammas = [3.0, 30.0, 300.0]
    ref = H.oracle_path(oracle, prob, gammas, 60, proj_method=1)
    h = B.cc_create(n, wl.p, X, None, None, None, W, B.cc_default_params(dense=1))
    U = torch.empty(n, wl.p, device=dev)
    lab = torch.empty(n, dtype=torch.int32, device=dev)
    for g, r in zip(gammas, ref):
        B.cc_solve(h, g, 0.0, 60)
        B.cc_get_U(h, -1, U)
        _, k = B.cc_clusters(h, -1, lab)
        assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= TOL, g
        assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"]), (g, k, r["nclusters"])
    B.cc_destroy(h)


def test_two_points_closed_form_and_single_point(B, torch_):
    """The n = 2 problem has the exact solution (north_star; pin P2): fused at the mean iff ||x1-x2|| <= 2 gamma w,
    else each point moves gamma w along the unit difference -- checked on the GPU path directly, no oracle involved.
    n = 1 (no pairs) must return U = X."""
    torch = torch_
    dev = torch.device("cuda:0")
    x = np.array([[0.0, 0.0, 1.0], [3.0, 4.0, 1.0]], np.float32)
    delta, w = 5.0, 0.7
    rowptr = torch.tensor([0, 1, 2], dtype=torch.int64, device=dev)
    col = torch.tensor([1, 0], dtype=torch.int32, device=dev)
    wv = torch.tensor([w, w], dtype=torch.float32, device=dev)
    prm = B.cc_default_params(rho_abs=40.0, kappa=1e-2)
    h = B.cc_create(2, 3, torch.from_numpy(x).to(dev), None, rowptr, col, wv, prm)
    U = torch.empty(2, 3, device=dev)
    lab = torch.empty(2, dtype=torch.int32, device=dev)
    B.cc_solve(h, 1.0, 0.0, 20000)                      # unfused: delta = 5 > 2 gamma w = 1.4
    B.cc_get_U(h, -1, U)
    u = U.cpu().numpy().astype(np.float64)
    e = (x[0] - x[1]).astype(np.float64) / delta
    assert np.abs(u[0] - (x[0] - 1.0 * w * e)).max() < 2e-4 and np.abs(u[1] - (x[1] + 1.0 * w * e)).max() < 2e-4
    assert B.cc_clusters(h, -1, lab)[1] == 2
    B.cc_reset(h)
    B.cc_solve(h, 5.0, 0.0, 20000)                      # fused: delta = 5 <= 2 gamma w = 7
    B.cc_get_U(h, -1, U)
    u = U.cpu().numpy().astype(np.float64)
    assert B.cc_clusters(h, -1, lab)[1] == 1
    assert np.abs((u[0] + u[1]) / 2 - x.mean(axis=0)).max() < 1e-5
    kap = 1e-2                                          # residual gap of the smoothed iteration: 3 kappa delta / (2 + 3 kappa)
    assert abs(np.linalg.norm(u[0] - u[1]) - 3 * kap * delta / (2 + 3 * kap)) < 5e-3
    B.cc_destroy(h)
    h = B.cc_create(1, 3, torch.from_numpy(x[:1].copy()).to(dev), None, torch.zeros(2, dtype=torch.int64, device=dev), None, None, None)
    B.cc_solve(h, 3.0, 0.0, 5)
    U1 = torch.empty(1, 3, device=dev)
    B.cc_get_U(h, -1, U1)
    assert np.array_equal(U1.cpu().numpy(), x[:1])
    B.cc_destroy(h)


def test_cc_path_dense_mode_snapshots(B, torch_, oracle):
    torch = torch_
    wl = synth.make("genotype", n=20, p=1000)
    prob = H.build_problem(oracle, wl)
    n = wl.n
    W = np.zeros((n, n), np.float32)
    W[prob["ei"], prob["ej"]] = prob["w64"].astype(np.float32)
    W = W + W.T
    gammas = [float(g) for g in synth.gamma_grid(4.0, 40.0, 4)]
    ref = H.oracle_path(oracle, prob, gammas, 60, proj_method=1)
    dev = torch.device("cuda:0")
    h = B.cc_create(n, wl.p, torch.from_numpy(wl.X).to(dev), None, None, None, torch.from_numpy(W).to(dev),
                    B.cc_default_params(dense=1))
    its, phis = B.cc_path(h, gammas, 0.0, 60)
    U = torch.empty(n, wl.p)
    lab = torch.empty(n, dtype=torch.int32)
    for gi, r in enumerate(ref):
        B.cc_get_U(h, gi, U)
        assert H.relerr(U.numpy().astype(np.float64), r["U"]) <= TOL
        _, k = B.cc_clusters(h, gi, lab)
        assert k == r["nclusters"] and np.array_equal(lab.numpy(), r["labels"])
    B.cc_destroy(h)


@pytest.mark.parametrize("n,iters", [(1024, 40), (1100, 12), (548, 12)])
def test_dense_tensor_core_path_multi_tile(B, torch_, oracle, n, iters):
    """n = 1024 (8 row tiles, 36 pair tiles, two accumulator chunks in the contraction), sharper weights so the path
    goes 1024 -> 264 -> 1 clusters: the TMA-fed tcgen05 kernels against the oracle at every gamma.  n = 1100: 35 K blocks
    = two full chunks + one of three blocks (both accumulators reused, a drain left for after the loop), ragged row tile;
    n = 548: 18 K blocks, the second chunk too short to be drained inside the loop."""
    torch = torch_
    wl = synth.make("dense_weight", n=n, p=64, n_clusters=8)
    X64 = wl.X.astype(np.float64)
    si, sj = synth.sample_pairs(wl.n, 200000, 0)
    wl.phi_rule, wl.phi = "fixed", 6.0 / float(np.median(oracle.pair_dist2(X64, None, si, sj)))
    prob = H.build_problem(oracle, wl)
    n = wl.n
    assert len(prob["ei"]) == n * (n - 1) // 2
    gammas = [300.0, 1500.0, 6000.0]
    ref = H.oracle_path(oracle, prob, gammas, iters, proj_method=1)
    if n == 1024:
        assert ref[0]["nclusters"] == n and 1 < ref[1]["nclusters"] < n
    dev = torch.device("cuda:0")
    X = torch.from_numpy(wl.X).to(dev)
    W = B.cc_dense_weights(n, wl.p, X, None, float(wl.phi))          # a0 for complete graphs feeds the solver directly
    Wref = np.zeros((n, n)); Wref[prob["ei"], prob["ej"]] = prob["w64"]; Wref = Wref + Wref.T
    assert np.abs(W.cpu().numpy() - Wref).max() <= 2e-5 * Wref.max()
    W = torch.from_numpy(Wref.astype(np.float32)).to(dev)            # identical fp32 weights on both sides
    h = B.cc_create(n, wl.p, X, None, None, None, W, B.cc_default_params(dense=1))
    U = torch.empty(n, wl.p, device=dev)
    lab = torch.empty(n, dtype=torch.int32, device=dev)
    for g, r in zip(gammas, ref):
        B.cc_solve(h, g, 0.0, iters)
        B.cc_get_U(h, -1, U)
        _, k = B.cc_clusters(h, -1, lab)
        ph, dd = B.cc_get_history(h)
        assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= TOL, g
        assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"]), (g, k, r["nclusters"])
        assert np.allclose(ph, r["phi"], rtol=1e-4) and np.allclose(dd, r["d"], rtol=5e-4), g
    B.cc_destroy(h)


def test_full_size_genotype_elementwise(B, torch_, oracle):
    """configs[2] at full size (52 x 200,000, complete graph, the fused kd_small kernel, 296 CTAs as in bench.py):
    every element of U against the oracle."""
    torch = torch_
    wl = synth.make("genotype")
    prob = H.build_problem(oracle, wl)
    n = wl.n
    W = np.zeros((n, n), np.float32)
    W[prob["ei"], prob["ej"]] = prob["w64"].astype(np.float32)
    W = W + W.T
    gammas = [10.0, 30.0]
    ref = H.oracle_path(oracle, prob, gammas, 8, proj_method=1)
    dev = torch.device("cuda:0")
    h = B.cc_create(n, wl.p, torch.from_numpy(wl.X).to(dev), None, None, None, torch.from_numpy(W).to(dev),
                    B.cc_default_params(dense=1))
    U = torch.empty(n, wl.p, device=dev)
    lab = torch.empty(n, dtype=torch.int32, device=dev)
    for g, r in zip(gammas, ref):
        B.cc_solve(h, g, 0.0, 8)
        B.cc_get_U(h, -1, U)
        _, k = B.cc_clusters(h, -1, lab)
        ph, dd = B.cc_get_history(h)
        diff = U.cpu().numpy().astype(np.float64) - r["U"]
        assert np.linalg.norm(diff) / np.linalg.norm(r["U"]) <= TOL, g
        assert np.abs(diff).max() <= 1e-5, g                      # element-wise (allele frequencies are in [0, 1])
        assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"])
        assert np.allclose(ph, r["phi"], rtol=1e-4) and np.allclose(dd, r["d"], rtol=5e-4)
    B.cc_destroy(h)


def test_full_size_expression_elementwise(B, torch_, oracle):
    """configs[1] at full size (100 x 5000, 10 % missing, 10-NN, the precomputed-inverse projection)."""
    wl = synth.make("expression")
    prob = H.build_problem(oracle, wl)
    gammas = [0.5, 5.0, 50.0]
    ref = H.oracle_path(oracle, prob, gammas, 60)
    _run_path(B, torch_, prob, gammas, 60, ref)


def test_full_size_dense_weight_properties(B, torch_):
    """configs[4] at full size (8192 x 256; the oracle's explicit V would be 68 GB), in the launch configuration bench.py
    times: the properties that hold at any size -- Phi non-increasing, d > 0, the column sums of U
    conserved when nothing is missing (pin P6) -- and determinism (two runs bit-identical).  The same kernels are
    compared element-wise with the oracle at p = 256, n = 2048 and at n = 8192, p = 8 below."""
    torch = torch_
    wl = synth.make("dense_weight")
    dev = torch.device("cuda:0")
    X = torch.from_numpy(wl.X).to(dev)
    n, p = wl.n, wl.p
    si, sj = synth.sample_pairs(n, 200000, 0)
    d = X[torch.from_numpy(si).to(dev)] - X[torch.from_numpy(sj).to(dev)]
    phi = 1.0 / float((d * d).sum(1).median())
    W = B.cc_dense_weights(n, p, X, None, phi)
    outs = []
    for rep in range(2):
        h = B.cc_create(n, p, X, None, None, None, W, B.cc_default_params(dense=1))
        for g in (5.0, 20.0):
            it, phi_v, _ = B.cc_solve(h, g, 0.0, 6)
            ph, dd = B.cc_get_history(h)
            assert it == 6 and np.all(np.diff(ph) <= 1e-6 * np.abs(ph[:-1])) and np.all(dd > 0)
        U = torch.empty(n, p, device=dev)
        B.cc_get_U(h, -1, U)
        rel = (U.double().sum(0) - X.double().sum(0)).abs().max().item() / X.double().abs().sum(0).max().item()
        assert rel <= 1e-6, rel
        outs.append(U.clone())
        B.cc_destroy(h)
    assert torch.equal(outs[0], outs[1])


def test_dense_weight_p256_against_oracle(B, torch_, oracle):
    """configs[4]'s generator at its real width p = 256 (16 K steps per tensor-core tile pass) and n = 2048 (16 row
    tiles, 136 pair tiles): the oracle's explicit V still fits (2.1 M pairs x 256 x 8 B = 4.3 GB).  Element-wise
    against the oracle along a short path; kappa = 0.1 (a parameter of the iteration, the same on both sides) lets
    the short run reach fusion, so that the labels are compared on fused pairs too."""
    torch = torch_
    n, p = 2048, 256
    wl = synth.make("dense_weight", n=n, p=p, n_clusters=32)
    prob = H.build_problem(oracle, wl)
    assert len(prob["ei"]) == n * (n - 1) // 2
    gammas = [80.0, 160.0, 320.0]
    ref = H.oracle_path(oracle, prob, gammas, 4, proj_method=1, kappa=0.1)
    dev = torch.device("cuda:0")
    W = np.zeros((n, n), np.float32)
    W[prob["ei"], prob["ej"]] = prob["w64"].astype(np.float32)
    W = W + W.T
    h = B.cc_create(n, p, torch.from_numpy(wl.X).to(dev), None, None, None, torch.from_numpy(W).to(dev),
                    B.cc_default_params(dense=1, kappa=0.1))
    U = torch.empty(n, p, device=dev)
    lab = torch.empty(n, dtype=torch.int32, device=dev)
    ks = []
    for g, r in zip(gammas, ref):
        B.cc_solve(h, g, 0.0, 4)
        B.cc_get_U(h, -1, U)
        _, k = B.cc_clusters(h, -1, lab)
        ph, dd = B.cc_get_history(h)
        assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= TOL, g
        assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"]), (g, k, r["nclusters"])
        assert np.allclose(ph, r["phi"], rtol=1e-4) and np.allclose(dd, r["d"], rtol=5e-4), g
        ks.append(k)
    B.cc_destroy(h)
    print("dense p=256 n=2048: clusters along the path", ks)
    assert ks[-1] < n


def test_dense_n8192_against_oracle_small_p(B, torch_, oracle):
    """The full number of points of configs[4] (8192, 33.5 M pairs) with p = 8 so that the oracle's explicit V fits:
    the tensor-core kernels against the oracle."""
    torch = torch_
    n, p = 8192, 8
    wl = synth.make("dense_weight", n=n, p=p, n_clusters=32)
    prob = H.build_problem(oracle, wl)
    assert len(prob["ei"]) == n * (n - 1) // 2
    gammas = [0.5, 2.0]
    ref = H.oracle_path(oracle, prob, gammas, 6, proj_method=1)
    dev = torch.device("cuda:0")
    W = np.zeros((n, n), np.float32)
    W[prob["ei"], prob["ej"]] = prob["w64"].astype(np.float32)
    W = W + W.T
    Wd, X = torch.from_numpy(W).to(dev), torch.from_numpy(wl.X).to(dev)
    h = B.cc_create(n, p, X, None, None, None, Wd, B.cc_default_params(dense=1))
    U = torch.empty(n, p, device=dev)
    lab = torch.empty(n, dtype=torch.int32, device=dev)
    for g, r in zip(gammas, ref):
        B.cc_solve(h, g, 0.0, 6)
        B.cc_get_U(h, -1, U)
        _, k = B.cc_clusters(h, -1, lab)
        ph, dd = B.cc_get_history(h)
        assert H.relerr(U.cpu().numpy().astype(np.float64), r["U"]) <= 1e-5, g
        assert k == r["nclusters"] and np.array_equal(lab.cpu().numpy(), r["labels"])
        assert np.allclose(ph, r["phi"], rtol=1e-5) and np.allclose(dd, r["d"], rtol=1e-4), g
    B.cc_destroy(h)


def test_full_size_large_sparse_elementwise(B, torch_, oracle):
    """configs[3] at full size (100,000 x 64, 856,602 pairs), in the launch configuration bench.py times.
    (1) The graph from cc_knn_weights IS the oracle's brute-force graph: rowptr and col identical (index output is
    held to identity: the fp32 tile pass only shortlists, the k nearest are decided in fp64 on the fp32 inputs).
    (2) Every element of U after 2 x 4 iterations of the contract iteration (kappa = 1e-2) from the cold start.
    (3) A run in which pairs really fuse, so that identical labels mean something at this size: kappa = 0.1
    (a parameter of the iteration, S2; the same on both sides) makes the first thresholds gamma w kappa comparable
    to the neighbour distances, 3 gammas x 6 iterations, thousands of fused pairs at the last gamma."""
    torch = torch_
    wl = synth.make("large_sparse")
    prob = H.build_problem(oracle, wl)
    dev = torch.device("cuda:0")
    X = torch.from_numpy(wl.X).to(dev)
    rowptr, col, w = B.cc_knn_weights(wl.n, wl.p, X, None, wl.k, prob["phi"])
    assert np.array_equal(rowptr.cpu().numpy(), prob["rowptr"])
    assert np.array_equal(col.cpu().numpy(), prob["col"])
    assert np.abs(w.cpu().numpy() - prob["wcsr32"]).max() <= 1e-6 * prob["wcsr32"].max()
    gammas = [5.0, 80.0]
    ref = H.oracle_path(oracle, prob, gammas, 4, proj_method=1)
    out = _run_path(B, torch, prob, gammas, 4, ref)
    print("full-size large_sparse: relerr, clusters =", out)
    gammas = [40.0, 70.0, 110.0]
    ref = H.oracle_path(oracle, prob, gammas, 6, proj_method=1, kappa=0.1)
    out = _run_path(B, torch, prob, gammas, 6, ref, kappa=0.1)
    print("full-size large_sparse, kappa = 0.1: relerr, clusters =", out)
    assert out[-1][1] < wl.n - 2000          # the comparison of labels is not vacuous


# ----------------------------------------------------------------------------- f1: kappa continuation (S26)
def _continuation_case(B, torch, oracle, prob, h, g, k0, factor, stage_it, last_it, proj_method=0):
    X, m = prob["X64"], prob["mask"]
    U0, V0 = oracle.cold_start(X, m, prob["ei"], prob["ej"])
    ref = oracle.mm_continuation(X, m, prob["ei"], prob["ej"], prob["w64"], g, U0, V0, k0, factor, stage_it, last_it,
                                 tol=0.0, proj_method=proj_method)
    its, phi, rc = B.cc_solve_continuation(h, g, k0, factor, stage_it, 0.0, last_it)
    assert rc == B.CC_OK and its == ref["stage_iters"]
    n, p = prob["n"], prob["p"]
    U = torch.empty(n, p)
    B.cc_get_U(h, -1, U)
    lab = torch.empty(n, dtype=torch.int32)
    _, k = B.cc_clusters(h, -1, lab)
    rl, rk = oracle.labels(ref["V"], prob["ei"], prob["ej"], n)
    assert H.relerr(U.numpy().astype(np.float64), ref["U"]) <= TOL
    assert k == rk and np.array_equal(lab.numpy(), rl)
    assert abs(phi - ref["phi"][-1]) <= 1e-4 * abs(phi)
    st = B.cc_get_stats(h)
    assert abs(st["rho"] - ref["rho"]) <= 1e-6 * ref["rho"]
    assert abs(st["eps"] - (ref["kappas"][-1] * ref["rho"]) ** 2) <= 1e-6 * st["eps"]     # the last stage is the contract's
    return ref


def test_kappa_continuation_matches_oracle_sparse(B, torch_, oracle):
    """Stages kappa = 1, 0.1, 0.01 with fixed lengths, cold start, on the k-NN path: element-wise against the oracle's
    staged iteration (tiny, masked expression-like, 3,000 large-sparse points)."""
    torch = torch_
    for wl, g in ((synth.make("tiny"), 100.0), (synth.make("expression", n=40, p=300), 2.0),
                  (synth.make("large_sparse", n=3000), 20.0)):
        prob = H.build_problem(oracle, wl)
        h = H.gpu_create(B, torch, prob)
        _continuation_case(B, torch, oracle, prob, h, g, 1.0, 0.1, 25, 40)
        B.cc_destroy(h)


def test_kappa_continuation_matches_oracle_dense(B, torch_, oracle):
    torch = torch_
    wl = synth.make("dense_weight", n=300, p=40, n_clusters=6)
    X64 = wl.X.astype(np.float64)
    si, sj = synth.sample_pairs(wl.n, 200000, 0)
    wl.phi_rule, wl.phi = "fixed", 6.0 / float(np.median(oracle.pair_dist2(X64, None, si, sj)))
    prob = H.build_problem(oracle, wl)
    n = wl.n
    W = np.zeros((n, n), np.float32)
    W[prob["ei"], prob["ej"]] = prob["w64"].astype(np.float32)
    W = W + W.T
    dev = torch.device("cuda:0")
    h = B.cc_create(n, wl.p, torch.from_numpy(wl.X).to(dev), None, None, None, torch.from_numpy(W).to(dev),
                    B.cc_default_params(dense=1))
    _continuation_case(B, torch, oracle, prob, h, 300.0, 0.5, 0.2, 20, 40, proj_method=1)
    B.cc_destroy(h)


def test_kappa_continuation_stop_rule_and_arguments(B, torch_, oracle):
    """With tol > 0 every stage stops by S3 near the oracle's count, the staged run needs fewer iterations than the
    plain one for the same rule, and both end at the same U to the accuracy the rule gives."""
    torch = torch_
    wl = synth.make("tiny")
    prob = H.build_problem(oracle, wl)
    X, m = prob["X64"], prob["mask"]
    U0, V0 = oracle.cold_start(X, m, prob["ei"], prob["ej"])
    g, tol = 100.0, 1e-7
    ref = oracle.mm_continuation(X, m, prob["ei"], prob["ej"], prob["w64"], g, U0, V0, 1.0, 0.1, 400, 20000, tol=tol)
    h = H.gpu_create(B, torch, prob)
    its, phi, rc = B.cc_solve_continuation(h, g, 1.0, 0.1, 400, tol, 20000)
    assert len(its) == 3
    for a, b in zip(its, ref["stage_iters"]):
        assert abs(a - b) <= max(3, b // 20), (its, ref["stage_iters"])
    Uc = torch.empty(wl.n, wl.p)
    B.cc_get_U(h, -1, Uc)
    B.cc_reset(h)
    it_plain, _, _ = B.cc_solve(h, g, tol, 20000)
    Up = torch.empty(wl.n, wl.p)
    B.cc_get_U(h, -1, Up)
    assert sum(its) < it_plain, (its, it_plain)
    assert H.relerr(Uc.numpy().astype(np.float64), Up.numpy().astype(np.float64)) <= 2e-2
    # kappa_start at or below the contract kappa: one stage, bit-identical to cc_solve
    B.cc_reset(h)
    its1, _, _ = B.cc_solve_continuation(h, g, 1e-2, 0.5, 7, 0.0, 30)
    U1 = torch.empty(wl.n, wl.p)
    B.cc_get_U(h, -1, U1)
    B.cc_reset(h)
    B.cc_solve(h, g, 0.0, 30)
    B.cc_get_U(h, -1, Up)
    assert its1 == [30] and np.array_equal(U1.numpy(), Up.numpy())
    for bad in ((0.0, 0.5, 5), (1.0, 1.0, 5), (1.0, 0.0, 5), (1.0, 0.5, 0)):
        with pytest.raises(B.CCError) as e:
            B.cc_solve_continuation(h, g, bad[0], bad[1], bad[2], 0.0, 10)
        assert e.value.code == B.CC_EINVAL
    B.cc_destroy(h)
    h = H.gpu_create(B, torch, prob, eps_abs=1e-3)
    with pytest.raises(B.CCError) as e:
        B.cc_solve_continuation(h, g, 1.0, 0.5, 5, 0.0, 10)
    assert e.value.code == B.CC_ESTATE
    B.cc_destroy(h)


def test_path_continuation_matches_oracle(B, torch_, oracle):
    """cc_path_continuation: staged solves at every gamma, warm-started along the path, snapshots as cc_path."""
    torch = torch_
    wl = synth.make("tiny")
    prob = H.build_problem(oracle, wl)
    X, m = prob["X64"], prob["mask"]
    gammas = [float(g) for g in synth.gamma_grid(1.0, 1e3, 5)]
    U, V = oracle.cold_start(X, m, prob["ei"], prob["ej"])
    h = H.gpu_create(B, torch, prob)
    its, phis = B.cc_path_continuation(h, gammas, 0.5, 0.2, 15, 0.0, 30)
    Ug = torch.empty(wl.n, wl.p)
    lab = torch.empty(wl.n, dtype=torch.int32)
    for gi, g in enumerate(gammas):
        r = oracle.mm_continuation(X, m, prob["ei"], prob["ej"], prob["w64"], g, U, V, 0.5, 0.2, 15, 30)
        U, V = r["U"], r["V"]
        assert its[gi] == sum(r["stage_iters"]) == 15 * 3 + 30
        B.cc_get_U(h, gi, Ug)
        assert H.relerr(Ug.numpy().astype(np.float64), U) <= TOL
        _, k = B.cc_clusters(h, gi, lab)
        rl, rk = oracle.labels(V, prob["ei"], prob["ej"], wl.n)
        assert k == rk and np.array_equal(lab.numpy(), rl)
        assert abs(phis[gi] - r["phi"][-1]) <= 1e-5 * abs(phis[gi])
    B.cc_destroy(h)
