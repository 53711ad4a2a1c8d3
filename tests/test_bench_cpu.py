"""Host logic of bench.py that needs no GPU: the roofline byte counts must be SURVEY.md 8(d)'s formulas."""
import importlib.util
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_sweep_bytes_are_survey_8d_formulas_at_the_bench_graph():
    """large_sparse as benched: n = 100,000, p = 64, nnz = 1,713,204 directed entries (|E| = 856,602).  SURVEY 8(d):
    a1 nnz(4p+12) + 3*4np, a2 nnz(4p+4) + 7*4np, a3 |E|(8p+12) + 2*4np, a5+a6 4*4np + np -- the numbers VERDICT.md recomputed
    (535.9, 624.6, 500.1, 108.8 MB)."""
    b = _bench()
    n, p, nnz = 100_000, 64, 1_713_204
    sw = b.sweep_bytes(n, p, nnz, False)
    npb, E = 4 * n * p, nnz // 2
    want = {"a1_rhs": nnz * (4 * p + 12) + 3 * npb, "a2_sweep": nnz * (4 * p + 4) + 7 * npb,
            "a3_norms": E * (8 * p + 12) + 2 * npb, "a5_update": 4 * npb + n * p}
    assert {k: v[0] for k, v in sw.items()} == want
    mb = {k: round(v[0] / 1e6, 1) for k, v in sw.items()}
    assert mb == {"a1_rhs": 535.9, "a2_sweep": 624.6, "a3_norms": 500.1, "a5_update": 108.8}
    assert sw["a2_sweep"][1] == ("k_cg_spmv", "k_cg_update")          # the inner sweep is charged to both kernels together


def test_dense_sweep_bytes_and_flops():
    """Dense path: genotype-like = 7 node arrays per iteration; dense-weight = W (n x n) once + node arrays;
    useful flops of the contraction 2 n^2 p and of the pair norms 6p per unordered pair (FMA = 2)."""
    b = _bench()
    n, p = 52, 200_000
    sw = b.sweep_bytes(n, p, n * (n - 1), False, dense=True)
    assert sw["a9_small"][0] == 7 * 4 * n * p == 291_200_000
    n, p = 8192, 256
    assert b.alg_flops("kd_proj", n, p, False) == 2.0 * n * n * p
    assert b.alg_flops("kd_pairs", n, p, False) == 2.0 * (n * (n - 1) / 2) * p
    tot = b.alg_flops("kd_proj", n, p, False) + b.alg_flops("kd_pairs", n, p, False)
    # 6p flops per unordered pair: 51.5 GFLOP per iteration (the bench line weights each kernel by the launches its device
    # timer saw -- the first launch after a timer reset is not timed -- hence the 49.8 GFLOP in profiles/r2_summary.md)
    assert tot == (3.0 * n * n - n) * p and abs(tot - 6.0 * p * (n * (n - 1) / 2)) < 0.001 * tot
