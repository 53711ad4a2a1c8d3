"""CPU-only checks of the boundary (-m "not gpu"): libcc_b200.so builds with nvcc for sm_100a, loads,
exports every symbol include/cc_b200.h declares, and fails loudly (no CPU fallback) without a GPU."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1409_2065_b200 import build
    return build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "cc_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cc_[a-z_A-Z0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(lib_path):
    names = _declared()
    assert {"cc_create", "cc_solve", "cc_path", "cc_get_U", "cc_clusters", "cc_knn_weights"} <= set(names)
    lib = ctypes.CDLL(lib_path)
    for nm in names:
        assert hasattr(lib, nm), nm
    from paper_1409_2065_b200 import binding
    assert sorted(binding.SYMBOLS) == names


def test_library_is_sm100a_only(lib_path):
    out = subprocess.run(["cuobjdump", "-lelf", lib_path], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_params_struct_layout_matches_header():
    from paper_1409_2065_b200 import binding as B
    prm = B.cc_default_params()
    assert (prm.rho_scale, prm.kappa, prm.proj_tol) == (1.1, 1e-2, 1e-5)
    assert (prm.proj_maxit, prm.min_it, prm.dense, prm.use_graph) == (500, 10, 0, 1)
    assert ctypes.sizeof(B.cc_params) == 5 * 8 + 7 * 4 + 4   # 5 doubles, 7 int32, tail padding to 8


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1409_2065_b200 import binding as B
    X = torch.zeros(2, 2)
    with pytest.raises(B.CCError) as e:
        B.cc_create(2, 2, X, None, torch.zeros(3, dtype=torch.int64), torch.zeros(2, dtype=torch.int32),
                    torch.ones(2), None)
    assert e.value.code == B.CC_ECUDA and "no CPU fallback" in str(e.value)


def test_product_path_never_touches_the_oracle():
    """The package must not import, read or run anything under oracle/ (task rule 3)."""
    pkg = os.path.join(ROOT, "paper_1409_2065_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
                assert "cc_oracle" not in txt and "oracle/" not in txt.replace("the oracle", ""), f


def _rank_main(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms, units = bench.aggregate(dist, torch.device("cpu"), [10.0 + rank, 20.0 - rank], [100.0 * (rank + 1), 7.0])
    q.put((rank, ms, units))
    dist.destroy_process_group()


def test_multi_rank_aggregation_gloo_world2():
    """bench.py at N > 1 runs independent replicas; the only cross-rank step is max(time) / sum(units)."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p_ in procs:
        p_.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p_ in procs:
        p_.join(timeout=60)
    for _, ms, units in res:
        assert ms == [11.0, 20.0] and units == [300.0, 14.0]
