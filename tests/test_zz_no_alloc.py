"""cc_dense_weights_noalloc (include/cc_b200.h): the all-pairs weight build for callers that must not allocate.
Checked against the existing path cc_dense_weights on the same inputs, two calls in a row (the calls share one static
scratch array that keeps the previous call's contents).  Kept in a file of its own that pytest collects last."""
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


def test_dense_weights_noalloc_matches_the_allocating_path_on_consecutive_calls(B):
    import torch
    cases = [
        # (workload, sizes, phi): few pair tiles and many columns -> column slices -> the scratch array is used
        ("genotype", dict(n=52, p=40000), 0.002),            # 1 tile x ~296 slices: 0.8 M floats of scratch
        ("expression", dict(n=30, p=5000), 0.0002),          # masked: sums and counts, both in the scratch; fewer slices,
                                                             # so most of the array still holds the previous call's numbers
        ("genotype", dict(n=52, p=3001), 0.01),              # ragged p, again over stale contents
        ("dense_weight", dict(n=1300, p=24, n_clusters=5), 0.01),   # enough tiles to fill the GPU: no scratch at all
    ]
    for name, kw, phi in cases:
        wl = synth.make(name, **kw)
        X, M = _dev(torch, wl.X), _dev(torch, wl.mask)
        ref = B.cc_dense_weights(wl.n, wl.p, X, M, phi).cpu().numpy()
        W = torch.full((wl.n, wl.n), -1.0, dtype=torch.float32, device="cuda:0")
        for call in range(2):                                # two calls in a row on every case
            W.fill_(-1.0)
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            B.cc_dense_weights_noalloc(wl.n, wl.p, X, M, phi, W)
            free1 = torch.cuda.mem_get_info()[0]
            got = W.cpu().numpy()
            # the tolerance of the a0 tests (tests/test_gpu_api.py::test_dense_weights_match_oracle) ...
            assert np.abs(got - ref).max() <= 2e-5 * ref.max(), (name, call)
            # ... and in fact the same partial sums added in the same order: identical
            assert np.array_equal(got, ref), (name, call)
            assert np.array_equal(got, got.T) and np.all(np.diag(got) == 0), (name, call)
            if call == 1:
                assert free1 >= free0, (name, free0, free1)   # no device memory was taken by the call


def test_dense_weights_noalloc_rejects_what_does_not_fit(B):
    import torch
    wl = synth.make("genotype", n=64, p=200000)
    X = _dev(torch, wl.X)
    W = torch.empty(wl.n, wl.n, dtype=torch.float32, device="cuda:0")
    B.cc_dense_weights_noalloc(wl.n, wl.p, X, None, 0.001, W)           # 291 slices x 64 x 64 = 1.19 M floats: fits
    assert torch.equal(W, B.cc_dense_weights(wl.n, wl.p, X, None, 0.001))
    M = torch.ones(wl.n, wl.p, dtype=torch.uint8, device="cuda:0")       # with a mask: sums and counts, 2.38 M > 2 Mi floats
    M[0, 0] = 0
    with pytest.raises(B.CCError) as e:
        B.cc_dense_weights_noalloc(wl.n, wl.p, X, M, 0.001, W)
    assert e.value.code == B.CC_EINVAL and "scratch" in str(e.value)
    Ms = M[:52].contiguous()                                             # configs[2]'s 52 rows fit even with a mask (1.57 M)
    Ws = torch.empty(52, 52, dtype=torch.float32, device="cuda:0")
    B.cc_dense_weights_noalloc(52, wl.p, X[:52].contiguous(), Ms, 0.001, Ws)
    assert torch.equal(Ws, B.cc_dense_weights(52, wl.p, X[:52].contiguous(), Ms, 0.001))
    with pytest.raises(B.CCError) as e:
        B.cc_dense_weights_noalloc(1, 4, X, None, 0.001, W)
    assert e.value.code == B.CC_EINVAL
