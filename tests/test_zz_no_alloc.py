"""best_rminus1_noalloc (scratch in a static __device__ array, no allocation) against best_rminus1, the existing
path, on two calls in a row.  Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2606_04895_b200 import binding
    binding.lib()
    return binding


def _trace(seed, n, nb, d):
    import torch
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((d, d)) / np.sqrt(d) + np.eye(d)
    x = (rng.standard_normal((n, nb, d)) + 0.7 * rng.standard_normal((1, nb, d))) @ A.T + 5.0
    return torch.from_numpy(x.astype(np.float32)).cuda()


def test_rminus1_noalloc_matches_rminus1_twice_in_a_row(B):
    import torch
    # ragged tails in every kernel, the paper's d = 29 / 27; the second call is SMALLER than the first, so it
    # runs on a scratch array that still holds the first call's (larger) contents
    first, second = _trace(11, 67, 4099, 29), _trace(12, 41, 130, 27)
    want = [B.rminus1(first), B.rminus1(second)]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    got = [B.rminus1_noalloc(first), B.rminus1_noalloc(second)]
    assert free0 - torch.cuda.mem_get_info()[0] < (2 << 20)      # no device allocation (the driver's granule is 2 MiB)
    # same kernels, grids and summation order: the tests of best_rminus1 use rel 1e-8 against the oracle;
    # against the existing path the values are the same bits
    for g, w in zip(got, want):
        assert g == pytest.approx(w, rel=1e-8) and g == w
    # and again in the other order, twice each (the array keeps the last call's contents)
    assert B.rminus1_noalloc(second) == want[1] and B.rminus1_noalloc(second) == want[1]
    assert B.rminus1_noalloc(first) == want[0] and B.rminus1_noalloc(first) == want[0]
    # a non-default stream
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        assert B.rminus1_noalloc(first, stream=s.cuda_stream) == want[0]


def test_rminus1_noalloc_rejects_sizes_beyond_the_static_array(B):
    import torch
    cap = B.rminus1_noalloc_max_doubles()
    assert cap == 1 << 20
    d, n = 32, 10

    def need(nb):                                                 # the header's formula
        return nb * d + d + (min(-(-n * nb // 64), 592) + min(-(-nb // 64), 148)) * d * d + 2

    nb_ok = max(nb for nb in range(8000, 10000) if need(nb) <= cap)   # the largest B that fits at d = 32
    assert need(nb_ok + 1) > cap
    out = C.c_double()
    x = torch.zeros(10, nb_ok + 1, d, device="cuda")
    x.normal_()
    assert B.lib().best_rminus1_noalloc(x.data_ptr(), 10, nb_ok + 1, d, C.byref(out), None) == B.BEST_ERR_ARG
    msg = B.lib().best_last_error().decode()
    assert "static array" in msg and str(cap) in msg
    y = x[:, :nb_ok].contiguous()
    assert B.rminus1_noalloc(y) == B.rminus1(y)                  # exactly at the limit
    # the argument checks of best_rminus1
    z = torch.randn(10, 8, 3, device="cuda")
    for args in ((1, 8, 3), (10, 1, 3), (10, 8, 33)):
        assert B.lib().best_rminus1_noalloc(z.data_ptr(), *args, C.byref(out), None) == B.BEST_ERR_ARG
    assert B.lib().best_rminus1_noalloc(z.cpu().numpy().ctypes.data, 10, 8, 3, C.byref(out), None) == B.BEST_ERR_ARG
