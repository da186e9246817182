"""gamma_sort_pairs_noalloc against gamma_sort_pairs (and the sort oracle).

The no-allocation entry point exists for callers that cannot let the library call cudaMalloc: code running while a
stream is being captured in the global mode, code with a latency budget, code in a process where one pool owns the
device memory.  Its scratch is a fixed array inside libgamma_b200.so that every call shares and that is never
cleared, so the interesting failure is the SECOND call: something left behind by the first one (tile histograms of a
longer input, a stale element counter, the other half of the ping-pong buffers) leaking into it.  Each case below
therefore makes two calls in a row, of different lengths and different bit ranges, and compares both with what the
allocating path returns on the same input -- bit for bit, the bar every sort test here uses (integer work, stable
sort: one right answer).

The file sorts last in the collection on purpose: `pytest -x` stops at the first failure, and a failure here should
not hide the parity tests.  It does not depend on what ran before it: it passes alone in a fresh process (then its
first call is also the first CUDA work of the library, address look-up included) and after the whole suite.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_1012_1900_b200 import binding

pytestmark = pytest.mark.gpu

LIMIT = binding.SORT_NOALLOC_MAX_PAIRS


def _pairs(n, seed, ties):
    rng = np.random.default_rng([n, seed])
    if ties:
        keys = rng.integers(0, 2 ** 32, size=n, dtype=np.uint64).astype(np.uint32)
        keys[: n // 2] &= 0x00FF00FF                       # long runs of equal digits: stability is visible in vals
    else:
        keys = np.abs(rng.normal(0, 3, size=n)).astype(np.float32).view(np.uint32)   # the gamma keys: fp32 bit patterns
    vals = rng.permutation(n).astype(np.uint32)
    return keys, vals


def _both_paths(keys, vals, bits):
    out = []
    for fn in (binding.gamma_sort_pairs_noalloc, binding.gamma_sort_pairs):
        k = torch.from_numpy(keys.view(np.int32).copy()).cuda()
        v = torch.from_numpy(vals.view(np.int32).copy()).cuda()
        fn(k, v, bits[0], bits[1])
        out.append((k, v))
    torch.cuda.synchronize()
    return [(k.cpu().numpy().view(np.uint32), v.cpu().numpy().view(np.uint32)) for k, v in out]


@pytest.mark.parametrize("first,second", [
    # (n, bits, ties) of the first call, then of the second; the second is the one a dirty scratch would break
    ((LIMIT, (0, 32), True), (100_003, (0, 32), False)),       # the limit itself, then a shorter ragged list
    ((300_001, (8, 32), False), (LIMIT - 1, (16, 32), True)),  # odd number of passes (result comes back by copy), then even
    ((4097, (24, 32), True), (4096, (0, 8), True)),            # two tiles then exactly one; one pass each
    ((1, (0, 32), False), (31, (8, 16), True)),                # less than a warp
])
def test_noalloc_sort_equals_allocating_sort_on_two_calls_in_a_row(first, second):
    from oracle import aux_oracle
    for n, bits, ties in (first, second):
        keys, vals = _pairs(n, bits[0], ties)
        (k_na, v_na), (k_ws, v_ws) = _both_paths(keys, vals, bits)
        assert np.array_equal(k_na, k_ws) and np.array_equal(v_na, v_ws)
        ek, ev = aux_oracle.sort_pairs(keys, vals, bits[0], bits[1])       # and both are the definition's answer
        assert np.array_equal(k_na, ek) and np.array_equal(v_na, ev)


def test_noalloc_sort_same_input_twice_gives_the_same_answer():
    keys, vals = _pairs(77_777, 5, True)
    a = _both_paths(keys, vals, (0, 32))[0]
    b = _both_paths(keys, vals, (0, 32))[0]
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_noalloc_sort_rejects_more_than_the_limit_and_leaves_the_data_alone():
    n = LIMIT + 1
    k = torch.arange(n, 0, -1, dtype=torch.int32, device="cuda")
    v = torch.arange(n, dtype=torch.int32, device="cuda")
    with pytest.raises(binding.GammaError) as err:
        binding.gamma_sort_pairs_noalloc(k, v)
    assert "GAMMA_SORT_NOALLOC_MAX_PAIRS" in str(err.value) and str(LIMIT) in str(err.value)
    torch.cuda.synchronize()
    assert int(k[0]) == n and int(k[-1]) == 1 and int(v[-1]) == n - 1     # nothing was launched
    lib = binding.load_library()
    assert lib.gamma_sort_pairs_noalloc(None, None, 0, 0, 32, None) == 0          # empty input: no-op
    assert lib.gamma_sort_pairs_noalloc(ctypes.c_void_p(k.data_ptr()), None, 8, 0, 32, None) == 1
    assert lib.gamma_sort_pairs_noalloc(ctypes.c_void_p(k.data_ptr()), ctypes.c_void_p(v.data_ptr()), 8, 4, 32, None) == 1


def test_noalloc_sort_does_not_touch_the_workspaces():
    """The point of the entry point: the library's own device allocations do not change across its calls."""
    binding.gamma_release()
    before = binding.gamma_workspace_bytes()
    free0, _ = torch.cuda.mem_get_info()
    keys, vals = _pairs(200_000, 9, False)
    k = torch.from_numpy(keys.view(np.int32).copy()).cuda()
    v = torch.from_numpy(vals.view(np.int32).copy()).cuda()
    binding.gamma_sort_pairs_noalloc(k, v)             # first use may load the kernels' code: not what is measured
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        binding.gamma_sort_pairs_noalloc(k, v)
    torch.cuda.synchronize()
    free2, _ = torch.cuda.mem_get_info()
    assert binding.gamma_workspace_bytes() == before
    assert free2 == free1, (free0, free1, free2)       # no device memory taken after the inputs were in place
    assert bool((k[1:].view(torch.int32) >= k[:-1].view(torch.int32)).all())      # non-negative fp32 patterns: int order
