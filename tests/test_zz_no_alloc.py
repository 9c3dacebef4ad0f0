"""GPU test of sg_get_state_hash_noalloc (include/sg.h): the state hash for callers that must not allocate.

Who needs it: a host program that has given all device memory to its own pool allocator (a raw cudaMalloc from a library
then fails or eats into that pool), a hook that fires inside a running simulation loop (cudaMalloc / cudaFree stall
every stream of the device), or a caller handed a context on somebody else's workspace with no allocator of its own.
For them the per-system hashes are staged in one fixed 512 KiB device array inside the library image instead of a
buffer sized with the pool, so the call makes no allocation at all; the price is a size limit
(sg.NOALLOC_MAX_SYSTEMS systems) and one array shared by every call on a GPU.

What is checked, always against the ordinary sg_get_state_hash on the same context and bit for bit (hashes are
integers, so the tolerance of the other state comparisons in this suite applies: none):
  - two calls in a row with the state changed in between: the second must show the NEW state although the array still
    held the first call's hashes when it started;
  - a small Gaussian context right after a larger +-J one: what the larger call left further up the array must not
    leak into the smaller result;
  - the L = 32 path, whose launches hand the state from one buffer to the other and defer exchanges, gives the same
    hashes through both calls;
  - a pool above the limit is refused with a message that names the limit, and the context stays usable.

This file is named test_zz_* so that pytest collects it last: under `pytest -x` a failure here cannot hide a failure in
any other test.  Every test builds its own contexts, so the file passes alone in a fresh process (where the very first
call on the device also does the one-time address look-up) as well as after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _sg():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1403_4560_b200 import sg
    return sg


def _ladder(n):
    from paper_1403_4560_b200 import workloads as W
    return W.ladder(0.5, 2.0, n)


def test_two_calls_in_a_row_follow_the_state():
    sg = _sg()
    sim = sg.Simulation(8, 0.1, 96, 4, _ladder(6), sg.PMJ, seed=11)
    try:
        sim.sg_run(5, 1, 0)
        want1 = sim.sg_get_state_hash()
        got1 = sim.sg_get_state_hash_noalloc()
        assert got1.dtype == np.uint64 and got1.shape == want1.shape == (3, 4, 6)
        assert np.array_equal(got1, want1)
        sim.sg_run(3, 1, 0)                      # the array still holds got1 when the next call starts
        got2 = sim.sg_get_state_hash_noalloc()
        want2 = sim.sg_get_state_hash()
        assert np.array_equal(got2, want2)
        assert not np.array_equal(got2, got1), "the state moved, so must the hashes"
        # and once more without a change: same answer, no side effect on the state
        assert np.array_equal(sim.sg_get_state_hash_noalloc(), want2)
        assert np.array_equal(sim.sg_get_state_hash(), want2)
    finally:
        sim.close()


def test_smaller_pool_after_a_larger_one_and_gaussian_bytes():
    sg = _sg()
    big = sg.Simulation(4, 0.2, 2048, 4, _ladder(16), sg.PMJ, seed=3)        # 64 words x 4 x 16 = 4096 systems
    small = sg.Simulation(4, 0.3, 5, 2, _ladder(3), sg.GAUSS, seed=4)        # 5 x 2 x 3 = 30 systems of byte spins
    try:
        big.sg_run(4, 2, 0)
        small.sg_run(4, 2, 0)
        for _ in range(2):
            assert np.array_equal(big.sg_get_state_hash_noalloc(), big.sg_get_state_hash())
            got = small.sg_get_state_hash_noalloc()
            assert got.shape == (5, 2, 3)
            assert np.array_equal(got, small.sg_get_state_hash())
            small.sg_sweep(1)
            big.sg_sweep(1)
    finally:
        big.close()
        small.close()


def test_L32_resident_path_with_deferred_exchanges():
    sg = _sg()
    a = sg.Simulation(32, 0.1, 32, 2, _ladder(4), sg.PMJ, seed=9)
    b = sg.Simulation(32, 0.1, 32, 2, _ladder(4), sg.PMJ, seed=9)
    try:
        a.sg_run(4, 4, 0)                        # the exchange after sweep 4 is applied by the time sg_run returns
        b.sg_run(4, 4, 0)
        got = a.sg_get_state_hash_noalloc()      # first thing to look at `a` after the run
        want = b.sg_get_state_hash()
        assert np.array_equal(got, want)
        a.sg_run(4, 4, 0)
        b.sg_run(4, 4, 0)
        assert np.array_equal(a.sg_get_state_hash_noalloc(), b.sg_get_state_hash())
    finally:
        a.close()
        b.close()


def test_pool_above_the_limit_is_refused():
    sg = _sg()
    n_words = sg.NOALLOC_MAX_SYSTEMS // (4 * 64) + 1                         # 257 words x 4 x 64 = 65792 > 65536
    sim = sg.Simulation(4, 0.1, 32 * n_words, 4, _ladder(64), sg.PMJ, seed=5)
    try:
        with pytest.raises(sg.SgError) as e:
            sim.sg_get_state_hash_noalloc()
        assert e.value.code == sg.EINVAL and str(sg.NOALLOC_MAX_SYSTEMS) in str(e.value)
        h = sim.sg_get_state_hash()                                          # the ordinary call has no such limit
        assert h.shape == (n_words, 4, 64)
    finally:
        sim.close()
    # exactly at the limit it works
    n_words -= 1
    sim = sg.Simulation(4, 0.1, 32 * n_words, 4, _ladder(64), sg.PMJ, seed=5)
    try:
        sim.sg_sweep(1)
        assert np.array_equal(sim.sg_get_state_hash_noalloc(), sim.sg_get_state_hash())
    finally:
        sim.close()
