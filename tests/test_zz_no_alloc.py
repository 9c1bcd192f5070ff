"""emx_refill_plan_static (include/emx.h): the refill hook whose scratch is a file-scope device array, for callers
that may not allocate device memory.  Its results must be those of emx_refill_plan (integer work: bit-exact, the
bar of tests/test_gpu_parity.py::test_refill_compaction_order_is_bit_exact), call after call on the shared array.

Collected last on purpose (the file name): the suite runs with pytest -x.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def emx():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2203_09467_b200 import emx as m
    m.lib()
    return m


def _case(n_live, capacity, n_queue, p_dead):
    rng = np.random.default_rng(7 * n_live + n_queue)
    return (rng.random(n_live) >= p_dead).astype(np.uint8), capacity, n_queue


def test_static_scratch_entry_point_matches_the_allocating_one(emx):
    assert emx.refill_plan_static_max() == 65536
    assert emx.lib().emx_refill_plan_static_setup() == 0
    # calls in a row on the one shared array: a large pool first, then smaller ones that would see its leftovers
    # (stale chunk tables, hole lists, alive flags, control block), then the largest size the array holds
    cases = [_case(60001, 65536, 999, 0.7), _case(777, 1024, 50, 0.3), _case(0, 300, 1000, 0.0),
             _case(129, 256, 3, 0.9), _case(5000, 8192, 10 ** 6, 0.02), _case(65536, 65536, 100, 1.0),
             _case(60001, 65536, 999, 0.7)]
    for alive, capacity, n_queue in cases:
        want_src, want_counts = emx.refill_plan(alive, capacity, n_queue)
        for _ in range(2):                                            # twice in a row: same answer both times
            got_src, got_counts = emx.refill_plan(alive, capacity, n_queue, static=True)
            assert got_counts == want_counts
            n_new = want_counts[0]
            assert np.array_equal(got_src[:n_new], want_src[:n_new])
            assert np.array_equal(got_src, want_src)                  # the untouched tail of src too (-1)


def test_static_scratch_entry_point_rejects_what_does_not_fit(emx):
    alive = np.ones(10, dtype=np.uint8)
    with pytest.raises(emx.EmxError) as e:
        emx.refill_plan(alive, 65537, 0, static=True)
    assert "-4" in str(e.value) and "65536" in str(e.value)          # EMX_E_CAPACITY, and the text names the limit
    src, counts = emx.refill_plan(alive, 65536, 0, static=True)       # the limit itself is accepted
    assert counts == (10, 0, 0)
