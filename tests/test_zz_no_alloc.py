"""sg_correlation_noalloc (include/sg.h): the correlation counts with the kernel's counters in the library's static device
array -- for callers that cannot call cudaMalloc -- against the existing sg_correlation path.  Integer work: EQUAL.

Kept in a file of its own that pytest collects last (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sg():
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1906_11195_b200 import build as b

    b.build()
    import paper_1906_11195_b200 as sg

    return sg


@pytest.mark.parametrize("model,N,c,W", [(0, 20000, 4.0, 1), (0, 5000, 4.0, 4), (0, 3000, 6.0, 3), (2, 4096, 0.0, 64)])
def test_noalloc_counts_equal_the_existing_path_on_two_calls_in_a_row(sg, model, N, c, W):
    """Two calls in a row on different states (the static array keeps the previous call's counts and must be cleared),
    then a third on an unchanged state; W = 3 goes through the strided count kernel, W = 64 fills the array."""
    from paper_1906_11195_b200 import binding

    assert binding.sg_noalloc_max_words() == 64
    g = sg.Sim(model, N, c, 1.0, 31, W)
    g.snapshot(0)
    g.sweep(2)
    first = g.correlation_noalloc(0)
    assert np.array_equal(first, g.correlation(0))
    assert first.shape == (64 * W,) and first.min() > 0 and first.max() <= N
    g.sweep(3)
    g.snapshot(1)
    second = g.correlation_noalloc(0)
    assert np.array_equal(second, g.correlation(0))
    assert not np.array_equal(second, first)
    assert np.array_equal(g.correlation_noalloc(0), second)          # same state again: nothing left over from the last call
    assert np.all(g.correlation_noalloc(1) == 0)                     # against a snapshot of the current state
    g.close()


def test_noalloc_two_handles_share_the_array(sg):
    """The array belongs to the library, not to a handle: calls on two handles, one after the other, do not mix."""
    a = sg.Sim(sg.SG_MODEL_VB, 9000, 4.0, 1.0, 5, 2)
    b = sg.Sim(sg.SG_MODEL_VB, 700, 4.0, 0.6, 6, 8)
    for h in (a, b):
        h.snapshot(0)
        h.sweep(2)
    ca, cb = a.correlation_noalloc(0), b.correlation_noalloc(0)
    assert np.array_equal(ca, a.correlation(0)) and np.array_equal(cb, b.correlation(0))
    assert np.array_equal(a.correlation_noalloc(0), ca)
    a.close(); b.close()


def test_noalloc_rejects_what_it_cannot_serve(sg):
    from paper_1906_11195_b200.binding import SGError

    big = sg.Sim(sg.SG_MODEL_VB, 200, 4.0, 1.0, 1, 65)               # one word beyond the static array
    big.snapshot(0)
    with pytest.raises(SGError, match="at most 64 words"):
        big.correlation_noalloc(0)
    assert np.all(big.correlation(0) == 0)                           # the existing path is unaffected
    big.close()
    small = sg.Sim(sg.SG_MODEL_VB, 200, 4.0, 1.0, 1, 1)
    with pytest.raises(SGError, match="never written"):
        small.correlation_noalloc(3)
    small.close()
    sk = sg.Sim(sg.SG_MODEL_SK, 64, 0.0, 0.6, 1, 1)
    sk.snapshot(0)
    with pytest.raises(SGError, match="graph models only"):
        sk.correlation_noalloc(0)
    sk.close()
