"""cdz_sample_noalloc (include/cdz.h): the stochastic traceback (PAPER.md S4c, Alg S4.4) with its decision stacks in a
static device array instead of a stream-ordered allocation, for callers that cannot call cudaMalloc.  Same kernel, same uniforms: the
samples must be bit-identical to cdz_sample's (the tolerance of every sampler test here is exact equality).  Collected last on purpose
(pytest -x): a failure here hides no other test.  Runs alone in a fresh process as well as after the other tests: it
builds its own tables and depends on nothing they leave behind."""
import pytest

from paper_2604_19718_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2604_19718_b200 import binding, build

    build.build()
    return binding


def _pair(B, tab, J, seed, fill):
    """(existing path, no-alloc path) for one (J, seed); the no-alloc outputs are pre-filled so that unwritten entries would show."""
    import torch

    seq0, pair0 = tab.sample(J, seed)
    seq1 = torch.full((J, tab.n), fill, dtype=torch.uint8, device="cuda")
    pair1 = torch.full((J, tab.n), -7 - fill, dtype=torch.int32, device="cuda")
    tab.sample_noalloc(J, seed, seq1, pair1)
    torch.cuda.synchronize()
    return seq0, pair0, seq1, pair1


def test_noalloc_samples_equal_existing_path_two_calls_in_a_row(B):
    """Two calls back to back on the shared static scratch (different J and seed, the second smaller so that stale stack contents of
    the first lie beside and beyond it), then the first again: every sample bit-identical to cdz_sample's."""
    import torch

    d = I.design(5, 0, 60)  # 180 nt, codon-pair tensor train: multiloops and interior loops occur in the samples
    tab, _ = B.inside(B.Model(I.nn_model()), B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
    for J, seed, fill in ((300, 20260419, 9), (64, 7, 5), (300, 20260419, 3)):
        seq0, pair0, seq1, pair1 = _pair(B, tab, J, seed, fill)
        assert torch.equal(seq0, seq1)
        assert torch.equal(pair0, pair1)
        assert int(seq1.max()) <= 3 and int(pair1.min()) >= -1


def test_noalloc_single_codon_design_and_limit(B):
    """Config-1 design (60 nt, single-codon train) at the largest J the static scratch holds, one more is rejected with a message."""
    import torch

    d = I.design(1, 0)
    tab, _ = B.inside(B.Model(I.nn_model()), B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
    cap = tab.n // 4 + 16
    jmax = B.NOALLOC_STACK_ITEMS // cap
    seq0, pair0, seq1, pair1 = _pair(B, tab, jmax, 11, 8)
    assert torch.equal(seq0, seq1) and torch.equal(pair0, pair1)
    seq = torch.empty((jmax + 1, tab.n), dtype=torch.uint8, device="cuda")
    pair = torch.empty((jmax + 1, tab.n), dtype=torch.int32, device="cuda")
    with pytest.raises(B.CdzError, match="static scratch"):
        tab.sample_noalloc(jmax + 1, 11, seq, pair)
    # the rejected call launched nothing and the entry point still works
    seq0, pair0, seq1, pair1 = _pair(B, tab, 10, 12, 6)
    assert torch.equal(seq0, seq1) and torch.equal(pair0, pair1)
