"""SURVEY 8f-1 (PAPER.md S4f line 779): batched fixed-sequence evaluation of sampled sequences through the C ABI
(`cdz_eval_sequences`), against oracle pieces that share nothing with the tensor recursion: the scalar fixed-sequence McCaskill
(`orc_mccaskill`) for log Z(phi), `orc_logweight` of the structure-free state for log W(phi), and `orc_marginals` of the
one-operator-per-position train for the unpaired probabilities."""
import numpy as np
import pytest

from paper_2604_19718_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2604_19718_b200 import binding, build

    build.build()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle

    return oracle


@pytest.mark.parametrize("cfg,L,J", [(1, 12, 24), (5, 13, 24), (5, 150, 40), (1, 200, 12)])
def test_eval_sampled_sequences(B, O, cfg, L, J):
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    mg = B.Model(m)
    tt = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    tg, lz_design = B.inside(mg, tt)
    seq, _ = tg.sample(J, d.sample_seed)
    seq = seq.cpu().numpy()
    small = d.n <= 40
    lz, lw, un = B.eval_sequences(mg, tt, seq, want_unpaired=small, max_batch=16)
    tto = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    nopair = -np.ones(d.n, dtype=np.int32)
    for k in range(J):
        want = O.mccaskill(m, seq[k])
        assert abs(lz[k] - want) <= 1e-9 * max(abs(want), 1.0), (k, lz[k], want)
        assert abs(lw[k] - O.logweight(m, tto, seq[k], nopair)) <= 1e-11 * max(1.0, abs(lw[k]))
    # a sampled sequence contributes W(phi) Z(phi) to Z: every term is below the total, and they are not all negligible
    assert (lz + lw <= lz_design + 1e-9).all()
    if small:
        for k in (0, J - 1):
            ops = [[(0, int(b), 0, 1.0)] for b in seq[k]]
            bo, _, _ = O.inside(m, O.TT.from_ops(ops)).marginals()
            np.testing.assert_allclose(un[k], np.diag(bo), atol=1e-10, rtol=0)


def test_eval_rejects_bad_input(B):
    mg = B.Model(I.nn_model())
    tt = B.TensorTrain.build("MW", 0)
    with pytest.raises(B.CdzError):
        B.eval_sequences(mg, tt, np.full((2, 6), 7, dtype=np.uint8))
    with pytest.raises(B.CdzError):
        B.eval_sequences(mg, tt, np.zeros((2, 9), dtype=np.uint8))
    lz, lw, _ = B.eval_sequences(mg, tt, np.array([[0, 3, 2, 3, 2, 2], [0, 0, 0, 0, 0, 0]], dtype=np.uint8))  # AUGUGG, AAAAAA
    assert np.isfinite(lw[0]) and lw[1] == -np.inf and np.isfinite(lz).all()
