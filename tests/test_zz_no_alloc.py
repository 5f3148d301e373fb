"""tatrg_gram_static: the allocation-free Gram matrix (split-K scratch in a file-scope __device__ array) against tatrg_gram.
Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
EPS = 2.0 ** -52


@pytest.fixture(scope="module")
def torch():
    t = pytest.importorskip("torch")
    if not t.cuda.is_available():
        pytest.skip("no CUDA device")
    return t


def test_gram_static_matches_gram_on_two_calls_in_a_row(torch):
    import paper_2507_21909_b200 as T
    from tests import inputs
    limit = T.lib().tatrg_gram_static_max_scratch_bytes()
    assert limit == 16 << 20
    # two calls in a row on the same stream, different shapes, both split along K: the second must not see the first one's partials
    shapes = [(40000, 64), (33000, 300)]
    outs, refs = [], []
    for i, (m, n) in enumerate(shapes):
        assert 0 < T.lib().tatrg_gram_scratch_bytes(m, n) <= limit
        x = torch.from_numpy(inputs.random_tensor((m, n), 21 + i)).cuda()
        out = torch.empty((n, n), dtype=torch.float64, device="cuda")
        before = torch.cuda.memory_allocated()
        g = T.gram_static(x, out=out)
        assert torch.cuda.memory_allocated() == before          # torch allocated nothing either: x and out were there
        outs.append(g)
        refs.append((x, T.gram(x)))
    for (m, n), g, (x, ref) in zip(shapes, outs, refs):
        g, ref, xh = g.cpu().numpy(), ref.cpu().numpy(), x.cpu().numpy()
        assert np.abs(g - ref).max() <= 8 * EPS * m * np.abs(xh).max() ** 2      # tolerance of test_gram_symmetric_mode_matches_definition
        assert np.abs(g - xh.T @ xh).max() <= 8 * EPS * m * np.abs(xh).max() ** 2
        if n >= 256:
            assert np.array_equal(g, g.T)
    # the same input again after another call has used the array: identical bits
    again = T.gram_static(refs[0][0]).cpu().numpy()
    assert np.array_equal(again, outs[0].cpu().numpy())


def test_gram_static_rejects_sizes_beyond_the_array(torch):
    import paper_2507_21909_b200 as T
    m, n = 32768, 1024
    assert T.lib().tatrg_gram_scratch_bytes(m, n) > T.lib().tatrg_gram_static_max_scratch_bytes()
    x = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    with pytest.raises(T.TatrgError, match="static array holds"):
        T.gram_static(x)
