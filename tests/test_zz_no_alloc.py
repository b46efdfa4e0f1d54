"""mlcc_match_root_sets_noalloc: the matcher for callers that may not allocate device memory (its bins live in a static
4 MiB device array; n <= 8192 points per set).  Checked against the existing path, mlcc_match_root_sets, on two calls
in a row (the second finds the first call's contents in the shared scratch), and against the oracle's brute force.
Collected last on purpose (the file name): a failure here must not hide the other GPU tests under `pytest -x`."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2506_02121_b200 import api as a
    a.lib()
    return a


def _sets(S, n, seed, spread):
    """b: S sets of n distinct points; a: b permuted and displaced by ~1e-11; a few sets spoiled on purpose."""
    rng = np.random.default_rng(seed)
    b = rng.uniform(-spread, spread, size=(S, n, 2))
    a = np.empty_like(b)
    for s in range(S):
        a[s] = b[s][rng.permutation(n)] + rng.normal(scale=1e-11, size=(n, 2))
    if S > 3 and n > 1:
        a[1, 0] = a[1, 1]                       # one b_j taken twice, one missed: not a bijection
        a[3, n // 2] += 1e-6                    # a pair beyond the tolerance
    return a, b


def test_noalloc_matcher_equals_the_allocating_path_on_two_calls_in_a_row(api, orc):
    torch.cuda.synchronize()
    err = torch.empty((0,), dtype=torch.float64, device="cuda")
    # two calls in a row with different shapes and data, then the first again: stale scratch must not matter
    for S, n, seed, spread in ((40, 400, 1, 25.0), (7, 8192, 2, 300.0), (40, 400, 1, 25.0), (3, 1, 4, 1.0), (257, 20, 5, 5.0)):
        a, b = _sets(S, n, seed, spread)
        da, db = torch.as_tensor(a).cuda(), torch.as_tensor(b).cuda()
        want_err, want_bij = api.match_root_sets(da, db, 1e-10)                     # the existing path
        err = torch.full((S,), -1.0, dtype=torch.float64, device="cuda")
        bij = torch.full((S,), -1, dtype=torch.int32, device="cuda")
        before = torch.cuda.memory_allocated()
        api.match_root_sets_noalloc(da, db, 1e-10, err, bij)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before
        # same pairs, same arithmetic: the distances are the same numbers, the flags the same integers
        assert torch.equal(bij, want_bij)
        assert float((err - want_err).abs().max()) <= 1e-15 * (1.0 + float(want_err.max()))
        if S * n <= 20000:                                                          # and both equal the brute force
            o_err, o_bij = orc.match_root_sets(a, b, 1e-10)
            assert np.array_equal(bij.cpu().numpy(), o_bij)
            assert np.abs(err.cpu().numpy() - o_err).max() <= 1e-15 * (1.0 + o_err.max())
        if S > 3 and n > 1:
            assert int(bij[1]) == 0 and int(bij[3]) == 0 and int(bij[0]) == 1
    assert err.shape == (257,)


def test_noalloc_matcher_rejects_what_does_not_fit(api):
    a = torch.zeros((1, 8193, 2), dtype=torch.float64, device="cuda")
    err = torch.zeros((1,), dtype=torch.float64, device="cuda")
    bij = torch.zeros((1,), dtype=torch.int32, device="cuda")
    with pytest.raises(api.MlccError) as e:
        api.match_root_sets_noalloc(a, a, 1e-10, err, bij)
    assert "8192" in str(e.value)
    # an empty batch is a no-op, a non-finite point is reported as in the allocating path
    empty = torch.zeros((0, 5, 2), dtype=torch.float64, device="cuda")
    api.match_root_sets_noalloc(empty, empty, 1e-10, err[:0], bij[:0])
    bad = torch.rand((2, 50, 2), dtype=torch.float64, device="cuda")
    good = bad.clone()
    bad[1, 7, 0] = float("nan")
    err2 = torch.zeros((2,), dtype=torch.float64, device="cuda")
    bij2 = torch.zeros((2,), dtype=torch.int32, device="cuda")
    api.match_root_sets_noalloc(bad, good, 1e-10, err2, bij2)
    assert bij2.tolist() == [1, 0] and bool(torch.isinf(err2[1]))
