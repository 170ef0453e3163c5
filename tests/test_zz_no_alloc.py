"""The allocation-free entry point mrd_meshgen_orient2d_static (include/mrd.h) against the existing path
mrd_meshgen_orient2d: integer work, so the signs and the count of tests that took the exact path must be IDENTICAL -- on two
calls in a row that share the static scratch (the second with fewer undecided tests than the first, so that a stale work list
or a counter that was not cleared would show), on an empty call, and at the limit of the scratch; a call beyond the limit is
rejected with a message that says so.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mrdb():
    import torch
    assert torch.cuda.is_available()
    import paper_1705_02028_b200.binding as b
    return b


def grid_triples(n, seed, ulps):
    """Triples of points of a grid with exactly representable coordinates (many exactly collinear), each coordinate moved by
    up to `ulps` units in the last place: with ulps = 0 or 1 the filter cannot decide a good share of them."""
    rng = np.random.default_rng(seed)
    gi, gj = np.meshgrid(np.arange(24), np.arange(24))
    xy = np.stack([gi.ravel(), gj.ravel()], axis=1) / 16.0
    if ulps:
        xy = xy + np.spacing(np.abs(xy) + 0.0625) * rng.integers(-ulps, ulps + 1, size=xy.shape)
    idx = rng.integers(0, xy.shape[0], size=(n, 3)).astype(np.int32)
    return xy, idx


def both_paths(mrdb, xy, idx):
    import torch
    dxy = torch.tensor(xy, dtype=torch.float64, device="cuda")
    didx = torch.tensor(idx, dtype=torch.int32, device="cuda")
    ref, ref_exact = mrdb.meshgen_orient2d(dxy, didx)
    sign = torch.full((idx.shape[0],), 7, dtype=torch.int8, device="cuda")
    n_exact = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    mrdb.meshgen_orient2d_static(dxy, didx, sign, n_exact)
    torch.cuda.synchronize()
    return ref.cpu().numpy(), ref_exact, sign.cpu().numpy(), int(n_exact.item())


def test_static_scratch_entry_point_matches_the_allocating_path_on_calls_in_a_row(mrdb):
    import torch
    first = grid_triples(200000, 1, ulps=1)          # many undecided tests: a long work list
    second = grid_triples(50000, 2, ulps=40)         # fewer of them, other points: the list of call 1 must not leak in
    third = grid_triples(3000, 3, ulps=0)            # exactly collinear triples: sign 0 through the exact path
    counts = []
    for xy, idx in (first, second, third, first):
        ref, ref_exact, got, got_exact = both_paths(mrdb, xy, idx)
        assert np.array_equal(got, ref) and got_exact == ref_exact
        assert set(np.unique(got)) <= {-1, 0, 1}
        counts.append(got_exact)
    assert counts[0] > counts[1] > 0 and counts[2] > 0 and counts[3] == counts[0]
    xy3, idx3 = third                                   # on the unperturbed grid the determinant is an integer / 256: count the zeros exactly
    g = np.rint(xy3 * 16).astype(np.int64)[idx3]
    det = (g[:, 0, 0] - g[:, 2, 0]) * (g[:, 1, 1] - g[:, 2, 1]) - (g[:, 0, 1] - g[:, 2, 1]) * (g[:, 1, 0] - g[:, 2, 0])
    got3 = both_paths(mrdb, xy3, idx3)[2]
    assert np.array_equal(got3, np.sign(det)) and (det == 0).sum() > 10
    # a sample against the definition itself (the oracle's rational arithmetic)
    from oracle import meshgen as mg
    xy, idx = second
    got = both_paths(mrdb, xy, idx)[2]
    for k in range(0, 50000, 250):
        assert got[k] == mg.orient2d(*xy[idx[k]])
    # nothing to do, and no output asked for
    empty = torch.empty((0, 3), dtype=torch.int32, device="cuda")
    mrdb.meshgen_orient2d_static(torch.tensor(xy, device="cuda"), empty, torch.empty(0, dtype=torch.int8, device="cuda"))
    torch.cuda.synchronize()


def test_static_scratch_limit(mrdb):
    import torch
    nmax = mrdb.MESHGEN_STATIC_MAX_TESTS
    xy, idx = grid_triples(nmax, 4, ulps=0)          # the largest call, and one in which about a sixth of the tests go to the list
    ref, ref_exact, got, got_exact = both_paths(mrdb, xy, idx)
    assert np.array_equal(got, ref) and got_exact == ref_exact and got_exact > 1000
    dxy = torch.tensor(xy, dtype=torch.float64, device="cuda")
    big = torch.zeros((nmax + 1, 3), dtype=torch.int32, device="cuda")
    with pytest.raises(mrdb.MrdError) as ex:
        mrdb.meshgen_orient2d_static(dxy, big, torch.empty(nmax + 1, dtype=torch.int8, device="cuda"))
    assert ex.value.code == mrdb.MRD_EINVAL and "exceed the static scratch" in str(ex.value) and str(nmax) in str(ex.value)
    ref, ref_exact, got, got_exact = both_paths(mrdb, *grid_triples(1000, 5, ulps=1))   # still usable after the rejection
    assert np.array_equal(got, ref) and got_exact == ref_exact
