"""-m gpu: Monte-Carlo ranking (Table 2) through beagle_rank against
oracle/ranking.py (pins P20). Integer work: bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _gpu_rank(f, sample, maximise, want_hist=True):
    import torch
    from paper_2607_06731_b200 import api
    P = len(f)
    fd = torch.from_numpy(np.ascontiguousarray(f, np.float32)).cuda()
    sd = torch.from_numpy(np.ascontiguousarray(sample, np.int64)).cuda()
    dec = torch.full((max(P, 1),), 255, dtype=torch.uint8, device="cuda")
    hist = torch.full((10,), -1, dtype=torch.int64, device="cuda") if want_hist else None
    api.beagle_rank(fd if P else None, P, sd, len(sample), maximise, dec if P else None, hist, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return dec[:P].cpu().numpy(), (hist.cpu().numpy() if want_hist else None)


@pytest.mark.parametrize("P,n_sample,seed", [(1000, 100, 1), (1 << 20, 100, 2), (37, 100, 3), (5000, 7, 4), (300000, 1024, 5), (1, 1, 6)])
def test_ranking_matches_oracle(P, n_sample, seed):
    from oracle import ranking as R
    rng = np.random.default_rng(seed)
    f = rng.standard_normal(P).astype(np.float32) * 100
    f[rng.random(P) < 0.03] = np.nan
    f[rng.random(P) < 0.03] = np.inf
    if seed % 2:
        f = np.round(f, 0)                                     # many ties
    sample = rng.integers(0, P, n_sample)
    for mx in (False, True):
        dec, hist = _gpu_rank(f, sample, mx)
        if P <= 5000:
            want, whist, _ = R.rank_deciles(f, sample, mx)
        else:                                                  # the oracle's double loop on a sample of the population,
            pick = rng.integers(0, P, 3000)                    # the histogram through the pinned sort restatement (P20)
            want_s, _, _ = R.rank_deciles(np.concatenate([f[sample], f[pick]]), np.arange(n_sample), mx)
            assert np.array_equal(dec[pick], want_s[n_sample:])
            g = R.goodness(f, mx)
            want = np.minimum(9, (10 * np.searchsorted(np.sort(g[sample]), g, side="left")) // n_sample).astype(np.uint8)
            whist = np.bincount(want, minlength=10)
        assert np.array_equal(dec, want) and np.array_equal(hist, whist) and hist.sum() == P


def test_ranking_follows_scoring_on_device(oracle):
    """The step after scoring: fitness stays on the device; deciles of a scored colony equal the oracle's on the oracle's
    fitness wherever the two fitness vectors order the sample the same way (here: compared on the GPU's own fitness)."""
    import torch
    from paper_2607_06731_b200 import api, colonies as C
    from oracle import ranking as R
    col = C.make_colony(2, P=20000)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g, l, c, X, y = dev(col.genomes), dev(col.lengths), dev(col.consts), dev(col.X), dev(col.y)
    P, (N, d) = len(col.lengths), col.X.shape
    fit = torch.empty(P, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    rng = np.random.default_rng(0)
    sample = rng.integers(0, P, 100)
    sd = dev(sample.astype(np.int64))
    dec = torch.empty(P, dtype=torch.uint8, device="cuda")
    hist = torch.empty(10, dtype=torch.int64, device="cuda")
    for fitk, mx in ((api.FIT_MSE, False), (api.FIT_CORRELATION, True)):
        api.beagle_eval_fit(g, l, P, c, len(col.consts), X, y, N, d, fitk, 10000.0, 1.0, fit, st)
        api.beagle_rank(fit, P, sd, 100, mx, dec, hist, st)
        torch.cuda.synchronize()
        want, whist, kids = R.rank_deciles(fit.cpu().numpy(), sample, mx)
        assert np.array_equal(dec.cpu().numpy(), want) and np.array_equal(hist.cpu().numpy(), whist)
        births = float((hist.cpu().numpy() * np.array(api.TABLE2)).sum())
        assert abs(births - kids.sum()) < 1e-3 * P and 0.5 * P < births < 2.0 * P     # Table 2 keeps the colony near its size


def test_ranking_arguments():
    import torch
    from paper_2607_06731_b200 import api
    f = torch.zeros(4, device="cuda"); s = torch.zeros(2000, dtype=torch.int64, device="cuda"); d = torch.zeros(4, dtype=torch.uint8, device="cuda")
    assert api.raw_status("beagle_rank", api._ptr(f), 4, api._ptr(s), 0, 0, api._ptr(d), None, None) != 0
    assert api.raw_status("beagle_rank", api._ptr(f), 4, api._ptr(s), 2000, 0, api._ptr(d), None, None) != 0
    assert api.raw_status("beagle_rank", None, 4, api._ptr(s), 100, 0, api._ptr(d), None, None) != 0
    assert api.raw_status("beagle_rank", None, 0, api._ptr(s), 100, 0, None, None, None) == 0
    api.beagle_rank(f, 4, s, 100, False, d)           # no histogram wanted
    torch.cuda.synchronize()
    assert d.cpu().tolist() == [0, 0, 0, 0]          # everyone ties with the sample: nobody strictly worse
