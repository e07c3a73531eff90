"""-m gpu: the correlation fitness (Eq. 1-2) through beagle_eval_fit against
the oracle's orc_eval_corr (pinned by P19), under the same three-class parity rule as the MSE path."""
import numpy as np
import pytest

from paper_2607_06731_b200 import colonies as C
from paper_2607_06731_b200.colonies import OP, token
from tests import parity
from tests.util import asm, pack

pytestmark = pytest.mark.gpu

M = 10000.0
FIT_MSE, FIT_CORR = 0, 1
QNAN = 0x7FC00000


def _bits(a):
    return np.asarray(a, np.float32).view(np.uint32)


def _texts(rng, n, d, names):
    from tests.util import random_gcl_programs
    return random_gcl_programs(rng, n, d, names)


HOT = ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP"]


@pytest.mark.parametrize("N,d,seed", [(512, 5, 1), (1024, 9, 2), (200, 3, 3), (700, 16, 4), (33, 1, 5)])
def test_correlation_parity_random_programs(oracle, N, d, seed):
    from tests.gpu_util import gpu_eval_fit
    rng = np.random.default_rng(seed)
    X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
    y = (X[:, 0] * X[:, d - 1] + np.sin(X[:, 0]) + 0.1 * rng.standard_normal(N)).astype(np.float32)
    texts = _texts(rng, 1500, d, HOT) + ["x0", "1.5", "x0 x0 SUB", f"x0 x{d - 1} MUL x0 SIN ADD"]
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts)
    tax = M * N / 85.0 / 64.0
    a = gpu_eval_fit(g, l, c, X, y, FIT_CORR, M, tax)
    orc = oracle.evaluate_corr(g, l, c, X, y, M, tax)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    assert rep["strict"] > 0.5 * len(texts), parity.describe(rep, a, orc)
    # the model that is the target up to noise scores close to M N; a constant scores exactly -tax L
    assert a[-1] > 0.9 * M * N - tax * 7 and a[-3] == np.float32(-tax * 1)


def test_correlation_invalid_pairs_counts(oracle):
    """Eq. 2's c1 / c2 on the GPU: targets with NaN / Inf, model outputs that overflow or leave a domain."""
    from tests.gpu_util import gpu_eval_fit
    rng = np.random.default_rng(7)
    N, d = 777, 3
    X = rng.uniform(-2, 2, (N, d)).astype(np.float32)
    X[rng.integers(0, N, 40), 2] = 1e30                  # x2 * x2 overflows there
    y = (2.0 * X[:, 0] - X[:, 1]).astype(np.float32)
    y[rng.integers(0, N, 30)] = np.nan
    y[rng.integers(0, N, 30)] = np.inf
    texts = ["x0 2 MUL x1 SUB", "x0 2 MUL x1 SUB x2 x2 MUL 0 MUL ADD", "x0 ARCSIN", "x2 x2 MUL", "x0 x1 MUL x2 x2 MUL x2 MUL SUB",
             "x0 x1 DIV x2 x2 MUL x2 x2 MUL SUB ADD"] + _texts(rng, 400, d, HOT + ["SQUARE", "ARCSIN"])
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts)
    a = gpu_eval_fit(g, l, c, X, y, FIT_CORR, M, 0.0)
    orc = oracle.evaluate_corr(g, l, c, X, y, M, 0.0)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    st = orc["stats"]
    assert st[0, 2] > 0 and st[0, 3] == 0 and st[1, 3] > 0 and st[2, 2] > 100          # the cases really occur
    # perfect model on the valid pairs: the score is an exact integer combination of the counts
    assert a[0] == np.float32(M * st[0, 1] - M * (st[0, 2] - st[0, 3])) or abs(a[0] - (M * st[0, 1] - M * (st[0, 2] - st[0, 3]))) <= 1e-5 * M * N
    # all targets invalid
    yn = np.full(N, np.nan, np.float32)
    a = gpu_eval_fit(g, l, c, X, yn, FIT_CORR, M, 0.0)
    orc = oracle.evaluate_corr(g, l, c, X, yn, M, 0.0)
    assert len(parity.compare(a, orc)["bad"]) == 0
    assert a[0] == np.float32(-M * N)                    # f finite everywhere, y nowhere: c1 = N


def test_correlation_fast_and_blockwise_paths_bit_identical(oracle):
    """k_eval and k_eval_blockwise share the reduction: `A` (interpreter) and `A DUP DEL` (slow list, blockwise kernel)
    give the same bits at tax 0; so does a colony evaluated where the fitness cases do not fit tensor memory."""
    from tests.gpu_util import gpu_eval_fit
    rng = np.random.default_rng(8)
    for N, d in ((512, 4), (1024, 7), (300, 2)):
        X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
        y = (X[:, 0] - X[:, 1] ** 2).astype(np.float32)
        y[5] = np.inf
        texts = _texts(rng, 300, d, HOT)
        texts = [t for t in texts if len(t.split()) < 100]
        consts = []
        fast = [asm(t, consts)[0] for t in texts]
        slow = [asm(t + " DUP DEL", consts)[0] for t in texts]
        g, l, c = pack(fast + slow, consts)
        a = gpu_eval_fit(g, l, c, X, y, FIT_CORR, M, 0.0)
        n = len(texts)
        assert np.array_equal(_bits(a[:n]), _bits(a[n:]))
    # d = 20 at N = 1024 does not fit tensor memory: the whole call runs blockwise; columns >= 7 unused by the programs
    rng = np.random.default_rng(8)
    X = rng.uniform(-3, 3, (1024, 7)).astype(np.float32)
    Xw = np.concatenate([X, rng.uniform(-1, 1, (1024, 13)).astype(np.float32)], axis=1)
    y = (X[:, 0] - X[:, 1] ** 2).astype(np.float32)
    texts = [t for t in _texts(rng, 300, 7, HOT) if len(t.split()) < 100]
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts)
    a = gpu_eval_fit(g, l, c, X, y, FIT_CORR, M, 3.0)
    b = gpu_eval_fit(g, l, c, Xw, y, FIT_CORR, M, 3.0)
    assert np.array_equal(_bits(a), _bits(b))


def test_correlation_degenerate_and_malformed(oracle):
    from tests.gpu_util import gpu_eval_fit, gpu_eval
    N = 64
    X = np.linspace(-1, 1, N, dtype=np.float32).reshape(-1, 1)
    y = (3 * X[:, 0] + 1).astype(np.float32)
    T = token
    progs = [np.array([T(OP["LOAD"], 0)], np.int32),                                  # r = 1
             np.array([T(OP["LOAD"], 0), T(OP["SIGN"])], np.int32),                   # r = -1: same score
             np.array([T(OP["CONST"], 0)], np.int32),                                 # zero variance: r = 0
             np.array([T(OP["ADD"])], np.int32),                                      # malformed
             np.array([T(OP["LOAD"], 0), T(OP["LOAD"], 0), T(OP["SUB"])], np.int32)]  # exactly 0 everywhere
    g, l, c = pack(progs, np.array([0.37], np.float32))
    a = gpu_eval_fit(g, l, c, X, y, FIT_CORR, M, 2.0)
    assert abs(a[0] - (M * N - 2.0)) <= 1e-5 * M * N and abs(a[1] - (M * N - 4.0)) <= 1e-5 * M * N
    assert a[2] == np.float32(-2.0) and _bits(a[3:4])[0] == QNAN and a[4] == np.float32(-6.0)
    # constant target: r = 0 for everyone
    a = gpu_eval_fit(g, l, c, X, np.full(N, 2.5, np.float32), FIT_CORR, M, 0.0)
    assert a[0] == 0 and a[1] == 0 and a[2] == 0 and a[4] == 0
    # one valid pair only
    y1 = np.full(N, np.nan, np.float32); y1[7] = 1.0
    a = gpu_eval_fit(g, l, c, X, y1, FIT_CORR, M, 0.0)
    assert a[0] == np.float32(-M * (N - 1))
    # fit = MSE through the same entry point is beagle_eval; an unknown fit is refused
    m1 = gpu_eval_fit(g, l, c, X, y, FIT_MSE, 0.0, 0.5)
    m2 = gpu_eval(g, l, c, X, y, 0.5)
    assert np.array_equal(_bits(m1), _bits(m2))
    with pytest.raises(Exception):
        gpu_eval_fit(g, l, c, X, y, 7, M, 0.0)
    # and the MSE path is untouched by a correlation call before it
    m3 = gpu_eval(g, l, c, X, y, 0.5)
    assert np.array_equal(_bits(m2), _bits(m3))


def test_correlation_config_colony_sampled(oracle):
    """A colony with the structure of BASELINE.json's configs (ramped trees, 20 % unary) at N = 512: every individual
    against the oracle."""
    from tests.gpu_util import gpu_eval_fit
    col = C.make_colony(3, P=3000)
    g, l, c, X, y = col.genomes, col.lengths, col.consts, col.X, col.y
    a = gpu_eval_fit(g, l, c, X, y, FIT_CORR, M, 100.0)
    orc = oracle.evaluate_corr(g, l, c, X, y, M, 100.0)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    assert rep["strict"] > 900 and rep["exempt"] < 1500, parity.describe(rep, a, orc)


@pytest.mark.parametrize("fit,M_", [(FIT_CORR, M), (2, M), (5, M)])
def test_chunked_fit_bit_identical_to_resident(oracle, fit, M_):
    """beagle_eval_chunked_fit (host genomes, small device budget: several chunks) against beagle_eval_fit, bit for bit,
    for the correlation fitness and two of the Std family."""
    import torch
    from paper_2607_06731_b200 import api
    from tests.gpu_util import gpu_eval_fit
    col = C.make_colony(2, P=30000)
    g, l, c, X, y = col.genomes, col.lengths, col.consts, col.X, col.y
    a = gpu_eval_fit(g, l, c, X, y, fit, M_, 25.0)
    P, (N, d) = len(l), X.shape
    hg = torch.from_numpy(np.ascontiguousarray(g, np.int32)).pin_memory()
    hl = torch.from_numpy(np.ascontiguousarray(l, np.int32)).pin_memory()
    hc = torch.from_numpy(np.ascontiguousarray(c, np.float32)).pin_memory()
    Xd, yd = torch.from_numpy(X).cuda(), torch.from_numpy(y).cuda()
    out = torch.full((P,), -1.0, dtype=torch.float32, device="cuda")
    budget = 1 << 20                                           # about 1 MiB of staging: several chunks
    api.beagle_eval_chunked_fit(hg, hl, P, hc, len(c), Xd, yd, N, d, fit, M_, 25.0, out, budget, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(_bits(a), _bits(out.cpu().numpy()))
    assert api.raw_status("beagle_eval_chunked_fit", api._ptr(hg), api._ptr(hl), P, api._ptr(hc), len(c), api._ptr(Xd), api._ptr(yd),
                          N, d, 9, M_, 25.0, api._ptr(out), budget, None) != 0


@pytest.mark.parametrize("fit,power", [(FIT_CORR, 0), (2, 1)])
def test_full_size_config3_sampled_then_ranked(oracle, fit, power):
    """BASELINE.json's config 3 at full size (the launch configuration `bench.py --fit ...` times): every 701st
    individual and the 128 longest against the oracle; properties that hold at any size; then beagle_rank on the
    resident fitness vector against oracle/ranking.py's sort-based restatement (pinned by P20)."""
    import torch
    from paper_2607_06731_b200 import api
    from oracle import ranking as R
    col = C.make_colony(3)
    P, (N, d) = col.P, col.X.shape
    tax = M * N / 85.0
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g, l, c, X, y = dev(col.genomes), dev(col.lengths), dev(col.consts), dev(col.X), dev(col.y)
    out = torch.full((P,), -12345.0, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    api.beagle_eval_fit(g, l, P, c, len(col.consts), X, y, N, d, fit, M, tax, out, st)
    torch.cuda.synchronize()
    a = out.cpu().numpy()
    sel = np.unique(np.concatenate([np.arange(0, P, 701), np.argsort(-col.lengths, kind="stable")[:128]]))
    off = np.concatenate([[0], np.cumsum(col.lengths, dtype=np.int64)])
    gs = np.concatenate([col.genomes[off[p]:off[p + 1]] for p in sel]); ls = col.lengths[sel]
    orc = (oracle.evaluate_corr(gs, ls, col.consts, col.X, col.y, M, tax) if fit == FIT_CORR
           else oracle.evaluate_std(gs, ls, col.consts, col.X, col.y, power, M, tax))
    rep = parity.compare(a[sel], orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a[sel], orc)
    assert rep["strict"] + rep["conditioned"] > 0.4 * len(sel), parity.describe(rep, a[sel], orc)
    # any size: every individual got a value; a score cannot exceed M per case, nor fall below -M per case, tax aside
    assert not np.any(a == np.float32(-12345.0))
    fin = np.isfinite(a)
    sc = a[fin].astype(np.float64) + tax * col.lengths[fin]
    assert np.all(sc <= M * N * (1 + 1e-5)) and np.all(sc >= -M * N * (1 + 1e-5))
    # the step after scoring, on the vector still on the device
    rng = np.random.default_rng(3)
    sample = rng.integers(0, P, 100)
    dec = torch.empty(P, dtype=torch.uint8, device="cuda"); hist = torch.empty(10, dtype=torch.int64, device="cuda")
    api.beagle_rank(out, P, dev(sample.astype(np.int64)), 100, True, dec, hist, st)
    torch.cuda.synchronize()
    gd = R.goodness(a, True)
    want = np.minimum(9, np.searchsorted(np.sort(gd[sample]), gd, side="left") // 10).astype(np.uint8)
    assert np.array_equal(dec.cpu().numpy(), want) and np.array_equal(hist.cpu().numpy(), np.bincount(want, minlength=10))
