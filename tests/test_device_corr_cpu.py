"""CPU-only: the correlation fitness's reduction (Eq. 1-2; csrc/fit_corr.cuh) run on the host: the device's own
functions, compiled for the host as well (IEEE single precision throughout, so the host build computes the device's bits; the library's
SASS is unchanged), on one warp of the SIMT emulator in the kernels' layout (beagle_debug_corr).

Against the oracle (orc_eval_corr: the definition as two-pass sums in fp64 with a certified bound, pinned by P19), under the same
three-class parity rule as on the GPU: programs 'x_j' make the per-case outputs whatever the test wants them to be. And the two ways
the kernels take (the general pass of the blockwise kernel, the pass with the target's side precomputed of the interpreter kernel)
give the same bits.
"""
import numpy as np
import pytest

from paper_2607_06731_b200 import api, colonies
from tests import parity

M = 10000.0


def _outputs(rng, y, kind):
    n = len(y)
    yy = np.where(np.isfinite(y), y, 0.0).astype(np.float64)
    if kind == 0: f = 0.8 * yy + 0.6 * rng.standard_normal(n)                   # correlated
    elif kind == 1: f = rng.standard_normal(n)                                  # uncorrelated
    elif kind == 2: f = -3.0 * yy + 7.0                                         # r = -1
    elif kind == 3: f = np.full(n, 2.5)                                         # constant: zero variance, r = 0
    elif kind == 4: f = 1e6 + 0.5 * yy + 0.1 * rng.standard_normal(n)           # a large offset: what the shift is for
    elif kind == 5: f = 1e15 * (yy + 0.3 * rng.standard_normal(n))              # large magnitude (squares near 1e30)
    elif kind == 6: f = 1e-20 * (yy + rng.standard_normal(n))                   # tiny magnitude
    else: f = yy ** 3 + rng.standard_normal(n)
    f = f.astype(np.float32)
    if kind % 3 == 1 and n > 4:                                                 # some outputs invalid
        f[rng.integers(0, n, max(1, n // 20))] = rng.choice([np.nan, np.inf, -np.inf])
    return f


@pytest.mark.parametrize("N", [1, 2, 3, 17, 128, 511, 512, 513, 700, 1023, 1024])
@pytest.mark.parametrize("bad_targets", [False, True])
def test_device_reduction_on_the_host_against_the_oracle(oracle, N, bad_targets):
    rng = np.random.default_rng(N * 2 + bad_targets)
    y = (rng.standard_normal(N) * 3 + 1).astype(np.float32)
    if bad_targets and N > 2:
        y[rng.integers(0, N, max(1, N // 15))] = rng.choice([np.nan, np.inf])
    d = 16
    X = np.stack([_outputs(rng, y, j % 8) for j in range(d)], axis=1).astype(np.float32)
    tok = np.array([colonies.token(colonies.OP["LOAD"], j) for j in range(d)], np.int32)
    lengths = np.ones(d, np.int32)
    tax = M * N / 85.0 / 64.0
    orc = oracle.evaluate_corr(tok, lengths, np.zeros(1, np.float32), X, y, M, tax)
    got = np.array([api.beagle_debug_corr(X[:, j], y, 1, M, tax, pre=False) for j in range(d)], np.float32)
    pre = np.array([api.beagle_debug_corr(X[:, j], y, 1, M, tax, pre=True) for j in range(d)], np.float32)
    assert np.array_equal(got.view(np.uint32), pre.view(np.uint32)), "the two passes of the kernels disagree"
    sub = {k: orc[k] for k in ("fitness", "bound", "flags", "depth")}
    rep = parity.compare(got, sub)
    assert len(rep["bad"]) == 0, parity.describe(rep, got, sub)
    assert rep["strict"] + rep["conditioned"] + rep["invalid"] >= d // 2        # the rule is not vacuous
    # a constant output scores exactly the invalid-pair term minus the tax
    st = orc["stats"]
    j = 3
    assert got[j] == np.float32(np.float32(-M * np.float32(st[j, 2] - st[j, 3])) - np.float32(tax))


def test_closed_forms_and_exact_cases(oracle):
    rng = np.random.default_rng(9)
    N = 512
    y = rng.integers(-50, 50, N).astype(np.float32)                             # small integers: every sum below is exact in fp32
    # f = y: r = 1 exactly, the score is M N
    assert api.beagle_debug_corr(y, y, 3, M, 0.0) == np.float32(M * N)
    # f = -y: r = -1, r^4 = 1
    assert api.beagle_debug_corr(-y, y, 3, M, 0.0) == np.float32(M * N)
    # the tax: minus tax * length, exactly
    assert api.beagle_debug_corr(y, y, 7, M, 2.0) == np.float32(M * N - 14.0)
    # all targets invalid: every pair is one-sided (c1 = N): -M N; both sides invalid: +M N (Eq. 2)
    nan = np.full(N, np.nan, np.float32)
    assert api.beagle_debug_corr(y, nan, 1, M, 0.0) == np.float32(-M * N)
    assert api.beagle_debug_corr(nan, nan, 1, M, 0.0) == np.float32(M * N)
    # one valid pair is no correlation: r = 0, the rest counts as invalid pairs
    f = nan.copy(); f[5] = 1.0
    assert api.beagle_debug_corr(f, y, 1, M, 0.0) == np.float32(-M * (N - 1))
    # independent of the order of the cases up to rounding; exactly so for data whose sums are exact
    perm = rng.permutation(N)
    f = (2 * y + rng.integers(-3, 3, N)).astype(np.float32)
    a, b = api.beagle_debug_corr(f, y, 1, M, 0.0), api.beagle_debug_corr(f[perm], y[perm], 1, M, 0.0)
    assert abs(a - b) <= 2e-6 * abs(a)


def test_corr_argument_errors():
    import ctypes
    l = api.lib()
    one = np.zeros(1, np.float32)
    out = ctypes.c_float()
    assert l.beagle_debug_corr(None, one.ctypes.data, 1, 1, 1.0, 0.0, 0, ctypes.byref(out)) == api.ERR_INVALID_ARG
    assert l.beagle_debug_corr(one.ctypes.data, one.ctypes.data, 0, 1, 1.0, 0.0, 0, ctypes.byref(out)) == api.ERR_INVALID_ARG
    assert l.beagle_debug_corr(one.ctypes.data, one.ctypes.data, 1025, 1, 1.0, 0.0, 0, ctypes.byref(out)) == api.ERR_INVALID_ARG
    assert l.beagle_debug_corr(one.ctypes.data, one.ctypes.data, 1, 0, 1.0, 0.0, 0, ctypes.byref(out)) == api.ERR_INVALID_ARG


def test_random_offsets_scales_and_case_counts(oracle):
    """Breadth: outputs and targets with offsets up to 1e7 and spreads from 1e-3 to 1e4, any correlation, case counts on both sides of
    the pass boundary, both passes of the kernels: every individual within the oracle's rule (4,800 more were sent by hand: none outside)."""
    rng = np.random.default_rng(31)
    tok = np.array([colonies.token(colonies.OP["LOAD"], j) for j in range(16)], np.int32)
    n_checked = 0
    for _ in range(25):
        N = int(rng.choice([2, 5, 33, 300, 512, 513, 640, 777, 1000, 1024]))
        yoff = float(rng.choice([0, 1, 1e3, 1e6, -1e5])) * rng.uniform(0.5, 2)
        ysp = 10 ** rng.uniform(-3, 3)
        y = (yoff + ysp * rng.standard_normal(N)).astype(np.float32)
        z = (y.astype(np.float64) - yoff) / ysp
        cols = []
        for j in range(16):
            off = float(rng.choice([0, 1, 1e2, 1e4, 1e6, 1e7, -1e6])) * rng.uniform(0.5, 2)
            sp = 10 ** rng.uniform(-3, 4)
            rho = rng.uniform(-1, 1)
            cols.append((off + sp * (rho * z + np.sqrt(1 - rho * rho) * rng.standard_normal(N))).astype(np.float32))
        X = np.stack(cols, 1)
        orc = oracle.evaluate_corr(tok, np.ones(16, np.int32), np.zeros(1, np.float32), X, y, M, 0.0)
        got = np.array([api.beagle_debug_corr(X[:, j], y, 1, M, 0.0, pre=bool(j % 2)) for j in range(16)], np.float32)
        sub = {k: orc[k] for k in ("fitness", "bound", "flags", "depth")}
        rep = parity.compare(got, sub)
        assert len(rep["bad"]) == 0, (N, yoff, ysp, parity.describe(rep, got, sub))
        n_checked += rep["strict"] + rep["conditioned"]
    assert n_checked > 300
