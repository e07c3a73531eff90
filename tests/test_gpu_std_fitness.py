"""-m gpu: the Std integer-reward fitness family (Eq. 5) through beagle_eval_fit
against the oracle's orc_eval_std (pins P21). Rewards are integers decided in fp32 on both sides: programs whose
commands are correctly rounded are bit-exact; the others fall under the three-class rule with the oracle's bound."""
import numpy as np
import pytest

from tests import parity
from tests.util import asm, pack

pytestmark = pytest.mark.gpu

M = 10000.0
FITS = {1: 2, 2: 3, 3: 4, 8: 5}          # power -> BEAGLE_FIT_STD*


def _bits(a):
    return np.asarray(a, np.float32).view(np.uint32)


def _texts(rng, n, d, names):
    from tests.util import random_gcl_programs
    return random_gcl_programs(rng, n, d, names)


@pytest.mark.parametrize("power", [1, 2, 3, 8])
def test_std_exact_for_correctly_rounded_programs(oracle, power):
    """+ - * only: per-case outputs equal the oracle's fp32 mirror (every command rounded to fp32), so every reward and
    the score are bit-exact."""
    from tests.gpu_util import gpu_eval_fit
    rng = np.random.default_rng(30 + power)
    N, d = 777, 3
    X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
    y = (X[:, 0] * X[:, 1] - X[:, 2]).astype(np.float32)
    y[::50] = 0.0; X[::50, :] = 0.0                                  # max(|f|, |y|) = 0 happens
    y[7] = np.nan; y[8] = np.inf
    X[9, 0] = 3e38; X[9, 1] = 2.0                                     # x0 * x1 overflows: an invalid output
    texts = _texts(rng, 500, d, ["ADD", "SUB", "MUL"]) + ["x0 x1 MUL x2 SUB", "x0 x0 ADD", "x2 x1 x0 MUL SUB"]
    texts = [t for t in texts if "." not in t]                       # variables only: no constant folding questions
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts if consts else np.zeros(1, np.float32))
    a = gpu_eval_fit(g, l, c, X, y, FITS[power], M, 117.0)
    orc = oracle.evaluate_std(g, l, c, X, y, power, M, 117.0, contract_=oracle.contract(oracle.CONTRACT_IEEE), mode=1)
    ok = orc["flags"] == 0
    assert ok.sum() > 0.8 * len(texts)
    assert np.array_equal(_bits(a[ok]), _bits(orc["fitness"][ok]))
    k = len(texts) - 3                                               # the perfect model: M per valid pair, -M / +M for the invalid ones
    nv = N - 2 - 1
    assert a[k] == np.float32(M * nv - M * 3 - 117.0 * 5)


@pytest.mark.parametrize("N,d,power,seed", [(512, 5, 1, 1), (1024, 9, 2, 2), (200, 3, 8, 3), (33, 2, 3, 4)])
def test_std_parity_random_programs(oracle, N, d, power, seed):
    from tests.gpu_util import gpu_eval_fit
    rng = np.random.default_rng(seed)
    X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
    y = (X[:, 0] * X[:, d - 1] + np.sin(X[:, 0])).astype(np.float32)
    texts = _texts(rng, 1200, d, ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP"])
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts)
    a = gpu_eval_fit(g, l, c, X, y, FITS[power], M, 50.0)
    orc = oracle.evaluate_std(g, l, c, X, y, power, M, 50.0)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    # non-vacuity: a floor on the STRICT share of the value-checked individuals (those held to north_star's tolerance
    # unchanged), as tests/test_gpu_parity.py has for the MSE. The Std bound charges |dt| + 1 for every case whose
    # unrounded reward is within dt of a rounding boundary, so it is coarser than the MSE bound: under the oracle alone
    # 75 % / 60 % / 42 % / 58 % of these four colonies are STRICT.
    checked = rep["strict"] + rep["conditioned"]
    print(f"std parity N={N} d={d} power={power}: {parity.describe(rep, a, orc)}; "
          f"bit-equal to the oracle: {int((a == orc['fitness']).sum())} of {len(texts)}")
    assert checked > 0.5 * len(texts)
    assert rep["strict"] >= 0.4 * checked, rep
    assert np.all(a[np.isfinite(a)] == np.round(a[np.isfinite(a)] + 50.0 * l[np.isfinite(a)]) - 50.0 * l[np.isfinite(a)])   # integer scores


def test_std_fast_and_blockwise_paths_bit_identical(oracle):
    from tests.gpu_util import gpu_eval_fit
    rng = np.random.default_rng(9)
    for N, d, power in ((512, 4, 1), (1024, 7, 8), (300, 2, 3)):
        X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
        y = (X[:, 0] - X[:, 1] ** 2).astype(np.float32)
        y[5] = np.inf
        texts = [t for t in _texts(rng, 300, d, ["ADD", "SUB", "MUL", "DIV", "SIN", "EXP", "SQRT"]) if len(t.split()) < 100]
        consts = []
        fast = [asm(t, consts)[0] for t in texts]
        slow = [asm(t + " DUP DEL", consts)[0] for t in texts]
        g, l, c = pack(fast + slow, consts)
        a = gpu_eval_fit(g, l, c, X, y, FITS[power], M, 0.0)
        n = len(texts)
        assert np.array_equal(_bits(a[:n]), _bits(a[n:]))
