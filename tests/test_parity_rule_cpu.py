"""The comparator every GPU-vs-oracle test goes through (tests/parity.py, the three-class rule of DESIGN.md §4) catches what it
has to catch: planted violations of each kind are reported, and nothing else is. CPU only."""
import numpy as np

from tests import parity

QNAN = np.array([0x7FC00000], np.uint32).view(np.float32)[0]


def orc(fitness, bound, flags):
    return dict(fitness=np.array(fitness, np.float32), bound=np.array(bound, np.float64), flags=np.array(flags, np.int32))


def test_strict_individuals_are_held_to_north_stars_tolerance():
    # E far below the tolerance: STRICT. rtol 1e-4 on |oracle|, atol 1e-6
    o = orc([100.0, 100.0, 100.0, 1e-9, 1e-9, -50.0], [1e-7] * 3 + [1e-12] * 2 + [1e-7], [0] * 6)
    gpu = np.array([100.0 + 0.009, 100.0 + 0.011, 100.0 - 0.011, 1e-9 + 0.9e-6, 1e-9 + 1.1e-6, -50.0 - 0.0051], np.float32)
    rep = parity.compare(gpu, o)
    assert rep["strict"] == 6 and rep["conditioned"] == 0
    assert list(rep["bad"]) == [1, 2, 4, 5] and rep["strict_bad"] == 4 and rep["class_bad"] == 0


def test_conditioned_individuals_get_the_tolerance_plus_twice_their_bound():
    # 4 E > tol: CONDITIONED; allowed |diff| <= tol + 2 E
    o = orc([10.0, 10.0, 10.0], [0.01, 0.01, 0.0003], [0, 0, 0])          # tol = 1e-3
    gpu = np.array([10.0 + 0.0205, 10.0 + 0.0215, 10.0 + 0.0017], np.float32)   # limits: 0.021, 0.021, 0.0016
    rep = parity.compare(gpu, o)
    assert rep["strict"] == 0 and rep["conditioned"] == 3
    assert list(rep["bad"]) == [1, 2] and rep["cond_bad"] == 2
    # the boundary between the classes: 4 E <= tol is STRICT
    o2 = orc([10.0, 10.0], [0.00025, 0.00026], [0, 0])
    rep2 = parity.compare(np.array([10.0, 10.0], np.float32), o2)
    assert (rep2["strict"], rep2["conditioned"]) == (1, 1)


def test_class_parity_is_exact_and_malformed_is_the_canonical_nan():
    inf, nan = np.inf, np.nan
    o = orc([inf, inf, nan, nan, 1.0, -inf, QNAN, QNAN, QNAN], [0] * 9, [0, 0, 0, 0, 0, 0, 1, 1, 1])
    other_nan = np.array([0x7FC00001], np.uint32).view(np.float32)[0]
    gpu = np.array([inf, 3e38, nan, inf, nan, inf, QNAN, other_nan, 1.0], np.float32)
    gpu[7] = other_nan
    rep = parity.compare(gpu, o)
    # 1: finite where the oracle overflows; 3: inf for NaN; 4: NaN for finite; 5: +inf for -inf; 7: a NaN that is not the canonical
    # one; 8: a number for a malformed program
    assert list(rep["bad"]) == [1, 3, 4, 5, 7, 8]
    assert rep["class_bad"] == 4 and rep["malformed"] == 3 and rep["invalid"] == 5
    # any NaN payload is a NaN for class parity (only malformed programs promise the bit pattern)
    rep2 = parity.compare(np.array([other_nan], np.float32), orc([nan], [0.0], [0]))
    assert len(rep2["bad"]) == 0


def test_unstable_individuals_are_exempt_and_counted():
    o = orc([1.0, 1.0, 1.0, 1.0], [1e-9] * 4, [2, 4, 6, 0])
    gpu = np.array([5.0, np.inf, np.nan, 1.0], np.float32)
    rep = parity.compare(gpu, o)
    assert rep["exempt"] == 3 and len(rep["bad"]) == 0 and rep["strict"] == 1
    # a malformed flag wins over an unstable one: the canonical NaN is still demanded
    rep2 = parity.compare(np.array([1.0], np.float32), orc([QNAN], [0.0], [1 | 2]))
    assert list(rep2["bad"]) == [0]


def test_report_counts_add_up():
    rng = np.random.default_rng(5)
    P = 1000
    fit = rng.normal(size=P).astype(np.float32)
    fit[rng.random(P) < 0.05] = np.inf
    fit[rng.random(P) < 0.05] = np.nan
    flags = rng.choice([0, 0, 0, 0, 1, 2, 4], size=P).astype(np.int32)
    fit[flags == 1] = QNAN
    bound = 10.0 ** rng.uniform(-12, -2, P)
    o = orc(fit, bound, flags)
    rep = parity.compare(fit.copy(), o)                     # the oracle against itself: nothing to report
    assert len(rep["bad"]) == 0
    assert rep["strict"] + rep["conditioned"] + rep["invalid"] + rep["exempt"] + rep["malformed"] == P
    assert "strict=" in parity.describe(rep, fit, o)
