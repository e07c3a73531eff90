"""Oracle of the Monte-Carlo ranking (Table 2). TEST INFRASTRUCTURE: only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this; the product never does.

The paper: "Beagle takes a random sample of 100 individuals and uses those 100 individuals to estimate the population
percentiles. Through one pass of the population then, individuals are assigned to their specific percentile and are
given rank proportional breeding rights", with the expected number of children per percentile group of Table 2.

Written as that definition, nothing else. The random draw is an INPUT (the sampled indices), so the step is
deterministic: for every individual, count the sampled individuals that are strictly worse; with n_sample samples the
individual is at or above the percentile 100 * count / n_sample, and its group is the decile of that percentile,
Table 2's rows from the bottom: group g means "percentile >= 10 g", g = 0 .. 9.

Readings (R24): "worse" is by fitness in the direction of the objective (lower MSE is better, higher
correlation score is better); a NaN fitness (an invalid individual) is worse than every number and ties with other
NaNs; ties are not "strictly worse", so equal fitnesses share the lower group.

Pins (tests/test_oracle_pins.py P20): Table 2 retyped from the paper and its mean of exactly one child per individual;
a population of distinct fitnesses with an evenly spread sample lands in deciles of its true rank; direction; NaN; ties;
brute force against a sort-based restatement on small random populations.
"""
import numpy as np

# Table 2, group 0 = "percentile >= 0" ... group 9 = "percentile >= 90"
EXPECTED_CHILDREN = np.array([0.01, 0.03, 0.06, 0.15, 0.25, 0.5, 1.0, 1.5, 2.5, 4.0], np.float64)


def goodness(fitness, maximise):
    """Higher is better; NaN is worst (R24)."""
    f = np.asarray(fitness, np.float64)
    g = f if maximise else -f
    return np.where(np.isnan(f), -np.inf, g)


def rank_deciles(fitness, sample_idx, maximise):
    """fitness float[P], sample_idx int[n_sample] (indices into fitness), maximise bool.
    Returns (decile uint8[P], hist int64[10], expected_children float64[P])."""
    g = goodness(fitness, maximise)
    s = g[np.asarray(sample_idx, np.int64)]
    n = len(s)
    decile = np.empty(len(g), np.uint8)
    for i in range(len(g)):                       # one pass of the population
        worse = 0
        for j in range(n):
            if s[j] < g[i]:
                worse += 1
        decile[i] = min(9, (10 * worse) // n)     # percentile 100 * worse / n, in steps of ten
    hist = np.bincount(decile, minlength=10).astype(np.int64)
    return decile, hist, EXPECTED_CHILDREN[decile]
