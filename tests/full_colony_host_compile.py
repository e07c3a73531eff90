"""The whole colony of a config through the host builds of the device's compilers (test infrastructure; run by hand, minutes).

The CPU suite sends samples; this sends every individual of BASELINE.json's config (default 3: 1,048,576 programs, 38.6 M tokens) through
beagle_debug_walk (both instantiations) and beagle_debug_compile with the plan the real launch uses, and checks: the walk takes every
program; its records are the general compiler's; the depth is the oracle's (static check, one case). DESIGN.md section 4 records the outcome.

    python tests/full_colony_host_compile.py [config] [first P individuals]
"""
import ctypes
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    from paper_2607_06731_b200 import api, colonies
    from oracle import binding
    binding.build()
    number = int(sys.argv[1]) if len(sys.argv) > 1 else 3
    cfg = colonies.CONFIGS[number]
    P = int(sys.argv[2]) if len(sys.argv) > 2 else cfg.P
    t0 = time.time()
    g, l, c = colonies.generate_programs(cfg, P)
    X, y, _ = colonies.make_dataset(cfg)
    depth = binding.evaluate_parallel(g, l, c, X[:1], y[:1], cfg.tax)
    assert not np.any(depth["flags"] & binding.FLAG_MALFORMED)
    plan = (ctypes.c_int32 * 12)()
    assert api.lib().beagle_debug_plan(cfg.N, cfg.d, api.FIT_MSE, 1, 232448, plan) == 0        # the B200's opt-in shared memory
    S_T, k_rcp, k_un = plan[5], plan[4] // (1 if plan[1] else (cfg.N + 511) // 512), plan[6]
    row_bytes = (512 if plan[1] else (cfg.N + 511) // 512 * 512) * 4
    unsafe = sum(1 << j for j in range(cfg.d) if np.any(np.abs(X[:, j]) < 1e-6))
    off = np.concatenate([[0], np.cumsum(l, dtype=np.int64)])
    n_rec = 0
    for p in range(P):
        tok = g[off[p]:off[p + 1]]
        gd, gslow, grec = api.beagle_debug_compile(tok, c, cfg.d, S_T, k_rcp, k_un, row_bytes, unsafe)
        assert gd == depth["depth"][p] and not gslow, p
        for f1 in (False, True):
            taken, d_, used, rec = api.beagle_debug_walk(tok, c, cfg.d, S_T, k_rcp, k_un, row_bytes, unsafe, f1=f1)
            assert taken and d_ == gd and not used and np.array_equal(rec, grec), (p, f1)
        n_rec += len(grec)
        if p % 100000 == 0 and p:
            print(f"  {p} individuals, {time.time() - t0:.0f} s", flush=True)
    print(f"config {number}: {P} individuals, {int(off[P])} tokens -> {n_rec} micro-ops ({n_rec / int(off[P]):.3f} per token), "
          f"plan S_T={S_T} k_rcp={k_rcp} k_un={k_un}: the walk (both instantiations) takes every one, records = the general compiler's, "
          f"depth = the oracle's; {time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()
