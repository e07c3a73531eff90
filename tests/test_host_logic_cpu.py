"""Host logic of the library that needs no device (-m "not gpu"): the plan of tensor memory and shared memory
(`tmem_plan` / `plan_for`) and the two tables that drive the tree compiler's walk (`make_walk2_tabs`,
compile_kernel.inc), through the host-only debug exports of include/beagle.h.

The expectations are restated here from the design (what a command emits given what its operands are: DESIGN.md §7
"k_compile", uop.cuh), not read back from the library's sources.
"""
import ctypes

import numpy as np
import pytest

from paper_2607_06731_b200 import api, colonies

SMEM_OPTIN_B200 = 232448          # 227 KB: sharedMemPerBlockOptin of sm_100
ROWS = 32                         # 512 tensor-memory columns / 16 cases per lane
STAGE_BYTES_MAX = ((512 + 3 + 1) & ~1) * 8      # records of a maximum-length program: every ring must hold one stage

PLAN_FIELDS = "fast split threads xrows rrows slots k_un ring smem off_ys off_un off_ring".split()


def plan(N, d, fit=api.FIT_MSE, fitness_only=True, smem=SMEM_OPTIN_B200):
    out = (ctypes.c_int32 * 12)()
    st = api.lib().beagle_debug_plan(N, d, fit, int(fitness_only), smem, out)
    assert st == api.OK, st
    return dict(zip(PLAN_FIELDS, list(out)))


def test_plan_of_the_five_configs_is_the_documented_one():
    # DESIGN.md §7 "The plan of the 32 TMEM rows": variable rows + reciprocal rows + warps per quarter x slot rows
    c3 = plan(512, 5)
    assert (c3["xrows"], c3["rrows"], c3["threads"], c3["slots"], c3["split"]) == (5, 5, 896, 3, 0)
    c4 = plan(1024, 9)                          # MSE, fitness only: split by passes, 9 + 2 + 7 x 3
    assert (c4["xrows"], c4["rrows"], c4["threads"], c4["slots"], c4["split"]) == (9, 2, 896, 3, 1)
    c4w = plan(1024, 9, fitness_only=False)     # per-case outputs: one launch, 18 + 0 + 7 x 2
    assert (c4w["xrows"], c4w["rrows"], c4w["threads"], c4w["slots"], c4w["split"]) == (18, 0, 896, 2, 0)
    c2 = plan(1024, 3)                          # three slot rows either way: one launch
    assert (c2["split"], c2["slots"], c2["xrows"]) == (0, 3, 6)
    c1 = plan(512, 2)
    assert (c1["threads"], c1["slots"]) == (1024, 3)
    # the correlation fitness is never split and keeps a second array of targets in shared memory
    cc = plan(1024, 9, api.FIT_CORRELATION)
    assert cc["split"] == 0 and cc["xrows"] == 18


def test_plan_invariants_over_all_shapes():
    n_fast = 0
    for N in sorted(set(list(range(1, 1025, 41)) + [511, 512, 513, 1023, 1024])):
        for d in range(1, 33):
            for fit in (api.FIT_MSE, api.FIT_CORRELATION, api.FIT_STD):
                for fo in (False, True):
                    p = plan(N, d, fit, fo)
                    passes = 1 if p["split"] else (N + 511) // 512
                    if not p["fast"]:
                        assert passes * d > ROWS, (N, d, fit, fo, p)      # only a variable block that cannot fit is refused
                        continue
                    n_fast += 1
                    wq = p["threads"] // 128
                    assert p["threads"] in (768, 896, 1024)
                    assert p["xrows"] == passes * d
                    assert p["xrows"] + p["rrows"] + wq * p["slots"] <= ROWS, (N, d, fit, fo, p)
                    assert 0 <= p["slots"] <= 3 and 0 <= p["k_un"] <= d
                    assert p["smem"] <= SMEM_OPTIN_B200
                    assert p["ring"] >= STAGE_BYTES_MAX, (N, d, fit, fo, p)   # run_eval would refuse the call otherwise
                    assert p["off_ys"] < p["off_un"] <= p["off_ring"] < p["smem"]
                    # between y and the unary rows: the padded targets (twice for the correlation fitness: y and the centred y)
                    # and one 64-entry window of the work queue per warp
                    npad = (N + 511) // 512 * 512
                    assert p["off_un"] - p["off_ys"] == 4 * npad * (2 if fit == api.FIT_CORRELATION else 1) + 64 * 16 * (p["threads"] // 32)
                    # bulk copies land on 128-byte boundaries: the rings start on one and are a multiple of it long
                    assert p["off_ring"] % 128 == 0 and p["ring"] % 128 == 0 and p["off_ys"] % 128 == 0
                    assert p["off_ring"] + p["ring"] * (p["threads"] // 32) <= p["smem"]
                    assert p["split"] == 0 or (fit == api.FIT_MSE and fo and N > 512)
    assert n_fast > 4000


def test_split_makes_wide_case_matrices_fit():
    # d > 16 at more than 512 cases: two passes of rows do not fit 32, one pass per launch does (MSE, fitness only)
    assert plan(1024, 17)["fast"] == 1 and plan(1024, 32)["fast"] == 1
    assert plan(1024, 17, fitness_only=False)["fast"] == 0
    assert plan(1024, 17, api.FIT_CORRELATION)["fast"] == 0
    assert plan(512, 32, api.FIT_STD)["fast"] == 1


def test_plan_rejects_bad_arguments():
    out = (ctypes.c_int32 * 12)()
    f = api.lib().beagle_debug_plan
    assert f(0, 1, 0, 1, SMEM_OPTIN_B200, out) == api.ERR_INVALID_ARG
    assert f(512, 33, 0, 1, SMEM_OPTIN_B200, out) == api.ERR_INVALID_ARG
    assert f(512, 5, 99, 1, SMEM_OPTIN_B200, out) == api.ERR_INVALID_ARG
    assert f(512, 5, 0, 1, SMEM_OPTIN_B200, None) == api.ERR_INVALID_ARG


# ---- the walk's tables ---------------------------------------------------------------------------------------------
# bit fields as DESIGN.md §7 / compile_kernel.inc name them (restated)
O_B, O_A, C_B, C_A = 1 << 8, 2 << 8, 1 << 10, 2 << 10
PUSH, SLOT, DBL, F_A = 1 << 12, 1 << 15, 1 << 16, 1 << 17
DIVC, DIVV, UNV = 1 << 20, 1 << 21, 1 << 22


def dc_of(e):
    v = (e >> 13) & 3
    return v - 4 if v & 2 else v


def nrec_of(e):
    return (e >> 18) & 3


@pytest.fixture(scope="module")
def tables():
    lut = (ctypes.c_uint32 * 160)()
    tok = (ctypes.c_uint32 * 130)()
    api.lib().beagle_debug_walk_tables(lut, tok)
    return np.array(lut, dtype=np.uint32), np.array(tok, dtype=np.uint32).reshape(65, 2)


def test_decision_table_binary_commands(tables):
    lut, _ = tables
    handlers = {}
    for j in range(4):                                    # ADD SUB MUL DIV: rows 6..9
        for key in range(16):
            ra, rb, xa, xb = (key >> 3) & 1, (key >> 2) & 1, (key >> 1) & 1, key & 1
            e = int(lut[(6 + j) * 16 + key])
            h = e & 0xFF
            assert 0 < h < 102
            if ra and rb:                                 # both computed: acc (b) with the slot below it (a)
                assert e & SLOT and not e & PUSH and dc_of(e) == -1 and nrec_of(e) == 1
                assert not e & (O_A | O_B | C_A | C_B | DBL)
                kind = "ss"
            elif ra:                                      # a computed, b a terminal: its value is the operand
                assert e & O_B and not e & O_A and dc_of(e) == 0 and nrec_of(e) == 1 and not e & (PUSH | SLOT | DBL | C_A | C_B)
                kind = "rx" if xb else "rc"
            elif rb:                                      # b computed, a a terminal: the reversed handlers
                assert e & O_A and not e & O_B and dc_of(e) == 0 and nrec_of(e) == 1 and not e & (PUSH | SLOT | DBL | C_A | C_B)
                kind = "xr" if xa else "cr"
            elif xa or xb:                                # a fresh value from a variable column and the other terminal
                assert e & PUSH and dc_of(e) == 1 and nrec_of(e) == 1 and not e & (SLOT | DBL)
                if xa:
                    assert e & C_A and e & O_B            # first operand: a's column; second: b's value
                else:
                    assert e & C_B and e & O_A            # a is a constant: b's column comes first, reversed handler
                kind = "xx" if xa and xb else ("xc" if xa else "cx")
            else:                                         # two constants: the first becomes acc, then acc op c
                assert e & DBL and e & F_A and e & O_B and dc_of(e) == 1 and nrec_of(e) == 2 and not e & (SLOT | PUSH)
                kind = "cc"
            # the division rewrites: by a variable (reciprocal row, if safe), by a constant (multiplication by rcp)
            assert bool(e & DIVV) == (j == 3 and xb and not rb and (ra or xa))
            assert bool(e & DIVC) == (j == 3 and not xb and not rb)
            assert not e & UNV
            handlers[(j, kind)] = h
    # a handler serves one command, except that dividing by a constant is multiplying (MULC with DIVC set) ...
    for kind in ("ss", "rx", "xx"):
        assert len({handlers[(j, kind)] for j in range(4)}) == 4
    for kind in ("rc", "xc", "cc"):
        assert handlers[(3, kind)] == handlers[(2, kind)]
        assert len({handlers[(j, kind)] for j in range(3)}) == 3
    # ... and that the commutative commands need no reversed handler
    for j in (0, 2):
        assert handlers[(j, "xr")] == handlers[(j, "rx")] and handlers[(j, "cr")] == handlers[(j, "rc")]
    for j in (1, 3):
        assert handlers[(j, "xr")] != handlers[(j, "rx")] and handlers[(j, "cr")] != handlers[(j, "rc")]


def test_decision_table_unary_commands(tables):
    lut, _ = tables
    hs = set()
    for kk in range(5):                                   # SIN COS LOG SQRT EXP: rows 1..5
        for key in range(16):
            rb, xb = (key >> 2) & 1, key & 1
            e = int(lut[(1 + kk) * 16 + key])
            if rb:                                        # f(acc)
                assert nrec_of(e) == 1 and dc_of(e) == 0 and not e & (PUSH | UNV | DBL | SLOT)
                hs.add(e & 0xFF)
            elif xb:                                      # f(x_j): the staged row
                assert e & UNV and e & PUSH and e & C_B and nrec_of(e) == 1 and dc_of(e) == 1
            else:                                         # f(c): load the constant, then f(acc)
                assert e & DBL and not e & F_A and nrec_of(e) == 2 and dc_of(e) == 1 and not e & UNV
            assert not e & (DIVC | DIVV | O_A | O_B)
    assert len(hs) == 5
    assert not lut[:16].any()                             # row 0: nothing (terminals, padding, violations)


def test_token_table(tables):
    _, tok = tables

    def px(y):
        d = (y >> 12) & 3
        return dict(kind=(y >> 2) & 1, or1=(y >> 3) & 1, delta=d - 4 if d & 2 else d, sh=(y >> 14) & 3,
                    need=(y >> 16) & 63, lim=(y >> 22) & 63)

    ops = colonies.OP
    seen_rows = set()
    for name, cls in (("CONST", "t"), ("LOAD", "t"), ("ADD", "b"), ("SUB", "b"), ("MUL", "b"), ("DIV", "b"),
                      ("SIN", "u"), ("COS", "u"), ("LOG", "u"), ("SQRT", "u"), ("EXP", "u")):
        x, y = int(tok[ops[name]][0]), int(tok[ops[name]][1])
        f = px(y)
        row = (x >> 16) // 64
        if cls == "t":
            assert (f["delta"], f["sh"], f["need"], f["lim"], f["or1"]) == (1, 0, 0, 31, 0) and row == 0
            assert f["kind"] == (1 if name == "LOAD" else 0)
        elif cls == "u":
            assert (f["delta"], f["sh"], f["need"], f["or1"]) == (0, 1, 1, 1) and 1 <= row <= 5
            seen_rows.add(row)
        else:
            assert (f["delta"], f["sh"], f["need"], f["or1"]) == (-1, 2, 2, 1) and 6 <= row <= 9
            seen_rows.add(row)
    assert seen_rows == set(range(1, 10))
    # everything else is not a command of the walk (need 63 can never be met), except the padding entry, which does nothing
    known = {ops[n] for n in ("CONST", "LOAD", "ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP")}
    for i in range(64):
        if i not in known:
            assert px(int(tok[i][1]))["need"] == 63 and int(tok[i][0]) == 0
    pad = px(int(tok[64][1]))
    assert (pad["delta"], pad["sh"], pad["need"], pad["lim"], pad["or1"], pad["kind"]) == (0, 1, 0, 63, 0, 0)


# ---- a8: how a budget is cut into staging buffers and a colony into chunks -------------------------------------------
def chunk_plan(lengths, budget):
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    max_ends = len(lengths) + 1
    ends = np.zeros(max_ends, dtype=np.int64)
    n, K, nbytes = ctypes.c_int64(0), ctypes.c_int32(0), ctypes.c_int64(0)
    st = api.lib().beagle_debug_chunk_plan(lengths.ctypes.data, len(lengths), budget, ends.ctypes.data, max_ends,
                                           ctypes.byref(n), ctypes.byref(K), ctypes.byref(nbytes))
    return st, ends[:n.value].copy(), K.value, nbytes.value


def check_chunks(lengths, budget):
    """The properties a chunking must have, whatever the algorithm: contiguous, whole individuals, every chunk fits its
    buffer, and greedy (the next individual would not have fitted)."""
    st, ends, K, nbytes = chunk_plan(lengths, budget)
    assert st == api.OK
    assert 2 <= K <= 8 and nbytes % 256 == 0 and K * nbytes <= budget
    lengths = np.asarray(lengths, dtype=np.int64)
    tok = np.where((lengths >= 1) & (lengths <= 512), lengths, 0)
    assert len(ends) >= 1 and ends[-1] == len(lengths) and (np.diff(np.concatenate(([0], ends))) > 0).all()
    p0 = 0
    for p1 in ends:
        np_, nt = p1 - p0, int(tok[p0:p1].sum())
        # the buffer holds the chunk's lengths (padded to a multiple of four) and then its tokens
        assert 4 * (((np_ + 3) & ~3) + nt) <= nbytes
        if p1 < len(lengths):
            assert 4 * (np_ + 1 + nt + int(tok[p1]) + 3) > nbytes          # greedy: one more would not fit
        p0 = p1
    return len(ends), K, nbytes


def test_chunk_plan_properties_on_random_colonies():
    rng = np.random.default_rng(20260705)
    for budget in (4608, 10_000, 64 << 10, 1 << 20, 5 << 20):
        for _ in range(3):
            P = int(rng.integers(1, 60_000))
            lengths = rng.integers(1, 513, size=P)
            lengths[rng.random(P) < 0.01] = 0                    # out-of-range lengths: an entry without tokens
            lengths[rng.random(P) < 0.01] = 700
            check_chunks(lengths, budget)
    # exactly one maximum-length individual per buffer at the smallest budget the call accepts
    n, K, nbytes = check_chunks(np.full(7, 512), 4608)
    assert (n, K) == (7, 2)


def test_chunk_plan_block_scan_with_out_of_range_lengths():
    # buffers large enough for the planner's fast path (whole blocks of 4096 lengths at a time), on a colony with lengths outside
    # 1..512 in it: they take a word each and no tokens, in the fast path as in the slow one
    rng = np.random.default_rng(4096)
    P = 150_000
    lengths = rng.integers(1, 513, size=P)
    lengths[rng.random(P) < 0.02] = 0
    lengths[rng.random(P) < 0.02] = 700
    lengths[rng.random(P) < 0.01] = -5
    n, K, nbytes = check_chunks(lengths, 64 << 20)
    assert K == 2 and n >= 2 and nbytes // 4 > 3 * 4096 * 257


def test_chunk_plan_buffers_follow_the_budget():
    ones = np.ones(10, dtype=np.int32)
    MiB = 1 << 20
    for budget, K in ((64 * MiB, 2), (96 * MiB, 3), (160 * MiB, 5), (256 * MiB, 8), (1024 * MiB, 8)):
        st, _, k, nbytes = chunk_plan(ones, budget)
        assert st == api.OK and k == K and nbytes == (budget // K) & ~255
    api.beagle_set_chunk_target(8 * MiB)
    try:
        assert chunk_plan(ones, 24 * MiB)[2] == 3
    finally:
        api.beagle_set_chunk_target(0)
    assert chunk_plan(ones, 24 * MiB)[2] == 2
    assert chunk_plan(ones, 4607)[0] == api.ERR_INVALID_ARG


def test_chunk_plan_of_config5_is_ten_chunks_over_eight_buffers():
    # BASELINE.json configs[4]: P = 4,194,304, lengths up to 512, a budget of 1 GiB: the chunking the full-size GPU
    # test and bench.py --config 5 run (more chunks than buffers: buffers are reused)
    cfg = colonies.CONFIGS[5]
    _, lengths, _ = colonies.generate_programs(cfg, cfg.P, seed_offset=0)
    n, K, nbytes = check_chunks(lengths, cfg.budget_bytes)
    assert K == 8 and n == 10
