"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these retypes the oracle's formulas: each compares it with a printed value, a closed form,
an invariant, a special case that reduces to numpy, or an independent brute-force evaluator.
All CPU (-m "not gpu").
"""
import itertools
import math
import os

import numpy as np
import pytest

from paper_2607_06731_b200 import colonies as C
from tests.util import asm, pack, symbolic

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_genomes.txt")
QNAN_BITS = 0x7FC00000


def _golden():
    rows = []
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        cite, n, text = [s.strip() for s in line.split("|")]
        rows.append((cite, int(n), text))
    return rows


def _gcl_to_asm(text):
    """GCL text of the paper ('LOAD b:1; CONST 0.5; MUL;') -> our test assembler text."""
    out = []
    for cmd in [c.strip() for c in text.split(";") if c.strip()]:
        parts = cmd.split()
        if parts[0] == "LOAD":
            out.append("x" + parts[1].split(":")[1])
        elif parts[0] == "CONST":
            out.append(parts[1])
        else:
            out.append({"LN": "LOG"}.get(parts[0], parts[0]))
    return " ".join(out)


def ev(oracle, progs, consts, X, y, tax=0.0, **kw):
    g, l, c = pack(progs, consts)
    return oracle.evaluate(g, l, c if len(c) else np.zeros(1, np.float32), X, y, tax, **kw)


# ---- P1: printed lengths ------------------------------------------------------------------------
def test_P1_printed_lengths_are_token_counts():
    rows = _golden()
    assert [n for _, n, _ in rows] == [12, 12, 24, 25]
    for cite, n, text in rows:
        cmds = [c for c in text.split(";") if c.strip()]
        assert len(cmds) == n, cite  # PAPER.md:314 "genome length (i.e., the number of GCL commands)"


def test_P1_oracle_taxes_every_token(oracle):
    # fitness - MSE == tax * L with L the printed length (genome of P:157, hot-path ops only)
    cite, n, text = _golden()[0]
    consts = []
    prog, c = asm(_gcl_to_asm(text), consts)
    rng = np.random.default_rng(1)
    X = rng.uniform(1, 3, (64, 3)).astype(np.float32)
    y = np.zeros(64, np.float32)
    f0 = ev(oracle, [prog], c, X, y, tax=0.0)["fitness"][0]
    f1 = ev(oracle, [prog], c, X, y, tax=0.5)["fitness"][0]
    assert f1 - f0 == pytest.approx(0.5 * n, rel=1e-6)


# ---- P2: closed forms of the paper's genomes ----------------------------------------------------
def test_P2_fig2_genome_closed_form(oracle):
    # P:157 = (sqrt(b*b) - b)/a*0.5 - 0.01603 = (|b|-b)/(2a) - 0.01603
    _, _, text = _golden()[0]
    prog, c = asm(_gcl_to_asm(text))
    rng = np.random.default_rng(2)
    X = rng.uniform(-4, 4, (256, 3)).astype(np.float32)
    X[np.abs(X[:, 0]) < 0.1, 0] = 1.0
    a, b = X[:, 0].astype(np.float64), X[:, 1].astype(np.float64)
    want = (np.abs(b) - b) / (2 * a) + np.float64(np.float32(-0.01603))
    r = ev(oracle, [prog], c, X, np.zeros(256, np.float32), want_outputs=True)
    np.testing.assert_allclose(r["outputs"][0], want, rtol=1e-12, atol=1e-12)
    # exactly -0.01603 for b >= 0
    pos = b >= 0
    assert np.all(r["outputs"][0][pos] == np.float64(np.float32(-0.01603)))


def test_P2_quadratic_formula_operand_order(oracle):
    # the P:316 genome with DUP/DEL expanded by hand: (sqrt(b^2-4ac)-b)/a*0.5
    prog, c = asm("x1 x1 MUL x0 x0 ADD x0 x0 ADD ADD x2 MUL SUB SQRT x1 SUB x0 DIV 0.5 MUL")
    rng = np.random.default_rng(3)
    X = np.empty((512, 3), np.float32)
    X[:, 0] = rng.uniform(0.5, 2, 512) * rng.choice([-1, 1], 512)
    X[:, 1] = rng.uniform(4, 8, 512)
    X[:, 2] = rng.uniform(-1, 1, 512)
    a, b, cc = (X[:, j].astype(np.float64) for j in range(3))
    assert np.all(b * b >= 4 * a * cc)
    root = (np.sqrt(b * b - 4 * a * cc) - b) / (2 * a)
    y = root.astype(np.float32)
    r = ev(oracle, [prog], c, X, y, want_outputs=True)
    np.testing.assert_allclose(r["outputs"][0], root, rtol=1e-13)
    mse_want = np.mean((root - y.astype(np.float64)) ** 2)
    assert r["fitness"][0] == pytest.approx(mse_want, rel=1e-6, abs=1e-25)
    # it IS a root: a r^2 + b r + c ~ 0 (pins SUB/DIV order independently of the formula above)
    o = r["outputs"][0]
    assert np.max(np.abs(a * o * o + b * o + cc)) < 1e-9


# ---- P3: north_star's example --------------------------------------------------------------------
def test_P3_x0_squared_is_exact(oracle):
    X = (np.arange(-256, 256, dtype=np.float64)[:, None] / 2048.0).astype(np.float32)  # <= 12 bits
    y = (X[:, 0].astype(np.float64) ** 2).astype(np.float32)
    assert np.all(y.astype(np.float64) == X[:, 0].astype(np.float64) ** 2)
    prog, c = asm("x0 x0 MUL")
    tax = np.float32(0.001)
    f = ev(oracle, [prog], c, X, y, tax=tax)["fitness"][0]
    assert f == np.float32(np.float64(tax) * 3)      # MSE exactly 0, fitness = (float)(tax*3)
    assert f == tax * np.float32(3)                  # same bits as the fp32 product


# ---- P4: single-terminal programs reduce to numpy -----------------------------------------------
def test_P4_terminals_reduce_to_numpy(oracle):
    rng = np.random.default_rng(4)
    X = rng.normal(size=(300, 4)).astype(np.float32)
    y = rng.normal(size=300).astype(np.float32)
    y64 = y.astype(np.float64)
    consts = []
    progs = [asm("1.75", consts, 0)[0]] + [asm(f"x{j}")[0] for j in range(4)]
    r = ev(oracle, progs, consts, X, y)
    assert r["fitness"][0] == pytest.approx((1.75 - y64.mean()) ** 2 + y64.var(), rel=1e-6)
    for j in range(4):
        assert r["fitness"][1 + j] == pytest.approx(np.mean((X[:, j].astype(np.float64) - y64) ** 2), rel=1e-6)
    assert list(r["depth"]) == [1] * 5


# ---- P5: identity insertion ----------------------------------------------------------------------
def test_P5_identity_insertion(oracle):
    col = C.make_colony(1, P=64)
    off = np.concatenate([[0], np.cumsum(col.lengths)])
    nC = len(col.consts)
    consts = list(col.consts) + [np.float32(0.0), np.float32(1.0)]
    zero, one = C.token(C.OP["CONST"], nC), C.token(C.OP["CONST"], nC + 1)
    ADD, MUL, DIV = (C.token(C.OP[k]) for k in ("ADD", "MUL", "DIV"))
    base = [col.genomes[off[p]:off[p + 1]] for p in range(64)]
    variants = {
        "post0add": [np.concatenate([b, [zero, ADD]]) for b in base],
        "post1mul": [np.concatenate([b, [one, MUL]]) for b in base],
        "post1div": [np.concatenate([b, [one, DIV]]) for b in base],
        "pre0add": [np.concatenate([[zero], b, [ADD]]) for b in base],
    }
    tax = 0.001
    r0 = ev(oracle, base, consts, col.X, col.y, tax=tax, want_outputs=True)
    m0 = ev(oracle, base, consts, col.X, col.y, tax=0.0)["fitness"]
    for name, progs in variants.items():
        r1 = ev(oracle, progs, consts, col.X, col.y, tax=tax, want_outputs=True)
        a, b = r0["outputs"], r1["outputs"]
        assert np.array_equal(np.isnan(a), np.isnan(b)), name
        ok = ~np.isnan(a)
        assert np.array_equal(a[ok], b[ok]), name              # bitwise (x+0, x*1, x/1 exact)
        m1 = ev(oracle, progs, consts, col.X, col.y, tax=0.0)["fitness"]
        np.testing.assert_array_equal(m0, m1)
        fin = np.isfinite(r0["fitness"])
        diff = r1["fitness"][fin].astype(np.float64) - r0["fitness"][fin]
        assert np.all(np.abs(diff - 2 * tax) <= 2e-7 * np.maximum(1, np.abs(r0["fitness"][fin])))


# ---- P6: commutativity, antisymmetry -> stack order ------------------------------------------------
def test_P6_commutativity_and_sub_antisymmetry(oracle):
    rng = np.random.default_rng(6)
    X = rng.uniform(-2, 2, (128, 2)).astype(np.float32)
    y = rng.normal(size=128).astype(np.float32)
    A, B = "x0 1.5 MUL SIN", "x1 x0 DIV 0.25 ADD"
    consts = []
    progs = [asm(f"{A} {B} ADD", consts)[0], asm(f"{B} {A} ADD", consts)[0],
             asm(f"{A} {B} MUL", consts)[0], asm(f"{B} {A} MUL", consts)[0],
             asm(f"{A} {B} SUB", consts)[0], asm(f"{B} {A} SUB", consts)[0],
             asm(f"{A} {B} DIV", consts)[0], asm(f"{B} {A} DIV", consts)[0]]
    r = ev(oracle, progs, consts, X, y, want_outputs=True)["outputs"]
    assert np.array_equal(r[0], r[1]) and np.array_equal(r[2], r[3])
    assert np.array_equal(r[4], -r[5]) and not np.array_equal(r[4], r[5])
    assert not np.allclose(r[6], r[7])
    # SUB is second-top minus top: "3 1 SUB" = 2; DIV second-top / top: "3 2 DIV" = 1.5
    r = ev(oracle, [asm("3 1 SUB")[0]], asm("3 1 SUB")[1], X, y, want_outputs=True)["outputs"]
    assert np.all(r == 2.0)
    r = ev(oracle, [asm("3 2 DIV")[0]], asm("3 2 DIV")[1], X, y, want_outputs=True)["outputs"]
    assert np.all(r == 1.5)


# ---- P7: protected operators at their edges (D2) ----------------------------------------
INF, NAN = math.inf, math.nan
EPSF = float(np.float32(1e-6))
E80 = math.exp(80.0)
EDGES = [
    ("x0 x1 DIV", (3.0, 0.0), 1.0), ("x0 x1 DIV", (0.0, 0.0), 1.0), ("x0 x1 DIV", (NAN, 0.0), 1.0),
    ("x0 x1 DIV", (1.0, INF), 0.0), ("x0 x1 DIV", (1.0, -INF), -0.0), ("x0 x1 DIV", (INF, INF), NAN),
    ("x0 x1 DIV", (2.0, EPSF), 2.0 / EPSF),                      # strict '<': |b| == EPS divides
    ("x0 x1 DIV", (2.0, float(np.nextafter(np.float32(1e-6), np.float32(0)))), 1.0),
    ("x0 x1 DIV", (2.0, -0.5e-6), 1.0), ("x0 x1 DIV", (2.0, NAN), NAN), ("x0 x1 DIV", (INF, 2.0), INF),
    ("x0 x1 DIV", (-INF, 2.0), -INF), ("x0 x1 DIV", (6.0, -3.0), -2.0),
    ("x0 LOG", (0.0,), 0.0), ("x0 LOG", (-math.e,), math.log(float(np.float32(math.e)))),
    ("x0 LOG", (INF,), INF), ("x0 LOG", (-INF,), INF), ("x0 LOG", (NAN,), NAN),
    ("x0 LOG", (0.5e-6,), 0.0), ("x0 LOG", (EPSF,), math.log(EPSF)), ("x0 LOG", (1.0,), 0.0),
    ("x0 SQRT", (-4.0,), 2.0), ("x0 SQRT", (0.0,), 0.0), ("x0 SQRT", (-0.0,), 0.0),
    ("x0 SQRT", (INF,), INF), ("x0 SQRT", (-INF,), INF), ("x0 SQRT", (NAN,), NAN),
    ("x0 SQRT", (1e-45,), math.sqrt(float(np.float32(1e-45)))),
    ("x0 EXP", (81.0,), E80), ("x0 EXP", (INF,), E80), ("x0 EXP", (80.0,), E80),
    ("x0 EXP", (-INF,), 0.0), ("x0 EXP", (NAN,), NAN), ("x0 EXP", (0.0,), 1.0),
    ("x0 EXP", (3.0e38,), E80), ("x0 EXP", (-200.0,), math.exp(-200.0)),
    ("x0 SIN", (INF,), NAN), ("x0 SIN", (-INF,), NAN), ("x0 COS", (INF,), NAN), ("x0 SIN", (0.0,), 0.0),
    ("x0 COS", (0.0,), 1.0), ("x0 SIN", (NAN,), NAN),
    ("x0 x1 ADD", (3.0e38, 3.0e38), INF), ("x0 x1 SUB", (INF, INF), NAN), ("x0 x1 MUL", (INF, 0.0), NAN),
    ("x0 x1 MUL", (3.0e38, -2.0), -INF), ("x0 x1 ADD", (3.4028234663852886e38, 0.0), 3.4028234663852886e38),
    ("x0 x1 SUB", (1.0, 2.5), -1.5),
]


@pytest.mark.parametrize("text,xs,want", EDGES)
def test_P7_edge_table(oracle, text, xs, want):
    X = np.array([list(xs) + [0.0] * (2 - len(xs))], np.float32)
    prog, c = asm(text)
    out = ev(oracle, [prog], c, X, np.zeros(1, np.float32), want_outputs=True)["outputs"][0, 0]
    if isinstance(want, float) and math.isnan(want):
        assert math.isnan(out)
    else:
        assert out == pytest.approx(want, rel=1e-15, abs=0.0)
        if want == 0.0:
            assert out == 0.0


def test_P7_signed_zero_constant_survives(oracle):
    # "CONST -0" is printed in the paper; -0 + b must give b, and 1/(-0 protected) = 1
    X = np.array([[2.0, 0.0]], np.float32)
    prog, c = asm("-0.0 x0 ADD")
    assert np.signbit(c[0])
    assert ev(oracle, [prog], c, X, np.zeros(1, np.float32), want_outputs=True)["outputs"][0, 0] == 2.0


# ---- P8: brute force against the independent recursive evaluator ----------------------------------
def test_P8_bruteforce_up_to_3_tokens(oracle):
    from oracle import infix_check
    consts = np.array([0.5, -2.25], np.float32)
    X = np.array([[0.0, 1.0], [-1.5, 2.0e-7], [3.0e19, -4.0], [88.0, 1.0e30]], np.float32)
    y = np.array([0.25, -1.0, 2.0, 0.0], np.float32)
    terms = [C.token(C.OP["LOAD"], 0), C.token(C.OP["LOAD"], 1), C.token(C.OP["CONST"], 0), C.token(C.OP["CONST"], 1)]
    un = [C.token(C.OP[k]) for k in ("SIN", "COS", "LOG", "SQRT", "EXP")]
    bn = [C.token(C.OP[k]) for k in ("ADD", "SUB", "MUL", "DIV")]
    progs = [[t] for t in terms]
    progs += [[t, u] for t in terms for u in un]
    progs += [[t, u1, u2] for t in terms for u1 in un for u2 in un]
    progs += [[t1, t2, b] for t1 in terms for t2 in terms for b in bn]
    assert len(progs) == 4 + 20 + 100 + 64  # = 188
    arrs = [np.array(p, np.int32) for p in progs]
    tax = 0.001
    r = ev(oracle, arrs, consts, X, y, tax=tax)
    n_nonfinite = 0
    for p, a in enumerate(arrs):
        want = infix_check.fitness(symbolic(a, consts), X, y, np.float32(tax))
        got = float(r["fitness"][p])
        want32 = float(np.float32(want)) if not math.isnan(want) else want
        if math.isnan(want32):
            assert math.isnan(got), (p, symbolic(a, consts))
            n_nonfinite += 1
        elif math.isinf(want32):
            assert got == want32, (p, symbolic(a, consts))
            n_nonfinite += 1
        else:
            assert got == pytest.approx(want32, rel=2e-7), (p, symbolic(a, consts))
    assert n_nonfinite > 10  # the cases were picked so that overflow/NaN paths are exercised


# ---- P9: power-of-two scaling ----------------------------------------------------------------------
@pytest.mark.parametrize("mode", [0, 1])
def test_P9_power_of_two_scaling(oracle, mode):
    col = C.make_colony(1, P=128)
    off = np.concatenate([[0], np.cumsum(col.lengths)])
    nC = len(col.consts)
    consts = list(col.consts) + [np.float32(2.0)]
    two, MUL = C.token(C.OP["CONST"], nC), C.token(C.OP["MUL"])
    base = [col.genomes[off[p]:off[p + 1]] for p in range(128)]
    scaled = [np.concatenate([b, [two, MUL]]) for b in base]
    f0 = ev(oracle, base, consts, col.X, col.y, tax=0.0, mode=mode)["fitness"].astype(np.float64)
    f1 = ev(oracle, scaled, consts, col.X, 2 * col.y, tax=0.0, mode=mode)["fitness"].astype(np.float64)
    fin = np.isfinite(f0) & np.isfinite(f1) & (f0 > 1e-30) & (f1 < 1e37)
    assert fin.sum() > 100
    assert np.array_equal(4.0 * f0[fin], f1[fin])   # exact, fp64 carrier and fp32 mirror alike


# ---- P10: overflow semantics (D4-D6) ---------------------------------------------------------------
def test_P10_overflow_semantics(oracle):
    X = np.ones((8, 1), np.float32)
    y0 = np.zeros(8, np.float32)
    consts = []
    progs = [asm("100 EXP 100 EXP MUL", consts)[0],                       # e80*e80 -> +inf
             asm("100 EXP 100 EXP MUL 100 EXP 100 EXP MUL SUB", consts)[0],  # inf - inf -> NaN
             asm("69 EXP", consts)[0],                                    # 9.3e29 finite, square overflows
             asm("40 EXP", consts)[0]]                                    # 2.35e17, square 5.5e34 finite
    r = ev(oracle, progs, consts, X, y0, want_outputs=True)
    assert np.all(np.isposinf(r["outputs"][0])) and np.isposinf(r["fitness"][0])
    assert np.all(np.isnan(r["outputs"][1])) and np.isnan(r["fitness"][1])
    assert np.all(np.isfinite(r["outputs"][2])) and np.isposinf(r["fitness"][2])
    assert np.isfinite(r["fitness"][3]) and r["fitness"][3] == pytest.approx(math.exp(80.0), rel=1e-6)
    # D5: the sum overflows before the division by N: 8 terms of 1e38 -> +inf although the mean is 1e38
    X2 = np.full((8, 1), 1.0e19, np.float32)
    r2 = ev(oracle, [asm("x0")[0]], np.zeros(1, np.float32), X2, y0)
    assert np.isposinf(r2["fitness"][0])
    r3 = ev(oracle, [asm("x0")[0]], np.zeros(1, np.float32), X2[:2], y0[:2])
    assert np.isfinite(r3["fitness"][0])


def test_malformed_programs_get_canonical_nan(oracle):
    X = np.ones((4, 2), np.float32)
    y = np.zeros(4, np.float32)
    consts = np.array([1.0], np.float32)
    T = C.token
    bad = [
        np.array([T(C.OP["ADD"])], np.int32),                               # pops from empty
        np.array([T(C.OP["LOAD"], 0), T(C.OP["ADD"])], np.int32),           # binary with one operand
        np.array([T(C.OP["LOAD"], 2)], np.int32),                           # LOAD arg >= d
        np.array([T(C.OP["CONST"], 1)], np.int32),                          # CONST arg >= n_consts
        np.array([T(0)], np.int32),                                         # opcode 0
        np.array([T(0x10)], np.int32),                                      # reserved (DUP)
        np.array([T(C.OP["LOAD"], 0), T(C.OP["SIN"], 5)], np.int32),        # operator with arg
        np.array([T(C.OP["LOAD"], 0)] * 33 + [T(C.OP["ADD"])] * 32, np.int32),  # depth 33
        np.array([T(C.OP["LOAD"], 0), T(C.OP["ADD"]), T(C.OP["LOAD"], 1)], np.int32),       # binary with one operand, depth 1 at the end
        np.array([T(C.OP["LOAD"], 0), T(C.OP["LOAD"], 1), T(C.OP["ADD"], 7)], np.int32),    # binary operator with arg
        np.array([T(C.OP["LOAD"], 0), T(C.OP["LOAD"], 1), T(C.OP["DIV"], 1)], np.int32),
    ]
    good = [np.array([T(C.OP["LOAD"], 0)] * 32 + [T(C.OP["ADD"])] * 31, np.int32),  # depth 32 is fine
            np.array([T(C.OP["LOAD"], 0), T(C.OP["LOAD"], 1)], np.int32)]            # final depth 2 (R8)
    r = ev(oracle, bad + good, consts, X, y)
    bits = r["fitness"].view(np.uint32)
    assert np.all(bits[:len(bad)] == QNAN_BITS)
    assert np.all(r["flags"][:len(bad)] & oracle.FLAG_MALFORMED)
    assert np.all(r["depth"][:len(bad)] == 0)
    assert r["fitness"][len(bad)] == 32.0 ** 2 and r["depth"][len(bad)] == 32
    assert r["fitness"][len(bad) + 1] == 1.0 and r["depth"][len(bad) + 1] == 2   # top of stack = x1
    # lengths outside [1,512] are malformed and count as 0 words
    g = np.array([T(C.OP["LOAD"], 0)], np.int32)
    l = np.array([0, -3, 600, 1], np.int32)
    rr = oracle.evaluate(g, l, consts, X, y, 0.0)
    assert np.all(rr["fitness"].view(np.uint32)[:3] == QNAN_BITS) and rr["fitness"][3] == 1.0
    # the longest program there is: 512 tokens exactly (x0, 255 times "x0 ADD", SIN) = sin(256) on X = 1; 513 tokens: malformed
    longest = [T(C.OP["LOAD"], 0)] + [T(C.OP["LOAD"], 0), T(C.OP["ADD"])] * 255 + [T(C.OP["SIN"])]
    assert len(longest) == 512
    g2 = np.array(longest + longest + [T(C.OP["SIN"])], np.int32)
    r5 = oracle.evaluate(g2, np.array([512, 513], np.int32), consts, X, y, 0.0, want_outputs=True)
    assert r5["depth"][0] == 2 and r5["outputs"][0][0] == pytest.approx(math.sin(256.0), rel=1e-12)
    assert r5["fitness"].view(np.uint32)[1] == QNAN_BITS


# ---- P11: the bound is a bound (fp32 mirror vs fp64 truth) -----------------------------------------
@pytest.mark.parametrize("cfg,P", [(1, 1024), (2, 6144)])
def test_P11_error_bound_covers_fp32_mirror(oracle, cfg, P):
    col = C.make_colony(cfg, P=P)
    ieee = oracle.contract(oracle.CONTRACT_IEEE)
    ieee.sum_per_case, ieee.sum_const = 0.0, 1.0   # the mirror sums in fp64: no fp32 summation error
    t = oracle.evaluate_parallel(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, contract_=ieee, mode=0)
    m = oracle.evaluate_parallel(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, contract_=ieee, mode=1)
    stable = (t["flags"] & (oracle.FLAG_UNSTABLE | oracle.FLAG_CLASS_UNSTABLE)) == 0
    ft, fm = t["fitness"].astype(np.float64), m["fitness"].astype(np.float64)
    # class parity on stable individuals
    assert np.array_equal(np.isnan(ft[stable]), np.isnan(fm[stable]))
    assert np.array_equal(np.isinf(ft[stable]), np.isinf(fm[stable]))
    fin = stable & np.isfinite(ft)
    slack = 2.0 ** -23 * np.abs(ft[fin])             # the two final float casts
    viol = np.abs(ft[fin] - fm[fin]) > t["bound"][fin] + slack
    assert not viol.any(), (np.flatnonzero(fin)[viol][:5], ft[fin][viol][:5], fm[fin][viol][:5], t["bound"][fin][viol][:5])
    assert stable.mean() > 0.98
    # and the bound is not vacuous: most individuals certify the north_star tolerance
    tol = np.maximum(1e-4 * np.abs(ft[fin]), 1e-6)
    assert (4 * t["bound"][fin] <= tol).mean() > 0.85


# ---- P12: duplicating the case set leaves the MSE unchanged ----------------------------------------
def test_P12_case_duplication(oracle):
    col = C.make_colony(1, P=256)
    X2, y2 = np.concatenate([col.X, col.X]), np.concatenate([col.y, col.y])
    a = oracle.evaluate(col.genomes, col.lengths, col.consts, col.X, col.y, 0.0)["fitness"]
    b = oracle.evaluate(col.genomes, col.lengths, col.consts, X2, y2, 0.0)["fitness"]
    fin = np.isfinite(a)
    assert np.array_equal(np.isfinite(a), np.isfinite(b))
    np.testing.assert_allclose(a[fin], b[fin], rtol=2e-7)


def test_parallel_fanout_equals_single_thread(oracle):
    col = C.make_colony(1)
    a = oracle.evaluate(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    b = oracle.evaluate_parallel(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, threads=4)
    for k in ("fitness", "bound", "flags", "depth"):
        assert np.array_equal(a[k], b[k], equal_nan=True)


# ---- P13-P15: the rest of GCL built so far: DUP SWAP DEL SIGN SQUARE CUBE ----------
def _quadratic_cases(seed, n=512):
    rng = np.random.default_rng(seed)
    X = np.empty((n, 3), np.float32)
    X[:, 0] = rng.uniform(0.5, 2, n) * rng.choice([-1, 1], n)
    X[:, 1] = rng.uniform(4, 8, n)
    X[:, 2] = rng.uniform(-1, 1, n)
    return X


@pytest.mark.parametrize("row", [2, 3])
def test_P13_paper_genomes_verbatim_are_the_quadratic_formula(oracle, row):
    """The 24- and 25-command genomes the paper prints (ASR 1.0 on its QuadraticEq setup, P:314,
    P:322) run verbatim, DUP / DEL / SQUARE included, and equal (sqrt(b^2 - 4ac) - b) / (2a): a closed form that
    pins what DUP duplicates, what DEL removes and the operand order around them. The leading 'CONST CONST CONST
    ADD DEL' of the first and 'CONST 3; CONST 4; SUB; CONST e; SUB; DUP; DIV; DEL' of the second are dead code."""
    cite, n, text = _golden()[row]
    prog, c = asm(_gcl_to_asm(text))
    assert len(prog) == n
    X = _quadratic_cases(13 + row)
    a, b, cc = (X[:, j].astype(np.float64) for j in range(3))
    root = (np.sqrt(b * b - 4 * a * cc) - b) / (2 * a)
    r = ev(oracle, [prog], c, X, root.astype(np.float32), want_outputs=True)
    if row == 2:      # b + (-0) is b; (b*b) - ((a+a)+(a+a))*c
        np.testing.assert_allclose(r["outputs"][0], root, rtol=1e-13)
    else:             # (c*a*-2) doubled is -4ac; added to b^2
        np.testing.assert_allclose(r["outputs"][0], root, rtol=1e-13)
    o = r["outputs"][0]
    assert np.max(np.abs(a * o * o + b * o + cc)) < 1e-9          # it is a root, whatever the formula above says
    assert r["depth"][0] >= 3 and not (r["flags"][0] & oracle.FLAG_MALFORMED)


def test_P14_stack_command_identities(oracle):
    rng = np.random.default_rng(14)
    X = rng.uniform(-3, 3, (64, 2)).astype(np.float32)
    y = np.zeros(64, np.float32)
    A, B = "x0 x1 MUL 1.5 ADD", "x1 SIN x0 SUB"
    pairs = [
        (f"{A} DUP DEL", A),                          # a duplicate removed again
        (f"{A} {B} SWAP SWAP", f"{A} {B}"),           # two swaps undo each other (output = top)
        (f"{A} {B} SWAP SUB", f"{B} {A} SUB"),        # SWAP exchanges the operands of SUB
        (f"{A} {B} SWAP DIV", f"{B} {A} DIV"),
        (f"{A} DUP MUL", f"{A} SQUARE"),              # SQUARE is a * a
        (f"{A} {A} MUL", f"{A} SQUARE"),
        (f"{A} DUP DUP MUL MUL", f"{A} CUBE"),        # CUBE is (a * a) * a; the product commutes bit for bit
        (f"{A} SIGN SIGN", A),
        (f"{A} {B} DEL", A),                          # a deleted value is dead code
        (f"x0 DEL {A}", A),                           # depth may touch zero in between
        (f"{A} {B} DUP DEL ADD", f"{A} {B} ADD"),
    ]
    for left, right in pairs:
        consts = []
        pl, pr = asm(left, consts)[0], asm(right, consts)[0]
        r = ev(oracle, [pl, pr], np.array(consts, np.float32), X, y, want_outputs=True, mode=1)
        assert np.array_equal(r["outputs"][0], r["outputs"][1]), (left, right)
    # SIGN is 0 - a (as values: the sign of a zero aside)
    consts = []
    r = ev(oracle, [asm(f"{A} SIGN", consts)[0], asm(f"0 {A} SUB", consts)[0]], np.array(consts, np.float32), X, y,
           want_outputs=True)
    assert np.all(r["outputs"][0] == r["outputs"][1])
    # the tax counts every command, stack commands included
    consts = []
    r = ev(oracle, [asm(A, consts)[0], asm(f"{A} DUP DEL", consts)[0]], np.array(consts, np.float32), X, y, tax=0.25)
    assert r["fitness"][1] - r["fitness"][0] == pytest.approx(0.5, rel=1e-6)


def test_P15_stack_command_well_formedness(oracle):
    X = np.ones((4, 2), np.float32)
    y = np.zeros(4, np.float32)
    T = C.token
    x0, x1 = T(C.OP["LOAD"], 0), T(C.OP["LOAD"], 1)
    bad = [
        np.array([T(C.OP["DUP"])], np.int32),                         # nothing to duplicate
        np.array([x0, T(C.OP["SWAP"])], np.int32),                    # SWAP needs two
        np.array([T(C.OP["DEL"])], np.int32),
        np.array([x0, T(C.OP["DEL"])], np.int32),                     # ends with an empty stack
        np.array([x0, T(C.OP["DUP"], 1)], np.int32),                  # operator with an argument
        np.array([x0] + [T(C.OP["DUP"])] * 32, np.int32),             # depth 33
        np.array([x0, T(0x13)], np.int32),                            # POW: reserved, not built yet
        np.array([x0, T(0x1D)], np.int32),                            # COPY: reserved
    ]
    good = [np.array([x0] + [T(C.OP["DUP"])] * 31 + [T(C.OP["ADD"])] * 31, np.int32),   # depth 32: 32 * x0
            np.array([x0, T(C.OP["DEL"]), x1, T(C.OP["SQUARE"])], np.int32)]
    r = ev(oracle, bad + good, np.zeros(1, np.float32), X, y)
    assert np.all(r["fitness"][:len(bad)].view(np.uint32) == QNAN_BITS)
    assert np.all(r["flags"][:len(bad)] & oracle.FLAG_MALFORMED)
    assert r["fitness"][len(bad)] == 32.0 ** 2 and r["depth"][len(bad)] == 32
    assert r["fitness"][len(bad) + 1] == 1.0


def test_P11b_bound_holds_with_the_new_commands(oracle):
    """|fit64 - fit32mirror| <= E_p on random programs that use the stack commands and SIGN SQUARE CUBE."""
    rng = np.random.default_rng(15)
    X = rng.uniform(-2, 2, (128, 3)).astype(np.float32)
    y = (X[:, 0] * X[:, 1]).astype(np.float32)
    names = ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "SQRT", "SIGN", "SQUARE", "CUBE", "DUP", "SWAP", "DEL"]
    progs, consts = [], []
    while len(progs) < 400:
        toks, depth = [], 0
        for _ in range(int(rng.integers(3, 40))):
            nm = names[int(rng.integers(len(names)))]
            need = 2 if nm in ("ADD", "SUB", "MUL", "DIV", "SWAP") else 1
            if depth < need or (nm == "DUP" and depth >= 8) or rng.random() < 0.35:
                toks.append(f"x{int(rng.integers(3))}" if rng.random() < 0.8 else f"{rng.uniform(-3, 3):.4f}"); depth += 1
            else:
                toks.append(nm); depth += {"DUP": 1, "DEL": -1}.get(nm, -1 if need == 2 and nm != "SWAP" else 0)
        if depth >= 1:
            progs.append(asm(" ".join(toks), consts)[0])
    c = np.array(consts, np.float32)
    t = ev(oracle, progs, c, X, y, contract_=oracle.contract(oracle.CONTRACT_IEEE))
    m = ev(oracle, progs, c, X, y, contract_=oracle.contract(oracle.CONTRACT_IEEE), mode=1)
    assert not np.any(t["flags"] & oracle.FLAG_MALFORMED)
    fin = np.isfinite(t["fitness"]) & np.isfinite(m["fitness"]) & ((t["flags"] & 6) == 0)
    assert fin.sum() > 200
    diff = np.abs(t["fitness"].astype(np.float64) - m["fitness"].astype(np.float64))
    assert np.all(diff[fin] <= t["bound"][fin] + 1e-30)


# ---- P16: CBRT TAN ARCSIN ARCCOS ARCTAN TANH reduce to library routines; identities; domain edges ----------
def test_P16_unary_functions_reduce_to_numpy_and_identities(oracle):
    rng = np.random.default_rng(16)
    X = np.empty((512, 2), np.float32)
    X[:, 0] = rng.uniform(-0.95, 0.95, 512)
    X[:, 1] = rng.uniform(-6, 6, 512)
    y = np.zeros(512, np.float32)
    a, b = X[:, 0].astype(np.float64), X[:, 1].astype(np.float64)
    cases = [("x1 CBRT", np.cbrt(b)), ("x0 TAN", np.tan(a)), ("x0 ARCSIN", np.arcsin(a)), ("x0 ARCCOS", np.arccos(a)),
             ("x1 ARCTAN", np.arctan(b)), ("x1 TANH", np.tanh(b))]
    for text, want in cases:
        r = ev(oracle, [asm(text)[0]], np.zeros(1, np.float32), X, y, want_outputs=True)
        np.testing.assert_allclose(r["outputs"][0], want, rtol=1e-14, atol=1e-300, err_msg=text)
    ident = [("x0 ARCSIN SIN", a), ("x0 ARCCOS COS", a), ("x0 TAN ARCTAN", a), ("x1 CBRT CUBE", b),
             ("x0 SIN x0 COS DIV", np.tan(a)),                       # tan = sin / cos
             ("x0 ARCSIN x0 ARCCOS ADD", np.full(512, np.pi / 2))]   # asin + acos = pi/2
    for text, want in ident:
        r = ev(oracle, [asm(text)[0]], np.zeros(1, np.float32), X, y, want_outputs=True)
        np.testing.assert_allclose(r["outputs"][0], want, rtol=1e-12, atol=1e-14, err_msg=text)
    # tanh through the exponential: (e^{2x} - 1) / (e^{2x} + 1)
    consts = []
    p1 = asm("x1 2 MUL EXP 1 SUB x1 2 MUL EXP 1 ADD DIV", consts)[0]
    p2 = asm("x1 TANH", consts)[0]
    r = ev(oracle, [p1, p2], np.array(consts, np.float32), X, y, want_outputs=True)
    np.testing.assert_allclose(r["outputs"][0], r["outputs"][1], rtol=1e-11, atol=1e-15)


def test_P16_domain_edges(oracle):
    vals = np.array([0.0, -0.0, 1.0, -1.0, 1.0000001, -2.0, np.inf, -np.inf, np.nan, 1e-30, -8.0, 27.0], np.float32)
    X = vals[:, None].copy()
    y = np.zeros(len(vals), np.float32)
    out = {}
    for nm in ("CBRT", "TAN", "ARCSIN", "ARCCOS", "ARCTAN", "TANH"):
        out[nm] = ev(oracle, [asm(f"x0 {nm}")[0]], np.zeros(1, np.float32), X, y, want_outputs=True)["outputs"][0]
    assert out["CBRT"][10] == -2.0 and out["CBRT"][11] == pytest.approx(3.0, rel=1e-15) and out["CBRT"][6] == np.inf and out["CBRT"][0] == 0.0
    assert out["ARCSIN"][2] == pytest.approx(np.pi / 2) and out["ARCSIN"][3] == pytest.approx(-np.pi / 2)
    assert np.isnan(out["ARCSIN"][4]) and np.isnan(out["ARCSIN"][5]) and np.isnan(out["ARCSIN"][6])   # outside [-1, 1]: NaN
    assert out["ARCCOS"][2] == 0.0 and out["ARCCOS"][3] == pytest.approx(np.pi) and np.isnan(out["ARCCOS"][4])
    assert out["ARCTAN"][6] == pytest.approx(np.pi / 2) and out["ARCTAN"][7] == pytest.approx(-np.pi / 2)
    assert out["TANH"][6] == 1.0 and out["TANH"][7] == -1.0 and out["TANH"][0] == 0.0
    assert np.isnan(out["TAN"][6]) and out["TAN"][0] == 0.0
    for nm in out:
        assert np.isnan(out[nm][8])                       # NaN in, NaN out


def test_P16_bound_is_a_bound_for_the_functions(oracle):
    rng = np.random.default_rng(17)
    X = rng.uniform(-1.5, 1.5, (128, 2)).astype(np.float32)
    y = np.zeros(128, np.float32)
    progs, consts = [], []
    fns = ["CBRT", "TAN", "ARCSIN", "ARCCOS", "ARCTAN", "TANH"]
    for i in range(300):
        f1, f2 = fns[int(rng.integers(6))], fns[int(rng.integers(6))]
        progs.append(asm(f"x0 x1 {['ADD','MUL','SUB'][i % 3]} {f1} x1 {f2} {['MUL','ADD'][i % 2]} {rng.uniform(0.2, 2):.3f} MUL", consts)[0])
    c = np.array(consts, np.float32)
    ieee = oracle.contract(oracle.CONTRACT_IEEE)
    t = ev(oracle, progs, c, X, y, contract_=ieee)
    m = ev(oracle, progs, c, X, y, contract_=ieee, mode=1)
    fin = np.isfinite(t["fitness"]) & np.isfinite(m["fitness"]) & ((t["flags"] & 6) == 0)
    assert fin.sum() > 60
    diff = np.abs(t["fitness"].astype(np.float64) - m["fitness"].astype(np.float64))
    assert np.all(diff[fin] <= t["bound"][fin] + 1e-30)


# ---- P17: POW; P18: COPY / PASTE ----------------------------------------------------------------------------
def test_P17_pow_reduces_to_numpy_and_identities(oracle):
    rng = np.random.default_rng(18)
    X = np.empty((512, 2), np.float32)
    X[:, 0] = rng.uniform(0.2, 4, 512)
    X[:, 1] = rng.uniform(-3, 3, 512)
    y = np.zeros(512, np.float32)
    a, b = X[:, 0].astype(np.float64), X[:, 1].astype(np.float64)
    r = ev(oracle, [asm("x0 x1 POW")[0]], np.zeros(1, np.float32), X, y, want_outputs=True)
    np.testing.assert_allclose(r["outputs"][0], np.power(a, b), rtol=1e-14)       # second-top ^ top
    consts = []
    progs = [asm(t, consts)[0] for t in ("x0 2 POW", "x0 SQUARE", "x0 3 POW", "x0 CUBE", "x0 0.5 POW", "x0 SQRT",
                                         "x0 x1 POW", "x0 LOG x1 MUL EXP", "x0 -1 POW", "1 x0 DIV")]
    r = ev(oracle, progs, np.array(consts, np.float32), X, y, want_outputs=True)
    for k in range(0, 10, 2):
        np.testing.assert_allclose(r["outputs"][k], r["outputs"][k + 1], rtol=1e-12, err_msg=str(k))
    # the C pow function at its edges: negative base with an integer / non-integer exponent, zero base, zero exponent
    vals = np.array([[-2.0, 3.0], [-2.0, 2.0], [-2.0, 0.5], [0.0, 2.0], [0.0, -1.0], [5.0, 0.0], [np.nan, 0.0], [-8.0, 1.0 / 3.0]], np.float32)
    o = ev(oracle, [asm("x0 x1 POW")[0]], np.zeros(1, np.float32), vals, np.zeros(len(vals), np.float32), want_outputs=True)["outputs"][0]
    assert o[0] == -8.0 and o[1] == 4.0 and np.isnan(o[2]) and o[3] == 0.0 and o[4] == np.inf and o[5] == 1.0 and o[6] == 1.0 and np.isnan(o[7])


def test_P17b_bound_is_a_bound_for_pow(oracle):
    """|fit64 - fit32mirror| <= E_p on random programs that contain POW: the corner bound of run_case's POW (the four
    corners of the operand box, UNSTABLE when the box reaches a base <= 0 or a NaN) is a bound, as P11 / P11b / P16 show
    for the other commands. Bases are kept positive by construction often enough that most programs stay unflagged."""
    rng = np.random.default_rng(171)
    X = rng.uniform(0.3, 3.0, (96, 3)).astype(np.float32)
    y = (X[:, 0] ** X[:, 1]).astype(np.float32)
    progs, consts = [], []
    shapes = ["x{a} x{b} POW", "x{a} {c:.3f} POW", "x{a} x{b} MUL x{c2} POW", "x{a} SQRT x{b} {c:.3f} MUL POW",
              "x{a} x{b} POW x{c2} ADD", "x{a} {c:.3f} ADD x{b} SIN POW", "x{a} x{b} POW x{c2} x{a} POW MUL",
              "x{a} x{b} DIV x{c2} POW {c:.3f} SUB", "{c:.3f} x{a} POW", "x{a} x{b} POW x{c2} POW"]
    for i in range(400):
        a, b, c2 = (int(v) for v in rng.integers(0, 3, 3))
        progs.append(asm(shapes[i % len(shapes)].format(a=a, b=b, c2=c2, c=float(rng.uniform(0.2, 2.5))), consts)[0])
    c = np.array(consts, np.float32)
    ieee = oracle.contract(oracle.CONTRACT_IEEE)
    t = ev(oracle, progs, c, X, y, contract_=ieee)
    m = ev(oracle, progs, c, X, y, contract_=ieee, mode=1)
    assert not np.any(t["flags"] & oracle.FLAG_MALFORMED)
    fin = np.isfinite(t["fitness"]) & np.isfinite(m["fitness"]) & ((t["flags"] & 6) == 0)
    assert fin.sum() >= 300, fin.sum()
    diff = np.abs(t["fitness"].astype(np.float64) - m["fitness"].astype(np.float64))
    slack = 2.0 ** -23 * np.abs(t["fitness"].astype(np.float64))          # the two final float casts
    assert np.all(diff[fin] <= t["bound"][fin] + slack[fin]), np.flatnonzero(fin & (diff > t["bound"] + slack))[:5]
    # and it is not vacuous: most of them certify north_star's tolerance
    tol = np.maximum(1e-4 * np.abs(t["fitness"][fin].astype(np.float64)), 1e-6)
    assert (4 * t["bound"][fin] <= tol).mean() > 0.8


def test_P18_copy_paste_variables(oracle):
    rng = np.random.default_rng(19)
    X = rng.uniform(-3, 3, (64, 2)).astype(np.float32)
    y = np.zeros(64, np.float32)
    A, B = "x0 x1 MUL 1.5 ADD", "x1 SIN x0 SUB"
    pairs = [
        (f"{A} COPY@1 PASTE@1 MUL", f"{A} SQUARE"),                 # COPY leaves the stack alone, PASTE pushes the copy
        (f"{A} COPY@2 DEL {B} PASTE@2 SUB", f"{B} {A} SUB"),        # the value survives while the stack moves on
        (f"{A} COPY@0 {B} COPY@31 DEL DEL PASTE@31 PASTE@0 DIV", f"{B} {A} DIV"),
        (f"{A} COPY@5 PASTE@5 DEL", A),
        (f"{A} COPY@1 PASTE@1 COPY@1 PASTE@1 ADD ADD", f"{A} DUP DUP ADD ADD"),   # a variable can be used again after its PASTE
    ]
    for left, right in pairs:
        consts = []
        pl, pr = asm(left, consts)[0], asm(right, consts)[0]
        r = ev(oracle, [pl, pr], np.array(consts, np.float32), X, y, want_outputs=True, mode=1)
        assert np.array_equal(r["outputs"][0], r["outputs"][1]), (left, right)
    bad = ["x0 PASTE@1", "x0 COPY@1", "x0 COPY@1 COPY@1 PASTE@1", "x0 COPY@1 PASTE@1 PASTE@1", "COPY@1 x0 PASTE@1", "x0 COPY@32 PASTE@32",
           "x0 COPY@1 PASTE@2"]
    progs = [asm(t)[0] for t in bad]
    r = ev(oracle, progs, np.zeros(1, np.float32), X, y)
    assert np.all(r["fitness"].view(np.uint32) == QNAN_BITS) and np.all(r["flags"] & oracle.FLAG_MALFORMED)
    # depth 32 through PASTE
    deep = asm("x0 COPY@3 " + "x0 " * 30 + "PASTE@3 " + "ADD " * 31)[0]
    r = ev(oracle, [deep], np.zeros(1, np.float32), np.ones((4, 2), np.float32), np.zeros(4, np.float32))
    assert r["depth"][0] == 32 and r["fitness"][0] == 32.0 ** 2


# ---- P19: the correlation fitness (Eq. 1-2; oracle orc_eval_corr) ---------------------------------
M_SCORE = 10000.0     # BConfig.MaxScore as the paper's logs imply it: ASR 0.32808 = 1,679,752 / 5,120,000 at N = 512


def evc(oracle, texts, X, y, M=M_SCORE, tax=0.0):
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts if consts else np.zeros(1, np.float32))
    return oracle.evaluate_corr(g, l, c, X, y, M, tax), l


def test_P19_correlation_worked_example_and_library(oracle):
    # by hand: y = 1 2 3 4, f = 1 3 2 4: both centred sums of squares are 5, the cross sum is 4: r = 0.8, r^4 = 0.4096
    X = np.array([[1.0], [3.0], [2.0], [4.0]], np.float32)
    y = np.array([1.0, 2.0, 3.0, 4.0], np.float32)
    r, _ = evc(oracle, ["x0"], X, y)
    assert abs(r["fitness"][0] - 10000.0 * 0.4096 * 4) < 1e-6 * 16384 and abs(r["stats"][0, 0] - 0.64) < 1e-14
    # the library routine on random data, outputs taken from the (pinned) evaluator
    rng = np.random.default_rng(5)
    X = rng.uniform(-2, 2, (300, 3)).astype(np.float32)
    y = (X[:, 0] * X[:, 1] + 0.3 * rng.standard_normal(300)).astype(np.float32)
    texts = ["x0 x1 MUL", "x0 x1 ADD SIN", "x2 x0 MUL x1 SUB", "x0 x1 MUL x2 0.1 MUL ADD"]
    r, _ = evc(oracle, texts, X, y)
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    outs = ev(oracle, progs, np.array(consts, np.float32), X, y, want_outputs=True)["outputs"]
    for k in range(len(texts)):
        rr = np.corrcoef(outs[k], y.astype(np.float64))[0, 1]
        assert abs(r["stats"][k, 0] - rr * rr) < 1e-12
        assert abs(r["fitness"][k] - M_SCORE * rr ** 4 * 300) <= 1e-6 * M_SCORE * 300
        assert r["stats"][k, 1] == 300 and r["stats"][k, 2] == 0 and r["stats"][k, 3] == 0


def test_P19_correlation_invariances_and_degenerate_cases(oracle):
    rng = np.random.default_rng(6)
    N = 128
    X = rng.uniform(-2, 2, (N, 2)).astype(np.float32)
    y = (X[:, 0] - 0.5 * X[:, 1]).astype(np.float32)
    # r^2 does not change under f -> a f + b (a != 0, either sign): power-of-two a and a small b keep fp64 exactness close
    r, l = evc(oracle, ["x0 x1 MUL x0 ADD", "x0 x1 MUL x0 ADD 4 MUL 3 ADD", "x0 x1 MUL x0 ADD -0.5 MUL 1 SUB"], X, y)
    assert np.allclose(r["stats"][:, 0], r["stats"][0, 0], rtol=1e-12) and 0.0 < r["stats"][0, 0] < 1.0
    # a perfect model, its negative and any increasing affine map of it all score M N; the score is linear in M
    r, _ = evc(oracle, ["x0 x1 0.5 MUL SUB", "x1 0.5 MUL x0 SUB", "x0 x1 0.5 MUL SUB 8 MUL 2 ADD"], X, y)
    assert np.allclose(r["fitness"], M_SCORE * N, rtol=1e-6)
    r2, _ = evc(oracle, ["x0 x1 MUL"], X, y, M=2.0 * M_SCORE)
    r1, _ = evc(oracle, ["x0 x1 MUL"], X, y)
    assert abs(r2["fitness"][0] - 2.0 * r1["fitness"][0]) <= 1e-6 * abs(r2["fitness"][0])
    # zero variance on the model's side: r = 0 (reading R23); the length tax is taken off the score per command
    r, l = evc(oracle, ["1.5", "x0 x1 MUL"], X, y, tax=7.0)
    assert r["fitness"][0] == -7.0 and r["stats"][0, 0] == 0.0
    assert abs(r["fitness"][1] - (r1["fitness"][0] - 7.0 * 3)) <= 1e-6 * abs(r1["fitness"][0])
    # independent of the order of the cases
    perm = rng.permutation(N)
    rp, _ = evc(oracle, ["x0 x1 MUL"], X[perm], y[perm])
    assert abs(rp["stats"][0, 0] - r1["stats"][0, 0]) < 1e-13


def test_P19_correlation_invalid_pairs(oracle):
    """Eq. 2's counts: c1 valid/invalid pairs cost M each, c2 invalid/invalid pairs earn M each, and r is taken over the
    valid pairs only. f = x0 * x1 with x1 = 1e30 where the model is to overflow, ARCSIN of 2 where it is to be NaN."""
    N = 16
    x0 = np.arange(1, N + 1, dtype=np.float32)
    big = np.ones(N, np.float32)
    big[[1, 5, 9]] = 1e30                       # f = x0 * big * big overflows at cases 1, 5, 9
    x0[12] = 40.0
    X = np.stack([x0, big], axis=1)
    y = (3.0 * x0 + 1.0).astype(np.float32)     # perfectly correlated with x0 wherever both are finite
    y[5] = np.nan                               # invalid / invalid at 5
    y[2] = np.inf                               # valid model / invalid target at 2
    r, _ = evc(oracle, ["x0 x1 MUL x1 MUL"], X, y)
    nv, c1, c2 = r["stats"][0, 1:]
    assert (nv, c1, c2) == (12, 3, 1)           # c1: cases 1, 9 (model) and 2 (target); c2: case 5
    assert abs(r["stats"][0, 0] - 1.0) < 1e-12
    assert abs(r["fitness"][0] - (M_SCORE * 12 - M_SCORE * (3 - 1))) < 1e-3
    # NaN on the model's side counts like Inf; the valid pairs that are left decide r
    X2 = np.stack([x0, np.where(np.arange(N) % 4 == 0, 2.0, 0.5).astype(np.float32)], axis=1)
    y2 = (x0 * 2).astype(np.float32)
    r, _ = evc(oracle, ["x1 ARCSIN 0 MUL x0 ADD"], X2, y2)
    assert tuple(r["stats"][0, 1:]) == (12, 4, 0) and abs(r["stats"][0, 0] - 1.0) < 1e-12
    assert abs(r["fitness"][0] - (M_SCORE * 12 - M_SCORE * 4)) < 1e-3
    # fewer than two valid pairs: r = 0, the counts still score
    y3 = np.full(N, np.nan, np.float32); y3[0] = 1.0
    r, _ = evc(oracle, ["x0"], np.stack([x0, big], axis=1), y3)
    assert tuple(r["stats"][0, :]) == (0.0, 1, 15, 0) and r["fitness"][0] == -M_SCORE * 15
    # brute force over tiny data: the definition retyped with numpy on every subset mask of valid targets
    rng = np.random.default_rng(9)
    xs = rng.uniform(-1, 1, (6, 1)).astype(np.float32)
    for mask in range(1, 64):
        yy = rng.uniform(-1, 1, 6).astype(np.float32)
        inv = np.array([(mask >> k) & 1 for k in range(6)], bool)
        yy[inv] = np.inf
        r, _ = evc(oracle, ["x0 SQUARE"], xs, yy)
        v = ~inv
        fo = xs[v, 0].astype(np.float64) ** 2
        want = 0.0
        if v.sum() >= 2:
            want = np.corrcoef(fo, yy[v].astype(np.float64))[0, 1] ** 4
        assert abs(r["fitness"][0] - (M_SCORE * want * v.sum() - M_SCORE * inv.sum())) <= 1e-6 * M_SCORE * 6 + 1e-3


def test_P19_correlation_bound_is_a_bound(oracle):
    """An fp32 evaluation of the same definition (IEEE per-command mirror outputs, numpy float32 two-pass sums) stays
    within the oracle's certified bound wherever the oracle does not flag the individual."""
    rng = np.random.default_rng(10)
    N, d = 512, 3
    X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
    y = (X[:, 0] * X[:, 1] - X[:, 2]).astype(np.float32)
    from tests.util import random_gcl_programs
    texts = random_gcl_programs(rng, 400, d, ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "SQRT", "EXP", "LOG"])
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, cst = pack(progs, consts)
    ieee = oracle.contract(oracle.CONTRACT_IEEE)
    ieee.sum_per_case = 1.0                          # numpy's pairwise float32 sums: any order
    r = oracle.evaluate_corr(g, l, cst, X, y, M_SCORE, 0.0, contract_=ieee)
    outs = oracle.evaluate(g, l, cst, X, y, 0.0, mode=1, want_outputs=True, contract_=ieee)["outputs"].astype(np.float32)
    ok = (r["flags"] == 0)
    assert ok.sum() > 100
    worst = 0.0
    for p in np.nonzero(ok)[0]:
        f = outs[p]
        v = np.isfinite(f) & np.isfinite(y)
        nv = int(v.sum()); c1 = int((np.isfinite(f) != np.isfinite(y)).sum()); c2 = N - nv - c1
        score = np.float32(0)
        if nv >= 2:
            fv, yv = f[v] - f[v][0], y[v] - y[v][0]
            df = fv - np.float32(fv.sum(dtype=np.float32) / np.float32(nv)); dy = yv - np.float32(yv.sum(dtype=np.float32) / np.float32(nv))
            sff, syy, sfy = (df * df).sum(dtype=np.float32), (dy * dy).sum(dtype=np.float32), (df * dy).sum(dtype=np.float32)
            r2 = np.float32(sfy * sfy) / np.float32(sff * syy) if sff > 0 and syy > 0 else np.float32(0)
            score = np.float32(M_SCORE) * np.float32(r2 * r2) * np.float32(nv)
        score = float(score) - M_SCORE * (c1 - c2)
        err = abs(score - float(r["fitness"][p]))
        assert err <= r["bound"][p] + np.spacing(np.float32(abs(score))), (p, err, r["bound"][p])
        worst = max(worst, err / max(r["bound"][p], 1e-300))
    print("worst err / bound:", worst)


# ---- P20: Monte-Carlo ranking (Table 2; oracle/ranking.py) ------------------------------------------
def test_P20_ranking_table_and_deciles():
    from oracle import ranking as R
    # Table 2 as printed, top row first; its mean is exactly one child per individual: a stable population
    printed = [4, 2.5, 1.5, 1, 0.5, 0.25, 0.15, 0.06, 0.03, 0.01]
    assert list(R.EXPECTED_CHILDREN[::-1]) == printed and abs(sum(printed) - 10.0) < 1e-12
    # distinct fitnesses 0..999 (to be maximised), sample = 5, 15, 25, ...: individual i has ceil((i - 5) / 10) samples below it
    f = np.arange(1000, dtype=np.float32)
    sample = np.arange(5, 1000, 10)
    dec, hist, kids = R.rank_deciles(f, sample, True)
    want = np.minimum(9, np.maximum(0, -(-(np.arange(1000) - 5) // 10)) // 10)
    assert np.array_equal(dec, want) and hist.sum() == 1000 and np.all(np.abs(hist - 100) <= 10)
    assert abs(kids.mean() - 1.0) < 0.05
    # minimised (MSE): the order flips
    dec2, _, _ = R.rank_deciles(f, sample, False)
    assert np.array_equal(dec2, R.rank_deciles(-f, sample, True)[0]) and dec2[0] == 9 and dec2[999] == 0
    # NaN is worse than everything, +inf MSE is worse than any finite MSE; ties share the lower group
    f3 = np.array([1.0, np.nan, np.inf, 2.0, 2.0, 0.5], np.float32)
    dec3, _, _ = R.rank_deciles(f3, np.arange(6), False)      # the sample is the whole population: 6 samples
    # strictly worse counts: 1.0 -> {nan, inf, 2, 2} = 4; nan -> 0; inf -> 0 (nan ties at -inf); 2.0 -> {nan, inf} = 2; 0.5 -> 5
    assert list(dec3) == [min(9, 10 * c // 6) for c in (4, 0, 0, 2, 2, 5)]


def test_P20_ranking_brute_force_against_sorting():
    from oracle import ranking as R
    rng = np.random.default_rng(20)
    for trial in range(20):
        P = int(rng.integers(5, 400))
        f = rng.standard_normal(P).astype(np.float32)
        f[rng.random(P) < 0.05] = np.nan
        f = np.round(f, 1) if trial % 2 else f                # ties
        sample = rng.integers(0, P, 100)
        for mx in (True, False):
            dec, hist, _ = R.rank_deciles(f, sample, mx)
            g = np.where(np.isnan(f), -np.inf, f if mx else -f).astype(np.float64)
            srt = np.sort(g[sample])
            worse = np.searchsorted(srt, g, side="left")      # samples strictly below
            assert np.array_equal(dec, np.minimum(9, worse // 10)) and np.array_equal(hist, np.bincount(dec, minlength=10))


# ---- P21: the Std integer-reward family (Eq. 5 at P:503-506; oracle orc_eval_std) ----------------------
def evs(oracle, texts, X, y, power=1, M=M_SCORE, tax=0.0):
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts if consts else np.zeros(1, np.float32))
    return oracle.evaluate_std(g, l, c, X, y, power, M, tax)


def test_P21_std_rewards_by_hand(oracle):
    # Eq. 5 case by case, M = 10000, model f = x0:
    #   f = 1, y = 2: 10000 * 1/2 = 5000;  f = -1, y = 2: round(5000 - 909.09..) = 4091;  f = y = 0: M;
    #   f = 3, y = 3: M;  f = 0, y = 5: 0;  f = -4, y = -1: 2500;  f = 2, y = -2: round(10000 - 909.09) = 9091;
    #   f = 1, y = 3: round(3333.33) = 3333;  f = 2, y = 3: round(6666.67) = 6667
    f = np.array([1, -1, 0, 3, 0, -4, 2, 1, 2], np.float32)
    y = np.array([2, 2, 0, 3, 5, -1, -2, 3, 3], np.float32)
    want = [5000, 4091, 10000, 10000, 0, 2500, 9091, 3333, 6667]
    for k in range(len(f)):
        r = evs(oracle, ["x0"], f[k:k + 1].reshape(1, 1), y[k:k + 1])
        assert r["fitness"][0] == want[k], (k, r["fitness"][0])
    r = evs(oracle, ["x0"], f.reshape(-1, 1), y)
    assert r["fitness"][0] == sum(want)                        # the score is the sum over the cases
    # Square, Cube, Hyper: the ratio to the power 2, 3, 8 (f = 1, y = 2: 2500, 1250, 39.0625 -> 39; opposite signs keep the penalty)
    for power, w in ((2, 2500), (3, 1250), (8, 39)):
        assert evs(oracle, ["x0"], np.array([[1.0]], np.float32), np.array([2.0], np.float32), power)["fitness"][0] == w
    assert evs(oracle, ["x0"], np.array([[-1.0]], np.float32), np.array([2.0], np.float32), 2)["fitness"][0] == 2500 - 909
    # round half to even: M = 1, q = 1/2 -> 0.5 -> 0;  M = 3, q = 1/2 -> 1.5 -> 2;  M = 5 -> 2.5 -> 2
    for M, w in ((1.0, 0), (3.0, 2), (5.0, 2), (7.0, 4)):
        assert evs(oracle, ["x0"], np.array([[1.0]], np.float32), np.array([2.0], np.float32), 1, M)["fitness"][0] == w
    # invalid pairs as in Eq. 2: one side finite -1 M each, neither +1 M; the tax per command comes off the score
    X = np.array([[1.0], [1e30], [1.0], [1e30]], np.float32)
    yy = np.array([1.0, 1.0, np.nan, np.inf], np.float32)
    r = evs(oracle, ["x0 x0 MUL"], X, yy, 1, M_SCORE, tax=3.0)           # f = 1, inf, 1, inf
    assert r["fitness"][0] == 10000 - 10000 - 10000 + 10000 - 3.0 * 3
    # symmetric in (f, y); a perfect model scores M N
    rng = np.random.default_rng(21)
    a = rng.uniform(-3, 3, 200).astype(np.float32); b = rng.uniform(-3, 3, 200).astype(np.float32)
    r1 = evs(oracle, ["x0"], a.reshape(-1, 1), b); r2 = evs(oracle, ["x0"], b.reshape(-1, 1), a)
    assert r1["fitness"][0] == r2["fitness"][0]
    assert evs(oracle, ["x0"], a.reshape(-1, 1), a)["fitness"][0] == M_SCORE * 200
    # numpy restatement on random data (float32 arithmetic, np.rint = half to even)
    q = np.minimum(np.abs(a), np.abs(b)) / np.maximum(np.abs(a), np.abs(b))
    for power in (1, 2, 3, 8):
        qp = {1: q, 2: q * q, 3: (q * q) * q, 8: ((q * q) * (q * q)) * ((q * q) * (q * q))}[power]
        t = np.float32(M_SCORE) * qp - np.where(a * b < 0, np.float32(M_SCORE) / np.float32(11), np.float32(0))
        assert evs(oracle, ["x0"], a.reshape(-1, 1), b, power)["fitness"][0] == np.rint(t.astype(np.float32)).sum()


@pytest.mark.parametrize("power", [1, 2, 3, 8])
def test_P21b_std_bound_is_a_bound(oracle, power):
    """The bound E of orc_eval_std is a bound: the score computed from the fp32 mirror's outputs (mode 1: every command
    rounded to fp32) differs from the score computed from the fp64 outputs (mode 0) by at most E, for every unflagged
    individual of >= 300 random programs per power; and E is not vacuous (most individuals have E below one reward
    step per 16 cases)."""
    rng = np.random.default_rng(210 + power)
    N, d = 256, 3
    X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
    y = (X[:, 0] * X[:, 1] + np.sin(X[:, 2])).astype(np.float32)
    from tests.util import random_gcl_programs
    texts = random_gcl_programs(rng, 500, d, ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "SQRT", "EXP", "LOG"])
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, cst = pack(progs, consts)
    ieee = oracle.contract(oracle.CONTRACT_IEEE)
    t = oracle.evaluate_std(g, l, cst, X, y, power, M_SCORE, 0.0, contract_=ieee, mode=0)
    m = oracle.evaluate_std(g, l, cst, X, y, power, M_SCORE, 0.0, contract_=ieee, mode=1)
    ok = (t["flags"] == 0) & np.isfinite(t["fitness"]) & np.isfinite(m["fitness"])
    assert ok.sum() >= 300, ok.sum()
    diff = np.abs(t["fitness"].astype(np.float64) - m["fitness"].astype(np.float64))
    assert np.all(diff[ok] <= t["bound"][ok]), (np.flatnonzero(ok & (diff > t["bound"]))[:5], diff[ok].max())
    assert (t["bound"][ok] <= N / 16).mean() > 0.6, (t["bound"][ok] <= N / 16).mean()



# ---- P22: the fp32 mirror (mode 1) is a step-by-step fp32 evaluator -------------------------------------------------
# The mirror is what the arithmetic-only GPU tests compare against bit for bit, so its own rounding points are pinned: every
# command's result, the residual, its square (D5) are rounded to fp32; the sum is carried in fp64 and rounded once.
def test_P22_mirror_rounds_every_step_like_numpy_float32(oracle):
    f32 = np.float32
    # (1) the residual is rounded before it is squared: out = 1, y = -2^-24: r = 1 + 2^-24 ties to 1.0 in fp32, r^2 = 1;
    #     squaring the unrounded residual would give 1 + 2^-23
    X = np.array([[1.0]], f32)
    y = np.array([-2.0 ** -24], f32)
    r = oracle.evaluate(*pack([asm("x0")[0]], np.zeros(1, f32))[:2], np.zeros(1, f32), X, y, 0.0, mode=1)
    assert r["fitness"][0] == f32(1.0)
    r0 = oracle.evaluate(*pack([asm("x0")[0]], np.zeros(1, f32))[:2], np.zeros(1, f32), X, y, 0.0, mode=0)
    assert r0["fitness"][0] == f32(1.0 + 2.0 ** -23)          # the truth mode keeps the fp64 residual
    # (2) random arithmetic programs against numpy float32, command by command, residual and square included
    rng = np.random.default_rng(22)
    N, d = 16, 3
    Xr = rng.uniform(-3, 3, (N, d)).astype(f32)
    yr = rng.uniform(-3, 3, N).astype(f32)
    consts = np.array([0.3, -1.7, 2.5], f32)
    texts = ["x0 x1 MUL x2 ADD", "x0 c0 SUB x1 c1 MUL MUL", "x0 x0 MUL x1 x1 MUL ADD x2 SUB", "c2 x1 SUB x0 MUL x2 x2 MUL ADD c1 ADD",
             "x0 x1 ADD x2 MUL x0 SUB x1 MUL c0 ADD"]
    vals = {"c0": consts[0], "c1": consts[1], "c2": consts[2]}
    progs = []
    for t in texts:
        toks = []
        for w in t.split():
            if w[0] == "x": toks.append(C.token(C.OP["LOAD"], int(w[1:])))
            elif w[0] == "c": toks.append(C.token(C.OP["CONST"], int(w[1:])))
            else: toks.append(C.token(C.OP[w]))
        progs.append(np.array(toks, np.int32))
    g, l, c = pack(progs, consts)
    got = oracle.evaluate(g, l, c, Xr, yr, 0.0, mode=1, want_outputs=True)
    for k, t in enumerate(texts):
        S = 0.0
        for i in range(N):
            st = []
            for w in t.split():
                if w[0] == "x": st.append(Xr[i, int(w[1:])])
                elif w[0] == "c": st.append(vals[w])
                else:
                    b, a = st.pop(), st.pop()
                    st.append({"ADD": a + b, "SUB": a - b, "MUL": a * b}[w])        # numpy float32 scalars: one rounding each
            assert isinstance(st[-1], np.float32) and got["outputs"][k][i] == float(st[-1])
            res = st[-1] - yr[i]
            S += float(res * res)                                                    # fp32 residual, fp32 square, fp64 sum
        assert got["fitness"][k] == f32(S / N)


# ---- P23: the parts of the bounds that only show when the INPUT of a command carries a large error ------------------------
# (found by mutating the oracle: with inputs that are only one rounding off, dropping the propagated input error of the library
# functions, half of POW's corners or the correlation's A / B terms went unnoticed). "noise(c)" = K x0 + c - K x0 is c exactly,
# and c +- K u |x0| in fp32: a value with a large, honest error bound.
def _noise(c, K=3000.0):
    return f"x0 {K:.1f} MUL {c:.4f} ADD x0 {K:.1f} MUL SUB"


def test_P23_bounds_hold_when_inputs_carry_large_errors(oracle):
    rng = np.random.default_rng(23)
    X = rng.uniform(0.5, 3.0, (128, 2)).astype(np.float32)
    y = np.zeros(128, np.float32)
    progs, consts = [], []
    for f in ["CBRT", "TAN", "ARCSIN", "ARCCOS", "ARCTAN", "TANH", "SIN", "COS", "EXP", "LOG", "SQRT", "SQUARE", "CUBE"]:
        for c0 in (0.31, -0.47, 0.83, 0.12):
            progs.append(asm(f"{_noise(c0)} {f}", consts)[0])
            progs.append(asm(f"{_noise(c0)} {f} x1 MUL", consts)[0])
    for c0, c1 in ((1.7, 0.6), (0.4, 2.3), (2.9, -1.2), (1.1, 1.9), (0.7, -0.4), (2.2, 0.3)):
        progs.append(asm(f"{_noise(c0)} {_noise(c1)} POW", consts)[0])         # both operands of POW uncertain: all four corners matter
        progs.append(asm(f"{_noise(c0)} x1 POW", consts)[0])
        progs.append(asm(f"x1 {_noise(c1)} POW", consts)[0])
        progs.append(asm(f"{_noise(c0)} {_noise(c1)} DIV", consts)[0])
        progs.append(asm(f"{_noise(c0)} {_noise(c1)} MUL", consts)[0])
    c = np.array(consts, np.float32)
    ieee = oracle.contract(oracle.CONTRACT_IEEE)
    t = ev(oracle, progs, c, X, y, contract_=ieee)
    m = ev(oracle, progs, c, X, y, contract_=ieee, mode=1)
    fin = np.isfinite(t["fitness"]) & np.isfinite(m["fitness"]) & ((t["flags"] & 6) == 0)
    assert fin.sum() >= 100, fin.sum()
    diff = np.abs(t["fitness"].astype(np.float64) - m["fitness"].astype(np.float64))
    slack = 2.0 ** -23 * np.abs(t["fitness"].astype(np.float64))
    bad = np.flatnonzero(fin & (diff > t["bound"] + slack))
    assert len(bad) == 0, bad[:5]
    # the errors are really large here (hundreds of roundings), and the bound is not orders of magnitude above them
    rel = diff[fin] / np.maximum(np.abs(t["fitness"][fin].astype(np.float64)), 1e-30)
    assert np.median(rel) > 20 * 2.0 ** -24
    assert np.median(t["bound"][fin] / np.maximum(diff[fin], 1e-300)) < 1e4


def test_P23_correlation_bound_with_noisy_outputs(oracle):
    rng = np.random.default_rng(231)
    N = 256
    X = rng.uniform(0.5, 3.0, (N, 2)).astype(np.float32)
    y = (X[:, 0] * 1.5 - X[:, 1]).astype(np.float32)
    consts = []
    # a small signal plus the noisy constant: the noise is a few per cent of the signal's spread, so r^2 really moves
    texts = [f"x0 1.5 MUL x1 SUB {sc:.4f} MUL {_noise(c0, K)} ADD" for sc in (0.01, 0.003) for c0 in (0.3, -0.8) for K in (3000.0, 20000.0)]
    texts += [f"x0 x1 MUL {sc:.4f} MUL {_noise(c0, K)} ADD" for sc in (0.01, 0.004) for c0 in (0.7,) for K in (3000.0, 10000.0)]
    progs = [asm(t, consts)[0] for t in texts]
    g, l, cst = pack(progs, consts)
    ieee = oracle.contract(oracle.CONTRACT_IEEE)
    r = oracle.evaluate_corr(g, l, cst, X, y, M_SCORE, 0.0, contract_=ieee)
    outs = oracle.evaluate(g, l, cst, X, y, 0.0, mode=1, want_outputs=True, contract_=ieee)["outputs"]      # the fp32 mirror's outputs
    checked, large = 0, 0
    for p in range(len(progs)):
        if r["flags"][p] != 0:
            continue
        f = outs[p]                                      # float64 holding fp32 values; the sums below in fp64: only the outputs differ
        df, dy = f - f.mean(), y.astype(np.float64) - y.astype(np.float64).mean()
        r2 = (df @ dy) ** 2 / ((df @ df) * (dy @ dy))
        score = M_SCORE * r2 * r2 * N
        err = abs(score - float(r["fitness"][p]))
        assert err <= r["bound"][p] + np.spacing(np.float32(score)), (texts[p], score, r["fitness"][p], r["bound"][p])
        large += err > 1000 * 2.0 ** -24 * abs(score)    # off by far more than rounding: only the terms A and B cover this
        checked += 1
    assert checked >= 6 and large >= 4, (checked, large)


def test_P23_summation_term_covers_an_fp32_sum(oracle):
    """E_S carries (sum_per_case N + sum_const) u S for the fp32 summation the device does and the oracle does not (its sum is
    fp64). One large square followed by 511 small ones that an fp32 running sum rounds away, in the device's order (DESIGN.md
    §7 'summation order', restated) and, under the IEEE contract ('any order'), plainly one after the other."""
    f32 = np.float32
    N = 512
    x = np.full(N, 2.0 ** -13 * 1.4, f32); x[0] = 1.0             # squares: 1 and 511 times about 0.98 * 2^-25 (under half an ulp of 1)
    X = x.reshape(N, 1)
    y = np.zeros(N, f32)
    prog = asm("x0")[0]
    q = (x.astype(np.float64)) ** 2
    # sequential fp32
    s = f32(0)
    for i in range(N):
        s = f32(s + f32(x[i] * x[i]))
    seq = float(f32(s / f32(N)))
    # the device's order: lane l holds cases 128 b + 4 l + e (b = block of 128, e = 0..3), fma chain, then a 5-level xor butterfly
    lanes = np.zeros(32, f32)
    for b in range(N // 128):
        for l in range(32):
            for e in range(4):
                i = 128 * b + 4 * l + e
                lanes[l] = f32(float(x[i]) * float(x[i]) + float(lanes[l]))      # fma: one rounding
    for m in (16, 8, 4, 2, 1):
        lanes = np.array([f32(lanes[l] + lanes[l ^ m]) for l in range(32)], f32)
    dev = float(f32(lanes[0] / f32(N)))
    exact = q.sum() / N
    ieee, b200 = oracle.contract(oracle.CONTRACT_IEEE), oracle.contract(oracle.CONTRACT_B200)
    ti = ev(oracle, [prog], np.zeros(1, f32), X, y, contract_=ieee)
    tb = ev(oracle, [prog], np.zeros(1, f32), X, y, contract_=b200)
    assert abs(float(ti["fitness"][0]) - exact) <= 2.0 ** -24 * exact
    assert abs(seq - exact) > 10 * 2.0 ** -24 * exact                       # the running sum really lost the small squares
    assert abs(seq - exact) <= ti["bound"][0]                               # any order: N u S
    assert abs(dev - exact) <= tb["bound"][0]                               # the device's order: (N / 32 + 5) u S
    assert tb["bound"][0] < ti["bound"][0] and ti["bound"][0] < 600 * 2.0 ** -24 * exact


def test_P23_overflow_edge_is_flagged_class_unstable(oracle):
    f32 = np.float32
    big = f32((2.0 - 2.0 ** -23) * 2.0 ** 63)                # big * 2^64 = FLT_MAX exactly
    prog = asm("x0 x1 MUL")[0]
    cases = [(big, f32(2.0 ** 64)),                          # the product is FLT_MAX itself: one rounding decides finite or +inf
             (big, f32(2.0 ** 63)),                          # half of it
             (big, f32(2.0 ** 64 * (1 + 2.0 ** -22)))]       # two ulps above: +inf for any evaluator within the contract
    out = []
    for a, b in cases:
        r = ev(oracle, [prog], np.zeros(1, f32), np.array([[a, b]], f32), np.zeros(1, f32), want_outputs=True)
        out.append((int(r["flags"][0]), float(r["outputs"][0][0])))
    assert out[0][0] & oracle.FLAG_CLASS_UNSTABLE and out[0][1] == 3.4028234663852886e38
    assert not out[1][0] & oracle.FLAG_CLASS_UNSTABLE and math.isfinite(out[1][1])
    assert not out[2][0] & oracle.FLAG_CLASS_UNSTABLE and out[2][1] == math.inf


def test_P23_published_contract_numbers(oracle):
    """orc_default_contract(1) is DESIGN.md §6's table, retyped there from the device's measured accuracy: the numbers the GPU
    contract test (tests/test_gpu_op_contract.py) holds the device to are the ones the oracle's bound uses."""
    c = oracle.contract(oracle.CONTRACT_B200)
    want = dict(c_add=1.0, c_mul=1.0, c_div=3.5, c_sqrt=3.0, c_exp=6.0, c_exp_arg=2.5, c_log_rel=5.0, c_log_abs=4.0,
                c_sin_abs=12.0, c_sin_arg=3.0, sum_per_case=1.0 / 32.0, sum_const=5.0, c_pow=10.0)
    for k, v in want.items():
        assert getattr(c, k) == v, k
    assert list(c.c_fun) == [3.0, 6.0, 4.0, 4.0, 4.0, 4.0]
    i = oracle.contract(oracle.CONTRACT_IEEE)
    assert (i.c_add, i.c_mul, i.c_div, i.c_sqrt, i.sum_per_case, i.sum_const) == (1.0, 1.0, 1.0, 1.0, 1.0, 0.0)
