"""CPU-only: the device's compiler of the whole language, run on the host (beagle_debug_compile = compile_general of
csrc/compile_kernel.inc compiled for the host too; the device code is the same source and its SASS is unchanged).

Two things are checked against the oracle, which shares nothing with it:
- the static check (D3): the maximum stack depth it reports is the oracle's depth_out, and it calls a program malformed
  exactly when the oracle does, on random programs of the whole language and on corrupted ones;
- the micro-ops it emits (csrc/uop.cuh) compute the program: a small micro-op machine, written here from uop.cuh's description of
  each handler (accumulator, slot stack in tensor memory, slots in local memory, folded terminals, reversed operands, staged unary
  rows, reciprocal rows), runs the records in numpy fp32 and the fitness it arrives at passes the same three-class parity rule
  against the oracle as the GPU does (tests/parity.py), for every plan of slots / reciprocal rows / staged rows.
What this does not cover: k_compile's table-driven walk (a different implementation of the same step, device only: its tables are
checked in test_host_logic_cpu.py and its output is compared bit for bit on the GPU) and the handlers' own arithmetic (GPU tests).
"""
import numpy as np
import pytest

from paper_2607_06731_b200 import api, colonies
from tests import parity
from tests.util import asm, pack, random_gcl_programs

EPS = np.float32(1e-6)
H_FRESH0, H_NFRESH = 33, 23
NAMES = {0: "END", 1: "SIN", 2: "COS", 3: "LOG", 4: "SQRT", 5: "EXP", 6: "NEG", 7: "SQR", 8: "CUBE",
         9: "ADDX", 10: "SUBX", 11: "MULX", 12: "DIVX", 13: "RSUBX", 14: "RDIVX",
         15: "ADDS", 16: "MULS", 17: "RSUBS", 18: "RDIVS", 19: "ADDM", 20: "MULM", 21: "RSUBM", 22: "RDIVM",
         23: "ADDC", 24: "SUBC", 25: "MULC", 26: "RSUBC", 27: "RDIVC", 28: "MULR",
         29: "POPS", 30: "POPM", 31: "SWAPS", 32: "SWAPM",
         33: "LX", 34: "LC", 35: "LX_SIN", 36: "LX_COS", 37: "LX_LOG", 38: "LX_SQRT", 39: "LX_EXP", 40: "LX_NEG", 41: "LX_SQR",
         42: "LX_CUBE", 43: "LX_ADDX", 44: "LX_SUBX", 45: "LX_MULX", 46: "LX_DIVX", 47: "LX_ADDC", 48: "LX_SUBC", 49: "LX_MULC",
         50: "LX_RSUBC", 51: "LX_RDIVC", 52: "LX_MULR", 53: "LS", 54: "LG", 55: "KEEP"}


def _f32(a):
    return np.asarray(a, np.float32)


def _div(a, b):                                    # DESIGN.md D2: |b| < 1e-6f ? 1 : a / b
    q = _f32(a) / _f32(b)
    return np.where(np.abs(b) < EPS, np.float32(1), q).astype(np.float32)


def _unary(name, a):
    a = _f32(a)
    if name == "SIN": return np.sin(a)
    if name == "COS": return np.cos(a)
    if name == "LOG": return np.where(np.abs(a) < EPS, np.float32(0), np.log(np.abs(a))).astype(np.float32)
    if name == "SQRT": return np.sqrt(np.abs(a))
    if name == "EXP": return np.exp(np.where(a > 80, np.float32(80), a)).astype(np.float32)      # NaN > 80 is false: NaN passes
    if name == "NEG": return -a
    if name == "SQR": return a * a
    if name == "CUBE": return (a * a) * a
    raise AssertionError(name)


def _binary(name, a, b):                           # a op b
    if name == "ADD": return _f32(a) + _f32(b)
    if name == "SUB": return _f32(a) - _f32(b)
    if name == "MUL": return _f32(a) * _f32(b)
    if name == "DIV": return _div(a, b)
    raise AssertionError(name)


def run_records(rec, X, d, S_T, k_rcp, k_un, un_row_bytes):
    """The micro-op machine of csrc/uop.cuh on N cases at once (fp32). Returns the accumulator after the last record.
    Also checks the discipline the compiler owes the interpreter: a tensor-memory push only while fewer than S_T slots are
    there, a pop only of what was pushed, local slots read only after they were written, reciprocal and staged rows only of
    the variables that have them."""
    N = X.shape[0]
    acc = None
    tstack, mem = [], {}
    fun = ["SIN", "COS", "LOG", "SQRT", "EXP"]

    def var(col):
        assert col % 16 == 0 and col // 16 < d, col
        return X[:, col // 16]

    def const(o):
        return np.full(N, np.array([o], np.uint32).view(np.float32)[0], np.float32)

    with np.errstate(all="ignore"):
        for h, o in rec.tolist():
            hn = h & 255
            assert hn != 0 and hn < H_FRESH0 + 3 * H_NFRESH, hn
            if hn >= H_FRESH0:                     # a fresh value: its push entry first
                push, hn = divmod(hn - H_FRESH0, H_NFRESH)
                hn += H_FRESH0
                if push == 1:
                    assert acc is not None and len(tstack) < S_T, (len(tstack), S_T)
                    tstack.append(acc)
                elif push == 2:
                    off = (h >> 10) & 0x7FF
                    assert acc is not None and off % 64 == 0 and off // 64 < 31 and len(tstack) == S_T
                    mem[off] = acc
            name = NAMES[hn]
            colA = h >> 21
            if name in ("SIN", "COS", "LOG", "SQRT", "EXP", "NEG", "SQR", "CUBE"):
                acc = _unary(name, acc)
            elif name[:-1] in ("ADD", "SUB", "MUL", "DIV", "RSUB", "RDIV") and name[-1] in "XSMC":
                if name[-1] == "X": x = var(o)
                elif name[-1] == "S": x = tstack.pop()
                elif name[-1] == "M": x = mem.pop(o)
                else: x = const(o)
                op = name[:-1]
                acc = _binary(op[1:], x, acc) if op[0] == "R" else _binary(op, acc, x)
            elif name == "MULR":
                assert o // 16 < k_rcp
                acc = acc * (np.float32(1) / var(o))
            elif name == "POPS": acc = tstack.pop()
            elif name == "POPM": acc = mem.pop(o)
            elif name == "SWAPS": acc, tstack[-1] = tstack[-1], acc
            elif name == "SWAPM": acc, mem[o] = mem[o], acc
            elif name == "LX": acc = var(colA)
            elif name == "LC": acc = const(o)
            elif name == "KEEP": pass
            elif name in ("LS", "LG"):
                assert un_row_bytes > 0 and o % un_row_bytes == 0
                f, j = divmod(o // un_row_bytes, k_un if name == "LS" else d)
                assert f < 5 and (j < k_un if name == "LS" else k_un <= j < d), (name, f, j)
                acc = _unary(fun[f], X[:, j])
            elif name == "LX_MULR":
                assert o // 16 < k_rcp
                acc = var(colA) * (np.float32(1) / var(o))
            elif name.startswith("LX_"):
                rest = name[3:]
                if rest in ("SIN", "COS", "LOG", "SQRT", "EXP", "NEG", "SQR", "CUBE"):
                    acc = _unary(rest, var(colA))
                else:
                    x = var(o) if rest[-1] == "X" else const(o)
                    op = rest[:-1]
                    acc = _binary(op[1:], x, var(colA)) if op[0] == "R" else _binary(op, var(colA), x)
            else:
                raise AssertionError(name)
            acc = _f32(acc)
    return acc                                     # (a program may leave more than its result on the stack: slots may still hold values)


def _fitness(out, y, tax, L):
    with np.errstate(all="ignore"):
        r = _f32(out) - _f32(y)
        return np.float32(np.float32(np.sum(r * r, dtype=np.float32)) / np.float32(len(y)) + np.float32(tax) * np.float32(L))


def _check_colony(oracle, genomes, lengths, consts, X, y, tax, plans, expect_slow=None):
    """Every program through the device's compiler (host build) for each plan; the records through the machine; against the oracle."""
    d = X.shape[1]
    orc = oracle.evaluate(genomes, lengths, consts, X, y, tax)
    unsafe = 0
    for j in range(d):
        if np.any(np.abs(X[:, j]) < EPS):
            unsafe |= 1 << j
    off = np.concatenate([[0], np.cumsum(lengths, dtype=np.int64)])
    n_slow = 0
    for S_T, k_rcp, k_un in plans:
        fit = np.full(len(lengths), np.nan, np.float32)
        ran = np.zeros(len(lengths), bool)
        for p in range(len(lengths)):
            tok = genomes[off[p]:off[p + 1]]
            depth, slow, rec = api.beagle_debug_compile(tok, consts, d, S_T, k_rcp, k_un, 4 * 512, unsafe)
            assert depth == orc["depth"][p], (p, depth, int(orc["depth"][p]))
            assert (depth == 0) == bool(orc["flags"][p] & oracle.FLAG_MALFORMED), p
            if depth == 0:
                continue
            if slow:
                n_slow += 1
                continue
            assert 1 <= len(rec) <= len(tok)                     # terminals are folded: never more records than tokens
            out = run_records(rec, X, d, S_T, k_rcp, k_un, 4 * 512)
            fit[p] = _fitness(out, y, tax, len(tok))
            ran[p] = True
        sel = np.nonzero(ran)[0]
        sub = {k: orc[k][sel] for k in ("fitness", "bound", "flags", "depth")}
        rep = parity.compare(fit[sel], sub)
        assert len(rep["bad"]) == 0, parity.describe(rep, fit[sel], sub)
        assert rep["strict"] >= 0.5 * (rep["strict"] + rep["conditioned"])          # the rule is not vacuous here either
    if expect_slow is not None:
        assert (n_slow > 0) == expect_slow
    return orc


PLANS = [(3, 0, 0), (0, 0, 0), (1, 2, 1), (2, 3, 3)]          # (slot rows in tensor memory, reciprocal rows, staged unary rows)


def _cases(rng, N, d, lo=-2.0, hi=2.0, zero_in=None):
    X = rng.uniform(lo, hi, size=(N, d)).astype(np.float32)
    if zero_in is not None:
        X[3, zero_in] = 0.0                        # a protected division by this variable: no reciprocal row for it
    y = (X[:, 0] * X[:, 1 % d] - X[:, (2 % d)]).astype(np.float32)
    return X, y


def test_hot_path_trees_compile_to_records_that_compute_them(oracle):
    """Colonies of the five configs' generators (the eleven tree commands; config 5's exact-length programs go 32 deep)."""
    for number, P in ((1, 300), (3, 300), (4, 200), (5, 400)):
        cfg = colonies.CONFIGS[number]
        g, l, c = colonies.generate_programs(cfg, P)
        X, y, _ = colonies.make_dataset(cfg)
        orc = _check_colony(oracle, g, l, c, X[:48], y[:48], cfg.tax, PLANS[:3] if number != 5 else PLANS, expect_slow=False)
        if number == 5:
            assert orc["depth"].max() >= 20        # deep stacks: slots beyond the tensor-memory rows are exercised


def test_the_papers_whole_language(oracle):
    """DUP SWAP DEL SIGN SQUARE CUBE are compiled (resolved on the abstract stack, a slot move for computed values); POW, the six
    library functions and COPY / PASTE are checked and handed to the blockwise kernel."""
    rng = np.random.default_rng(7)
    d = 3
    fast = ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP", "DUP", "SWAP", "DEL", "SIGN", "SQUARE", "CUBE"]
    texts = random_gcl_programs(rng, 700, d, fast)
    cl = []
    progs = [asm(t, cl)[0] for t in texts]
    g, l, c = pack(progs, cl)
    X, y = _cases(rng, 40, d, zero_in=1)
    _check_colony(oracle, g, l, c, X, y, 1e-3, PLANS, expect_slow=False)
    texts = random_gcl_programs(rng, 300, d, fast + ["POW", "TANH", "ARCTAN", "CBRT", "TAN", "ARCSIN", "ARCCOS"])
    texts += ["x0 COPY@3 x1 ADD PASTE@3 MUL", "x0 x1 COPY@0 ADD PASTE@0 SUB"]
    cl = []
    progs = [asm(t, cl)[0] for t in texts]
    g, l, c = pack(progs, cl)
    _check_colony(oracle, g, l, c, X, y, 1e-3, PLANS[:2], expect_slow=True)


def _gcl_to_asm(text):
    """GCL text as the paper prints it ('LOAD b:1; CONST 0.5; MUL;') -> the test assembler's text."""
    out = []
    for cmd in [c.strip() for c in text.split(";") if c.strip()]:
        parts = cmd.split()
        out.append("x" + parts[1].split(":")[1] if parts[0] == "LOAD" else parts[1] if parts[0] == "CONST" else {"LN": "LOG"}.get(parts[0], parts[0]))
    return " ".join(out)


def test_the_papers_printed_genomes(oracle):
    """tests/golden/paper_genomes.txt: the quadratic-formula genomes, DUP / DEL / SQUARE included,
    are compiled (none is handed to the blockwise kernel) and their records compute what the oracle computes."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_genomes.txt")
    rows = [ln.split("|") for ln in open(path) if ln.strip() and not ln.startswith("#")]
    assert [int(r[1]) for r in rows] == [12, 12, 24, 25]
    rng = np.random.default_rng(11)
    cl = []
    progs = [asm(_gcl_to_asm(r[2]), cl)[0] for r in rows]
    assert [len(t) for t in progs] == [12, 12, 24, 25]
    g, l, c = pack(progs, cl)
    X, y = _cases(rng, 40, 3, lo=1.0, hi=3.0)
    _check_colony(oracle, g, l, c, X, y, 1e-3, PLANS, expect_slow=False)


def test_corrupted_programs_are_malformed_exactly_when_the_oracle_says_so(oracle):
    """Single-token corruptions of well-formed programs (an unknown opcode, an argument on a command, a variable or a constant
    that does not exist, a token dropped or doubled, a COPY without its PASTE): the device's static check and the oracle's agree
    on every one, and on the depth of the ones that stay programs."""
    rng = np.random.default_rng(2607)
    d = 4
    names = ["ADD", "SUB", "MUL", "DIV", "SIN", "EXP", "DUP", "SWAP", "DEL", "SQUARE", "POW", "TANH"]
    texts = random_gcl_programs(rng, 600, d, names)
    cl = []
    progs = [asm(t, cl)[0].copy() for t in texts]
    OP = colonies.OP
    out = []
    for tok in progs:
        k = int(rng.integers(8))
        i = int(rng.integers(len(tok)))
        if k == 0: tok[i] = colonies.token(int(rng.choice([0, 0x0C, 0x0F, 0x1F, 0x40, 0xFF])), 0)
        elif k == 1: tok[i] = colonies.token(OP["ADD"], 1 + int(rng.integers(5)))
        elif k == 2: tok[i] = colonies.token(OP["LOAD"], d + int(rng.integers(3)))
        elif k == 3: tok[i] = colonies.token(OP["CONST"], len(cl) + int(rng.integers(3)))
        elif k == 4: tok = np.delete(tok, i)
        elif k == 5: tok = np.insert(tok, i, tok[i])
        elif k == 6: tok = np.insert(tok, len(tok), colonies.token(OP["COPY"], int(rng.integers(32))))
        elif k == 7: tok = np.insert(tok, i, colonies.token(OP["PASTE"], int(rng.integers(34))))
        if len(tok) >= 1:
            out.append(tok.astype(np.int32))
    # and the limits of the stack: 32 terminals are a program, 33 are not
    ld = colonies.token(OP["LOAD"], 0)
    add = colonies.token(OP["ADD"])
    out.append(np.array([ld] * 32 + [add] * 31, np.int32))
    out.append(np.array([ld] * 33 + [add] * 32, np.int32))
    g, l, c = pack(out, cl)
    X, y = _cases(rng, 8, d)
    orc = oracle.evaluate(g, l, c, X, y, 1e-3)
    off = np.concatenate([[0], np.cumsum(l, dtype=np.int64)])
    n_bad = 0
    for p in range(len(l)):
        depth, slow, rec = api.beagle_debug_compile(g[off[p]:off[p + 1]], c, d, 2, 1, 1, 2048, 0)
        assert depth == orc["depth"][p], (p, depth, int(orc["depth"][p]))
        assert (depth == 0) == bool(orc["flags"][p] & oracle.FLAG_MALFORMED), p
        n_bad += depth == 0
    assert 0.3 * len(l) < n_bad < 0.9 * len(l)     # the corruptions bite, and some programs survive them
    assert orc["depth"][-2] == 32 and orc["depth"][-1] == 0


def test_debug_compile_argument_errors():
    import ctypes
    l = api.lib()
    tok = np.array([colonies.token(colonies.OP["LOAD"], 0)], np.int32)
    rec = np.zeros((4, 2), np.uint32)
    n, dep, sl = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
    def call(tokens=tok.ctypes.data, ln=1, d=1, S=0, kr=0, ku=0):
        return l.beagle_debug_compile(tokens, ln, None, 0, d, S, kr, ku, 2048, 0, rec.ctypes.data, ctypes.byref(n), ctypes.byref(dep), ctypes.byref(sl))
    assert call() == api.OK and dep.value == 1 and n.value == 1
    assert call(tokens=None) == api.ERR_INVALID_ARG
    assert call(ln=0) == api.ERR_INVALID_ARG and call(ln=513) == api.ERR_INVALID_ARG
    assert call(d=0) == api.ERR_INVALID_ARG and call(d=33) == api.ERR_INVALID_ARG
    assert call(S=32) == api.ERR_INVALID_ARG and call(kr=2) == api.ERR_INVALID_ARG and call(ku=2) == api.ERR_INVALID_ARG


# ---- the Std family's reward: the device's function, compiled for the host, against the oracle's, bit for bit -----------------
def _oracle_rewards(oracle, f, y, power, M):
    """reward(f[k], y[i]) for every pair of the two sweeps, from the oracle: programs 'CONST f[k]' on the one-case dataset y[i],
    tax 0, so that the fitness of a program is the reward of its one case."""
    tok = np.array([colonies.token(colonies.OP["CONST"], k) for k in range(len(f))], np.int32)
    lengths = np.ones(len(f), np.int32)
    out = np.empty((len(y), len(f)), np.float32)
    X = np.zeros((1, 1), np.float32)
    for i, yi in enumerate(y):
        r = oracle.evaluate_std(tok, lengths, f, X, np.array([yi], np.float32), power, M, 0.0, mode=1)
        out[i] = r["fitness"]
    return out


@pytest.mark.parametrize("fit,power", [(api.FIT_STD, 1), (api.FIT_STD_SQUARE, 2), (api.FIT_STD_CUBE, 3), (api.FIT_STD_HYPER, 8)])
def test_std_reward_of_the_device_is_the_oracles_bit_for_bit(oracle, fit, power):
    """Eq. 5 decides an integer by floating point, so both sides take the decision in fp32 in one stated order (R25).
    Here the device's own function (csrc/fit_std.cuh, host build) meets the oracle's on a sweep that has every branch: equal and
    opposite signs, zeros of both signs, denormals, huge and tiny ratios, ratios on both sides of the rounding boundaries and ties,
    infinities and NaN on either side."""
    rng = np.random.default_rng(500 + power)
    M = 10000.0
    special = np.array([0.0, -0.0, 1e-45, -1e-45, 1e-38, 3.4e38, -3.4e38, np.inf, -np.inf, np.nan, 1.0, -1.0, 0.5, 2.0, 3.0, -3.0], np.float32)
    mags = np.exp(rng.uniform(np.log(1e-6), np.log(1e6), 150)).astype(np.float32) * rng.choice([-1, 1], 150).astype(np.float32)
    # ratios whose M q^p is near k + 1/2: q = ((k + 1/2) / M)^(1/p) against a target of 1, and its neighbours in fp32
    k = rng.integers(0, 10000, 60).astype(np.float64)
    q = (((k + 0.5) / M) ** (1.0 / power)).astype(np.float32)
    near = np.concatenate([q, np.nextafter(q, np.float32(0)), np.nextafter(q, np.float32(2)), -q])
    f = np.concatenate([special, mags, near]).astype(np.float32)
    y = np.concatenate([special, np.array([1.0, -1.0, 7.25, -0.3], np.float32), mags[:12]]).astype(np.float32)
    want = _oracle_rewards(oracle, f, y, power, M)
    n_ties = 0
    for i, yi in enumerate(y):
        got = api.beagle_debug_std_reward(f, np.full(len(f), yi, np.float32), fit, M)
        assert np.array_equal(got.view(np.uint32), want[i].view(np.uint32)), \
            (float(yi), [(float(a), float(b), float(c)) for a, b, c in zip(f, got, want[i]) if b != c][:5])
        assert np.all(got == np.rint(got)) and np.all(np.abs(got) <= M)          # integers within [-M, M]
    # the sweep reaches every branch of Eq. 5
    allw = want.ravel()
    assert (allw == M).any() and (allw == -M).any() and (allw < 0).any() and (allw == 0).any()
    assert len(np.unique(allw)) > 300


def test_std_reward_argument_errors():
    one = np.zeros(1, np.float32)
    l = api.lib()
    assert l.beagle_debug_std_reward(one.ctypes.data, one.ctypes.data, 1, api.FIT_MSE, 1.0, one.ctypes.data) == api.ERR_INVALID_ARG
    assert l.beagle_debug_std_reward(one.ctypes.data, one.ctypes.data, 1, api.FIT_CORRELATION, 1.0, one.ctypes.data) == api.ERR_INVALID_ARG
    assert l.beagle_debug_std_reward(None, one.ctypes.data, 1, api.FIT_STD, 1.0, one.ctypes.data) == api.ERR_INVALID_ARG
    assert l.beagle_debug_std_reward(None, None, 0, api.FIT_STD, 1.0, None) == api.OK


# ---- k_compile's own walk (csrc/walk_body.inc: the source the kernel and beagle_debug_walk are both compiled from) ---------------
HOT = {colonies.OP[n] for n in ("CONST", "LOAD", "ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP")}
F1 = {colonies.OP[n] for n in ("DUP", "SWAP", "DEL", "SIGN", "SQUARE", "CUBE")}


def _check_walk(oracle, genomes, lengths, consts, X, y, tax, plans, run_machine=True):
    """Every program through the walk's host build, both instantiations, for each plan. The walk takes a program exactly when it is
    a well-formed program of its commands (the oracle's static check decides well-formed); what it takes it compiles to the records
    the general compiler emits (the two are different code: a table-driven loop and a switch), with the oracle's depth; the records
    compute the program (the micro-op machine against the oracle's fitness)."""
    d = X.shape[1]
    orc = oracle.evaluate(genomes, lengths, consts, X, y, tax)
    unsafe = sum(1 << j for j in range(d) if np.any(np.abs(X[:, j]) < EPS))
    off = np.concatenate([[0], np.cumsum(lengths, dtype=np.int64)])
    taken_n = {False: 0, True: 0}
    for S_T, k_rcp, k_un in plans:
        fit = np.full(len(lengths), np.nan, np.float32)
        ran = np.zeros(len(lengths), bool)
        for p in range(len(lengths)):
            tok = genomes[off[p]:off[p + 1]]
            ops = set((tok.view(np.uint32) & 0xFF).tolist())
            wellformed = not (orc["flags"][p] & oracle.FLAG_MALFORMED)
            gdepth, gslow, grec = api.beagle_debug_compile(tok, consts, d, S_T, k_rcp, k_un, 2048, unsafe)
            # 2: the stack commands' vote passed at every token (neighbouring lanes); + (k << 8): a neighbouring lane's program is k longer
            for f1 in (0, 1, 2, 1 | 3 << 8, 0 | 17 << 8, 2 | 400 << 8):
                taken, depth, used, rec = api.beagle_debug_walk(tok, consts, d, S_T, k_rcp, k_un, 2048, unsafe, f1=f1)
                mine = ops <= (HOT | F1 if f1 & 0xff else HOT)
                assert taken == (wellformed and mine), (p, f1, taken, wellformed, sorted(ops))
                if not taken:
                    continue
                taken_n[bool(f1)] += f1 < 2
                assert depth == orc["depth"][p] and not gslow, (p, f1, depth, int(orc["depth"][p]))
                assert used == (bool(f1 & 0xff) and bool(ops & F1)), (p, f1, used)
                assert np.array_equal(rec, grec), (p, f1, rec.tolist(), grec.tolist())
            if run_machine and wellformed and ops <= HOT | F1:
                _, _, _, rec = api.beagle_debug_walk(tok, consts, d, S_T, k_rcp, k_un, 2048, unsafe, f1=True)
                fit[p] = _fitness(run_records(rec, X, d, S_T, k_rcp, k_un, 2048), y, tax, len(tok))
                ran[p] = True
        if run_machine:
            sel = np.nonzero(ran)[0]
            sub = {k: orc[k][sel] for k in ("fitness", "bound", "flags", "depth")}
            rep = parity.compare(fit[sel], sub)
            assert len(rep["bad"]) == 0, parity.describe(rep, fit[sel], sub)
    return taken_n


def test_walk_takes_and_compiles_the_hot_path_colonies(oracle):
    for number, P in ((1, 300), (2, 200), (3, 300), (4, 200), (5, 400)):
        cfg = colonies.CONFIGS[number]
        g, l, c = colonies.generate_programs(cfg, P)
        X, y, _ = colonies.make_dataset(cfg)
        taken = _check_walk(oracle, g, l, c, X[:48], y[:48], cfg.tax, PLANS if number == 5 else PLANS[:2])
        assert taken[False] == taken[True] == P * (len(PLANS) if number == 5 else 2)      # every program of the five configs is the walk's


def test_walk_f1_instantiation_takes_the_stack_commands(oracle):
    cfg = colonies.CONFIGS[3]
    g, l, c = colonies.generate_programs(cfg, 400, gcl_mix="f1")
    X, y, _ = colonies.make_dataset(cfg)
    taken = _check_walk(oracle, g, l, c, X[:40], y[:40], cfg.tax, PLANS[:3])
    assert taken[True] == 400 * 3 and taken[False] < 0.3 * 400 * 3          # 88 % of the f1 mix's programs use one of the six
    rng = np.random.default_rng(77)
    texts = random_gcl_programs(rng, 500, 3, ["ADD", "SUB", "MUL", "DIV", "SIN", "LOG", "EXP", "DUP", "SWAP", "DEL", "SIGN", "SQUARE", "CUBE"])
    cl = []
    progs = [asm(t, cl)[0] for t in texts]
    gg, ll, cc = pack(progs, cl)
    Xr, yr = _cases(rng, 40, 3, zero_in=0)
    _check_walk(oracle, gg, ll, cc, Xr, yr, 1e-3, PLANS)


def test_walk_turns_down_exactly_what_is_not_its_own(oracle):
    """Programs of the whole language and corrupted ones: the walk takes the well-formed programs of its commands and nothing else
    (a program it turns down is looked at again by the general compiler on the device: nothing is lost, only time)."""
    rng = np.random.default_rng(4242)
    d = 4
    names = ["ADD", "SUB", "MUL", "DIV", "SIN", "EXP", "SQRT", "DUP", "SWAP", "DEL", "SQUARE", "POW", "TANH"]
    texts = random_gcl_programs(rng, 500, d, names) + random_gcl_programs(rng, 300, d, ["ADD", "SUB", "MUL", "DIV", "COS", "LOG"])
    cl = []
    progs = [asm(t, cl)[0].copy() for t in texts]
    OP = colonies.OP
    out = []
    for tok in progs:
        k = int(rng.integers(10))                  # 0-5: one corruption; 6-9: left alone
        i = int(rng.integers(len(tok)))
        if k == 0: tok[i] = colonies.token(int(rng.choice([0, 0x0C, 0x0F, 0x13, 0x1F, 0x40, 0xFF])), 0)
        elif k == 1: tok[i] = colonies.token(int(tok[i]) & 0xFF, 1 + int(rng.integers(5))) if (int(tok[i]) & 0xFF) > 2 else tok[i]
        elif k == 2: tok[i] = colonies.token(OP["LOAD"], d + int(rng.integers(3)))
        elif k == 3: tok[i] = colonies.token(OP["CONST"], len(cl) + int(rng.integers(3)))
        elif k == 4: tok = np.delete(tok, i)
        elif k == 5: tok = np.insert(tok, i, tok[i])
        if len(tok) >= 1:
            out.append(tok.astype(np.int32))
    ld, add = colonies.token(OP["LOAD"], 0), colonies.token(OP["ADD"])
    out.append(np.array([ld] * 32 + [add] * 31, np.int32))          # the deepest stack that is a program
    out.append(np.array([ld] * 33 + [add] * 32, np.int32))          # one more is not
    out.append(np.array([ld] * 256 + [add] * 255, np.int32)[:512])  # (and a long one that overflows early)
    for text in ("x0 DEL", "x0 x1 ADD DEL", "x0 x1 DEL DEL", "x0 DUP DEL DEL", "x0 DEL x1"):      # an empty stack at the end is not a program; in between it is
        out.append(asm(text)[0])
    g, l, c = pack(out, cl)
    X, y = _cases(rng, 8, d)
    taken = _check_walk(oracle, g, l, c, X, y, 1e-3, [(2, 1, 1)], run_machine=False)
    assert 0.15 * len(l) < taken[False] < taken[True] < 0.85 * len(l)


def test_random_token_streams_agree_with_the_oracles_static_check(oracle):
    """Breadth: random words and loosely plausible programs of every length class (what tests/fuzz_device_compiler_asan.py sends through
    the sanitizer, a smaller dose): the general compiler's verdict (malformed or depth) is the oracle's on every one, the walk takes
    exactly the well-formed ones made of its commands and emits the general compiler's records, never more records than tokens."""
    rng = np.random.default_rng(20260)
    d, n_consts = 6, 16
    consts = rng.uniform(-3, 3, n_consts).astype(np.float32)
    valid_ops = np.array([1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11] + list(range(0x10, 0x1F)), np.uint32)
    progs = []
    for k in range(2500):
        L = int(rng.choice([1, 2, 3, 5, 8, 13, 40, 100, 255, 511, 512])) if rng.random() < 0.3 else int(rng.integers(1, 60))
        if k % 5 == 0:                             # random words (an opcode byte in range now and then)
            tok = rng.integers(0, 2**32, L, dtype=np.uint64).astype(np.uint32)
            tok = np.where(rng.random(L) < 0.5, (tok & 0xFFFFFF00) | rng.choice(valid_ops, L), tok).astype(np.uint32)
        else:                                      # plausible: stack-aware choice of commands, stray arguments and opcodes
            tok = np.empty(L, np.uint32)
            depth = 0
            for t in range(L):
                if depth < 2 or rng.random() < 0.45:
                    op = 1 if rng.random() < 0.3 else 2
                    arg = int(rng.integers(0, (n_consts if op == 1 else d) + (1 if rng.random() < 0.02 else 0)))
                    depth += 1
                else:
                    op = int(rng.choice(valid_ops))
                    arg = 0 if rng.random() < 0.98 else int(rng.integers(0, 40))
                    depth += {3: -1, 4: -1, 5: -1, 6: -1, 0x13: -1, 0x12: -1, 0x10: 1, 0x1E: 1}.get(op, 0)
                tok[t] = (arg << 8) | op
        progs.append(tok.view(np.int32))
    g, l, c = pack(progs, consts)
    X = rng.uniform(-2, 2, (1, d)).astype(np.float32)
    orc = oracle.evaluate(g, l, c, X, np.zeros(1, np.float32), 0.0)
    n_ok = n_taken = 0
    for p, tok in enumerate(progs):
        ops = set((tok.view(np.uint32) & 0xFF).tolist())
        wellformed = not (orc["flags"][p] & oracle.FLAG_MALFORMED)
        gdepth, gslow, grec = api.beagle_debug_compile(tok, c, d, 2, 3, 2, 2048, 0b101)
        assert gdepth == orc["depth"][p] and (gdepth == 0) == (not wellformed), (p, gdepth, int(orc["depth"][p]))
        assert len(grec) <= len(tok)
        n_ok += wellformed
        for f1 in (False, True):
            taken, depth, used, rec = api.beagle_debug_walk(tok, c, d, 2, 3, 2, 2048, 0b101, f1=f1)
            assert taken == (wellformed and ops <= (HOT | F1 if f1 else HOT)), (p, f1)
            if taken:
                n_taken += 1
                assert depth == gdepth and np.array_equal(rec, grec), (p, f1)
    assert 0.2 * len(progs) < n_ok < 0.9 * len(progs) and n_taken > 200
