"""-m gpu: edge cases, in-band error reporting and self-consistency of the CUDA path (SURVEY.md §4
items 2 and 4): bitwise determinism, permutation/duplication/chunking invariance, malformed programs,
limits, exact length tax, exact power-of-two scaling, and bit-exact per-case outputs for programs
made of correctly rounded commands only.
"""
import ctypes

import numpy as np
import pytest

from paper_2607_06731_b200 import colonies
from paper_2607_06731_b200.colonies import OP, token
from tests import parity
from tests.util import asm, pack, random_gcl_programs

pytestmark = pytest.mark.gpu

QNAN = np.uint32(0x7FC00000)


def _bits(a):
    return np.asarray(a, np.float32).view(np.uint32)


def _cases(N=64, d=2, seed=3):
    rng = np.random.default_rng(seed)
    X = (rng.integers(-2048, 2048, (N, d)) / 2048.0).astype(np.float32)   # 12 significant bits
    return X


def test_empty_population():
    import torch
    from paper_2607_06731_b200 import api
    X = torch.zeros((4, 1), device="cuda")
    y = torch.zeros(4, device="cuda")
    api.beagle_eval(None, None, 0, None, 0, X, y, 4, 1, 0.0, None, 0)
    assert api.beagle_last_launch_count() == 0


def test_argument_errors():
    import torch
    from paper_2607_06731_b200 import api
    l = api.lib()
    X = torch.zeros((4, 1), device="cuda"); y = torch.zeros(4, device="cuda")
    g = torch.zeros(4, dtype=torch.int32, device="cuda"); ln = torch.ones(4, dtype=torch.int32, device="cuda")
    out = torch.zeros(4, device="cuda")
    def call(**kw):
        a = dict(genomes=g.data_ptr(), lengths=ln.data_ptr(), P=4, consts=None, n_consts=0, X=X.data_ptr(),
                 y=y.data_ptr(), N=4, d=1, tax=0.0, out=out.data_ptr())
        a.update(kw)
        return l.beagle_eval(a["genomes"], a["lengths"], a["P"], a["consts"], a["n_consts"], a["X"], a["y"],
                             a["N"], a["d"], a["tax"], a["out"], None)
    assert call() == api.OK
    assert call(P=-1) == api.ERR_INVALID_ARG
    assert call(N=0) == api.ERR_INVALID_ARG
    assert call(N=1025) == api.ERR_INVALID_ARG
    assert call(d=0) == api.ERR_INVALID_ARG
    assert call(d=33) == api.ERR_INVALID_ARG
    assert call(n_consts=1) == api.ERR_INVALID_ARG            # consts NULL with n_consts > 0
    assert call(n_consts=(1 << 24) + 1, consts=g.data_ptr()) == api.ERR_INVALID_ARG
    assert call(genomes=None) == api.ERR_INVALID_ARG
    assert call(out=None) == api.ERR_INVALID_ARG
    assert l.beagle_eval_chunked(None, None, 4, None, 0, X.data_ptr(), y.data_ptr(), 4, 1, 0.0,
                                 out.data_ptr(), 1 << 20, None) == api.ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert "invalid" in api.beagle_status_string(api.ERR_INVALID_ARG)


def test_malformed_programs_give_canonical_nan(oracle):
    """DESIGN.md D3 / R9-R10: every kind of malformed program, mixed with valid ones."""
    from tests.gpu_util import gpu_eval
    X = _cases(64, 2)
    y = (X[:, 0] * X[:, 0]).astype(np.float32)
    consts = [np.float32(1.5)]
    good = asm("x0 x0 MUL")[0]
    progs = [
        good,
        np.array([token(OP["ADD"])], np.int32),                               # pops an empty stack
        np.array([token(OP["LOAD"], 0), token(OP["ADD"])], np.int32),         # binary on depth 1
        np.array([token(OP["SIN"])], np.int32),                               # unary on depth 0
        np.array([token(0)], np.int32),                                       # opcode 0
        np.array([token(0x10)], np.int32),                                    # reserved opcode (DUP)
        np.array([token(0xFF, 5)], np.int32),                                 # unknown opcode
        np.array([token(OP["LOAD"], 2)], np.int32),                           # variable >= d
        np.array([token(OP["CONST"], 1)], np.int32),                          # constant >= n_consts
        np.array([token(OP["LOAD"], 0), token(OP["SIN"], 1)], np.int32),      # operator with arg != 0
        np.array([token(OP["LOAD"], 0)] * 33 + [token(OP["ADD"])] * 32, np.int32),   # depth 33
        good,
        np.array([token(OP["LOAD"], 0)] * 32 + [token(OP["ADD"])] * 31, np.int32),   # depth 32: fine
        np.array([token(OP["LOAD"], 0), token(OP["LOAD"], 1)], np.int32),     # final depth 2: fine (R8)
    ]
    g, l, c = pack(progs, consts)
    fit = gpu_eval(g, l, c, X, y, 0.25)
    orc = oracle.evaluate(g, l, c, X, y, 0.25)
    assert np.all(_bits(fit[1:11]) == QNAN)
    assert np.all((orc["flags"][1:11] & 1) == 1)
    rep = parity.compare(fit, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, fit, orc)
    assert _bits(fit[0]) == _bits(np.float32(0.75)) and _bits(fit[11]) == _bits(np.float32(0.75))


def test_out_of_range_lengths_count_as_zero_words(oracle):
    from tests.gpu_util import gpu_eval
    X = _cases(32, 2)
    y = X[:, 1].copy()
    p = asm("x1")[0]
    genomes = np.concatenate([p, p, p]).astype(np.int32)
    lengths = np.array([1, 0, -7, 513, 1, 1 << 30, 1], np.int32)
    fit = gpu_eval(genomes, lengths, np.zeros(0, np.float32), X, y, 0.5)
    assert np.all(_bits(fit[[1, 2, 3, 5]]) == QNAN)
    assert np.all(fit[[0, 4, 6]] == np.float32(0.5))
    orc = oracle.evaluate(genomes, lengths, np.zeros(0, np.float32), X, y, 0.5)
    assert np.array_equal(_bits(fit), _bits(orc["fitness"]))


def test_length_tax_exact():
    """R15: a program with MSE exactly 0 returns (float)(tax*L) bit-exactly, for every length class."""
    from tests.gpu_util import gpu_eval
    X = _cases(96, 2)
    y = X[:, 0].copy()
    progs, consts = [], [np.float32(0.0)]
    for extra in (0, 1, 5, 30, 100, 255):
        t = [token(OP["LOAD"], 0)] + [token(OP["CONST"], 0), token(OP["ADD"])] * extra
        progs.append(np.array(t, np.int32))
    progs.append(np.array([token(OP["LOAD"], 0)] + [token(OP["CONST"], 0)] * 20 + [token(OP["ADD"])] * 20, np.int32))
    g, l, c = pack(progs, consts)
    for tax in (0.001, 0.3, 7.0):
        fit = gpu_eval(g, l, c, X, y, tax)
        want = (np.float32(tax) * l.astype(np.float32)).astype(np.float32)
        assert np.array_equal(_bits(fit), _bits(want)), (fit, want)


def test_power_of_two_scaling_exact():
    """Pin P9 on the GPU: `A 2 MUL` against 2y has exactly 4x the MSE of `A` against y."""
    from tests.gpu_util import gpu_eval
    col = colonies.make_colony(1)
    consts = list(col.consts)
    two = len(consts); consts.append(np.float32(2.0))
    off = np.concatenate([[0], np.cumsum(col.lengths)])
    progs2 = [np.concatenate([col.genomes[off[p]:off[p + 1]],
                              np.array([token(OP["CONST"], two), token(OP["MUL"])], np.int32)]) for p in range(col.P)]
    g2, l2, c2 = pack(progs2, consts)
    f1 = gpu_eval(col.genomes, col.lengths, c2, col.X, col.y, 0.0)
    f2 = gpu_eval(g2, l2, c2, col.X, (2 * col.y).astype(np.float32), 0.0)
    ok = np.isfinite(f1) & np.isfinite(f2) & (f1 > 1e-30) & (f1 < 1e30)
    assert ok.sum() > 900
    assert np.array_equal(_bits(f2[ok]), _bits((4 * f1[ok]).astype(np.float32)))
    assert np.array_equal(np.isnan(f1), np.isnan(f2))


def test_determinism_permutation_duplication():
    from tests.gpu_util import gpu_eval
    col = colonies.make_colony(5, 6000)
    f1 = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    f2 = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    assert np.array_equal(_bits(f1), _bits(f2))
    off = np.concatenate([[0], np.cumsum(col.lengths, dtype=np.int64)])
    rng = np.random.default_rng(11)
    perm = rng.permutation(col.P)
    perm = np.concatenate([perm, perm[:777]])                     # duplicates too
    gp = np.concatenate([col.genomes[off[p]:off[p + 1]] for p in perm])
    fp = gpu_eval(gp, col.lengths[perm], col.consts, col.X, col.y, col.tax)
    assert np.array_equal(_bits(fp), _bits(f1[perm]))


def test_blockwise_baseline_bitwise_equal():
    from tests.gpu_util import gpu_eval
    col = colonies.make_colony(2, 3000)
    for N in (1024, 517):
        a = gpu_eval(col.genomes, col.lengths, col.consts, col.X[:N], col.y[:N], col.tax)
        b = gpu_eval(col.genomes, col.lengths, col.consts, col.X[:N], col.y[:N], col.tax, fn="beagle_eval_blockwise")
        assert np.array_equal(_bits(a), _bits(b))


def test_grouped_record_copies_bitwise_equal_blockwise():
    """A colony large enough for the interpreter's warps to take several entries per visit to the work queue, so
    that one bulk copy brings a group of neighbouring programs (eval_kernel.inc; the small cases above never form
    a group). Malformed programs are sprinkled in: they end a group. Every fitness bit-identical to the blockwise
    kernel's (one block per individual, no groups), whose parity with the oracle test_gpu_parity.py checks."""
    from tests.gpu_util import gpu_eval
    col = colonies.make_colony(3, 300000)
    genomes = col.genomes.copy()
    off = np.concatenate([[0], np.cumsum(col.lengths, dtype=np.int64)])
    rng = np.random.default_rng(5)
    bad = rng.choice(col.P, 3000, replace=False)
    genomes[off[bad]] = token(OP["ADD"], 0)                         # an operator on an empty stack
    N = 80                                                         # (a ragged pass keeps the blockwise run short)
    a = gpu_eval(genomes, col.lengths, col.consts, col.X[:N], col.y[:N], col.tax)
    b = gpu_eval(genomes, col.lengths, col.consts, col.X[:N], col.y[:N], col.tax, fn="beagle_eval_blockwise")
    assert np.array_equal(_bits(a), _bits(b))
    assert np.all(_bits(a[bad]) == QNAN)
    assert np.isfinite(a).sum() > 0.9 * (col.P - len(bad))


@pytest.mark.parametrize("budget_frac,pinned", [(2.5, True), (0.37, True), (0.11, False), (0.013, True)])
def test_chunked_bitwise_equals_unchunked(budget_frac, pinned):
    from tests.gpu_util import gpu_eval, gpu_eval_chunked
    col = colonies.make_colony(5, 20000)
    ref = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    budget = max(int(col.T * 4 * budget_frac), 2 * 4 * 513 + 64)
    out = gpu_eval_chunked(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, budget, pinned)
    assert np.array_equal(_bits(out), _bits(ref))


def test_chunked_minimum_budget_and_errors():
    import torch
    from paper_2607_06731_b200 import api
    from tests.gpu_util import gpu_eval, gpu_eval_chunked
    col = colonies.make_colony(5, 300)
    ref = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    out = gpu_eval_chunked(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, 2 * 4 * 513 + 512)
    assert np.array_equal(_bits(out), _bits(ref))
    with pytest.raises(api.BeagleError):
        gpu_eval_chunked(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, 1000)
    torch.cuda.synchronize()


def test_outputs_bit_exact_for_correctly_rounded_commands(oracle):
    """SURVEY.md §8(c) cross-check: for programs made of ADD, SUB, MUL only the fp32-mirror oracle
    (fp64 result of two fp32 operands, rounded to fp32 = the correctly rounded fp32 result) must
    equal the GPU's per-case outputs bit for bit."""
    from tests.gpu_util import gpu_outputs
    cfg = colonies.CONFIGS[3]
    tokens, lengths, consts = colonies.generate_programs(cfg, 30000)
    X, y, _ = colonies.make_dataset(cfg)
    off = np.concatenate([[0], np.cumsum(lengths, dtype=np.int64)])
    ops = tokens & 0xFF
    bad = (ops >= OP["DIV"]).astype(np.int64)
    nbad = np.add.reduceat(bad, off[:-1])
    sel = np.nonzero(nbad == 0)[0][:1500]
    assert len(sel) > 500
    g = np.concatenate([tokens[off[p]:off[p + 1]] for p in sel])
    l = lengths[sel]
    out = gpu_outputs(g, l, consts, X)
    orc = oracle.evaluate(g, l, consts, X, y, 0.0, contract_=oracle.contract(oracle.CONTRACT_IEEE), mode=1,
                          want_outputs=True)
    want = orc["outputs"].astype(np.float32)
    # denormal results are not flushed by IEEE add/sub/mul; compare every bit (NaN payloads aside)
    same = (_bits(out) == _bits(want)) | (np.isnan(out) & np.isnan(want))
    assert np.all(same), np.argwhere(~same)[:5]


def test_limits_and_exports():
    from paper_2607_06731_b200 import api
    lim = api.beagle_limits()
    assert lim == dict(max_len=512, max_stack=32, max_n=1024, max_d=32)


@pytest.mark.parametrize("N", [512, 700, 1024])
def test_division_by_variable_reciprocal_rows(oracle, N):
    """Division by a variable runs as a multiplication by a staged reciprocal row only when no case of that
    variable is protected. x0 never triggers the protection; x1 does, in one case only (the
    last one, also inside a ragged tail); x2 is exactly zero everywhere. Outputs must be bit-identical to the
    blockwise kernel (the plain per-case division) and agree with the oracle."""
    from tests.gpu_util import gpu_eval, gpu_outputs
    rng = np.random.default_rng(11)
    d = 3
    X = rng.uniform(0.5, 4.0, (N, d)).astype(np.float32)
    X[N - 1, 1] = np.float32(3e-7)
    X[:, 2] = 0.0
    y = (X[:, 0] / 3.0).astype(np.float32)
    consts = []
    texts = ["x1 x0 DIV", "x0 x1 DIV", "x0 x2 DIV", "x0 x0 MUL x0 DIV", "x0 x0 MUL x1 DIV", "x1 SIN x2 DIV",
             "x0 x1 ADD x0 x1 MUL DIV x0 DIV", "2.5 x0 DIV", "x0 2.5 DIV x1 DIV", "x0 COS x0 x0 DIV x1 x0 DIV ADD SUB"]
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts)
    a = gpu_eval(g, l, c, X, y, 0.001)
    b = gpu_eval(g, l, c, X, y, 0.001, fn="beagle_eval_blockwise")
    assert np.array_equal(_bits(a), _bits(b))
    orc = oracle.evaluate(g, l, c, X, y, 0.001)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    out = gpu_outputs(g, l, c, X)
    assert np.all(out[1, N - 1] == np.float32(1.0))          # x0 / 3e-7 is protected: 1
    assert np.all(out[2] == np.float32(1.0))                 # x0 / 0 is protected everywhere


@pytest.mark.parametrize("N,d", [(512, 32), (1024, 16), (512, 20), (1000, 12)])
def test_full_tensor_memory_and_deep_stacks(oracle, N, d):
    """Shapes at the edge of the tensor-memory plan: the variable block fills all 32 rows
    (N <= 512 with d = 32, N > 512 with d = 16: no slot row at all, every push spills to local memory), or
    leaves only a few. Programs: right-deep chains that keep up to 31 computed values waiting, unary commands
    and divisions on every variable (staged rows in shared memory, in global memory, or none)."""
    from tests.gpu_util import gpu_eval
    rng = np.random.default_rng(5)
    X = rng.uniform(0.5, 3.0, (N, d)).astype(np.float32)
    y = np.sin(X[:, 0]).astype(np.float32)
    consts, progs = [], []
    for depth in (1, 2, 3, 4, 5, 8, 16, 30):
        # (x0*x1) (x1*x2) ... pushed one after the other, then folded from the right with alternating commands
        parts = [f"x{k % d} x{(k + 1) % d} MUL" for k in range(depth + 1)]
        ops = " ".join(("ADD", "SUB", "MUL", "DIV")[k % 4] for k in range(depth))
        progs.append(asm(" ".join(parts) + " " + ops, consts)[0])
    for j in range(d):
        progs.append(asm(f"x{j} SIN x{j} COS ADD x{j} LOG x{j} SQRT MUL SUB x{j} 0.1 MUL EXP ADD x{(j + 1) % d} DIV", consts)[0])
    g, l, c = pack(progs, consts)
    a = gpu_eval(g, l, c, X, y, 0.001)
    b = gpu_eval(g, l, c, X, y, 0.001, fn="beagle_eval_blockwise")
    assert np.array_equal(_bits(a), _bits(b))
    orc = oracle.evaluate(g, l, c, X, y, 0.001)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    assert rep["malformed"] == 0


@pytest.mark.parametrize("N,d", [(96, 2), (1024, 16)])
def test_every_operand_kind_combination(oracle, N, d):
    """Every case of the compiler's decision table: each binary command with each pair of operand
    kinds (variable, constant, tiny constant, computed value), each unary command on each kind, alone and with a
    computed value waiting underneath (the push entries; with d = 16, N = 1024 no slot row exists and every push
    goes to local memory). Bit-identical to the blockwise kernel and within the parity rule of the oracle."""
    from tests.gpu_util import gpu_eval
    rng = np.random.default_rng(9)
    X = rng.uniform(0.5, 3.0, (N, d)).astype(np.float32)
    X[0, 1] = 0.0                                           # x1 triggers the division protection in one case
    y = np.cos(X[:, 0]).astype(np.float32)
    kinds = {"x": "x0", "y": "x1", "c": "1.75", "t": "3e-7", "R": "x0 x1 ADD", "S": "x1 x0 SUB"}
    consts, progs = [], []
    bodies = []
    for op in ("ADD", "SUB", "MUL", "DIV"):
        for a in kinds.values():
            for b in kinds.values():
                bodies.append(f"{a} {b} {op}")
    for op in ("SIN", "COS", "LOG", "SQRT", "EXP"):
        for a in kinds.values():
            bodies.append(f"{a} {op}")
    for body in bodies:
        progs.append(asm(body, consts)[0])
        progs.append(asm(f"x1 SIN {body} ADD", consts)[0])                       # one value waiting
        progs.append(asm(f"x0 COS x1 SIN {body} MUL SUB", consts)[0])            # two values waiting
    g, l, c = pack(progs, consts)
    a = gpu_eval(g, l, c, X, y, 0.001)
    b = gpu_eval(g, l, c, X, y, 0.001, fn="beagle_eval_blockwise")
    assert np.array_equal(_bits(a), _bits(b))
    orc = oracle.evaluate(g, l, c, X, y, 0.001)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    assert rep["malformed"] == 0


@pytest.mark.parametrize("N,d", [(512, 3), (1024, 9), (200, 16)])
def test_stack_commands_and_exact_unaries(oracle, N, d):
    """DUP SWAP DEL SIGN SQUARE CUBE (Table 3): random programs mixing them with the eleven
    hot-path commands, and the paper's two printed genomes verbatim: bit-identical to the blockwise kernel, within
    the parity rule of the oracle; programs of + - * SIGN SQUARE CUBE and stack commands only are bit-exact per case."""
    from tests.gpu_util import gpu_eval, gpu_outputs
    rng = np.random.default_rng(21)
    X = rng.uniform(-2, 2, (N, d)).astype(np.float32)
    y = (X[:, 0] * X[:, 1]).astype(np.float32)
    names = ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP", "SIGN", "SQUARE", "CUBE", "DUP", "SWAP", "DEL",
             "CBRT", "TAN", "ARCSIN", "ARCCOS", "ARCTAN", "TANH", "POW"]
    texts = random_gcl_programs(rng, 600, d, names)
    texts += ["0 -9.280686 8.983309 ADD DEL x1 ADD DUP MUL x0 DUP ADD DUP ADD x2 MUL SUB SQRT x1 SUB x0 DIV 0.5 MUL",
              "x2 x0 MUL -2 MUL DUP ADD 3 4 SUB 2.7182817 SUB DUP DIV DEL x1 SQUARE ADD SQRT x1 SUB x0 DIV 0.5 MUL"]
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts)
    a = gpu_eval(g, l, c, X, y, 0.001)
    b = gpu_eval(g, l, c, X, y, 0.001, fn="beagle_eval_blockwise")
    assert np.array_equal(_bits(a), _bits(b))
    orc = oracle.evaluate(g, l, c, X, y, 0.001)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    assert rep["malformed"] == 0 and rep["strict"] > 100
    # correctly rounded commands only: per-case outputs equal the oracle's fp32 mirror bit for bit
    exact = random_gcl_programs(rng, 200, d, ["ADD", "SUB", "MUL", "SIGN", "SQUARE", "CUBE", "DUP", "SWAP", "DEL"])
    consts2 = []
    progs2 = [asm(t, consts2)[0] for t in exact]
    g2, l2, c2 = pack(progs2, consts2)
    out = gpu_outputs(g2, l2, c2, X)
    mir = oracle.evaluate(g2, l2, c2, X, y, 0.0, mode=1, want_outputs=True, contract_=oracle.contract(oracle.CONTRACT_IEEE))
    want = mir["outputs"].astype(np.float32)
    same = (out.view(np.uint32) == want.view(np.uint32)) | (np.isnan(out) & np.isnan(want)) | ((out == 0) & (want == 0))
    assert np.all(same)


def test_stack_command_malformed_programs(oracle):
    from tests.gpu_util import gpu_eval
    T = token
    x0 = T(OP["LOAD"], 0)
    progs = [np.array([T(OP["DUP"])], np.int32), np.array([x0, T(OP["SWAP"])], np.int32),
             np.array([x0, T(OP["DEL"])], np.int32), np.array([x0] + [T(OP["DUP"])] * 32, np.int32),
             np.array([x0, T(OP["POW"])], np.int32), np.array([x0, T(OP["SQUARE"], 3)], np.int32),   # POW needs two
             np.array([x0] + [T(OP["DUP"])] * 31 + [T(OP["ADD"])] * 31, np.int32),      # well-formed: depth 32
             np.array([x0, T(OP["DEL"]), x0, T(OP["CUBE"])], np.int32)]                 # well-formed
    g, l, c = pack(progs, np.zeros(1, np.float32))
    X = np.full((64, 1), 2.0, np.float32); y = np.zeros(64, np.float32)
    a = gpu_eval(g, l, c, X, y, 0.0)
    assert np.all(_bits(a[:6]) == QNAN)
    assert a[6] == np.float32(64.0 ** 2) and a[7] == np.float32(64.0)
    orc = oracle.evaluate(g, l, c, X, y, 0.0)
    assert len(parity.compare(a, orc)["bad"]) == 0


def _with_variables(rng, text, d):
    """Wrap a well-formed postfix text in COPY/PASTE pairs: some sub-results are copied to a variable
    and pasted back later; every COPY has its PASTE, no variable is copied to twice while it holds a value."""
    toks = text.split()
    out, live, free = [], [], list(rng.permutation(32))
    depth = 0
    for t in toks:
        out.append(t)
        depth += {"ADD": -1, "SUB": -1, "MUL": -1, "DIV": -1, "POW": -1, "DEL": -1, "DUP": 1}.get(t, 0 if t.isalpha() else 1)
        r = rng.random()
        if depth < 1 or depth > 30:
            continue
        if r < 0.15 and free:
            k = int(free.pop()); live.append(k); out.append(f"COPY@{k}")
        elif r < 0.30 and live:
            k = live.pop(int(rng.integers(len(live)))); free.append(k)
            out += [f"PASTE@{k}", ["ADD", "MUL", "SUB"][int(rng.integers(3))]]
    for k in live:
        out += [f"PASTE@{k}", "ADD"]
    return " ".join(out)


def test_copy_paste_variables(oracle):
    """COPY / PASTE: identities bit for bit, random programs with pairs against the
    oracle and the blockwise kernel, and the malformed cases of the pairing rule."""
    from tests.gpu_util import gpu_eval, gpu_outputs
    rng = np.random.default_rng(33)
    N, d = 700, 4
    X = rng.uniform(-2, 2, (N, d)).astype(np.float32)
    y = (X[:, 0] - X[:, 2]).astype(np.float32)
    consts = []
    pairs = [("x0 COPY@3 DEL x1 PASTE@3 SUB", "x1 x0 SUB"),
             ("x0 SIN COPY@31 x1 MUL PASTE@31 DIV", "x0 SIN x1 MUL x0 SIN DIV"),
             ("x2 COPY@0 PASTE@0 MUL COPY@0 PASTE@0 ADD", "x2 x2 MUL DUP ADD"),
             ("x0 COPY@1 x1 COPY@2 ADD PASTE@1 PASTE@2 DIV MUL", "x0 x1 ADD x0 x1 DIV MUL")]
    progs = [asm(t, consts)[0] for pr in pairs for t in pr]
    g, l, c = pack(progs, consts)
    out = gpu_outputs(g, l, c, X)
    for i in range(len(pairs)):
        assert np.array_equal(out[2 * i].view(np.uint32), out[2 * i + 1].view(np.uint32)), pairs[i]
    names = ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "SQRT", "EXP", "SQUARE", "DUP", "SWAP", "DEL", "TANH"]
    texts = [_with_variables(rng, t, d) for t in random_gcl_programs(rng, 400, d, names)]
    texts = [t for t in texts if len(t.split()) <= 200]
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts)
    a = gpu_eval(g, l, c, X, y, 0.001)
    b = gpu_eval(g, l, c, X, y, 0.001, fn="beagle_eval_blockwise")
    assert np.array_equal(_bits(a), _bits(b))
    orc = oracle.evaluate(g, l, c, X, y, 0.001)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
    assert rep["malformed"] == 0 and rep["strict"] > 50
    T = token
    x0 = T(OP["LOAD"], 0)
    bad = [[T(OP["PASTE"], 0)], [x0, T(OP["COPY"], 0)], [x0, T(OP["COPY"], 1), T(OP["COPY"], 1), T(OP["PASTE"], 1), T(OP["ADD"])],
           [x0, T(OP["COPY"], 32), T(OP["PASTE"], 32), T(OP["ADD"])], [x0, T(OP["COPY"], 2), T(OP["PASTE"], 3), T(OP["ADD"])],
           [T(OP["COPY"], 0), x0, T(OP["PASTE"], 0), T(OP["ADD"])],
           [x0, T(OP["COPY"], 5)] + [T(OP["DUP"])] * 31 + [T(OP["PASTE"], 5)]]                       # PASTE overflows the stack
    good = [[x0, T(OP["COPY"], 5)] + [T(OP["DUP"])] * 30 + [T(OP["PASTE"], 5)] + [T(OP["ADD"])] * 31]
    progs = [np.array(q, np.int32) for q in bad + good]
    g, l, c = pack(progs, np.zeros(1, np.float32))
    X1 = np.full((64, 1), 2.0, np.float32); y1 = np.zeros(64, np.float32)
    a = gpu_eval(g, l, c, X1, y1, 0.0)
    assert np.all(_bits(a[:len(bad)]) == QNAN) and a[len(bad)] == np.float32(64.0 ** 2)
    orc = oracle.evaluate(g, l, c, X1, y1, 0.0)
    assert len(parity.compare(a, orc)["bad"]) == 0


def test_eval_is_cuda_graph_capturable(oracle):
    """After beagle_reserve the call allocates nothing and never synchronises, so a generation loop can capture it in a
    CUDA graph (launch-bound small colonies); a replay gives the bits of a plain call, also after the inputs changed."""
    import torch
    from paper_2607_06731_b200 import api, colonies as C
    col = C.make_colony(1)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g, l, c, X, y = dev(col.genomes), dev(col.lengths), dev(col.consts), dev(col.X), dev(col.y)
    P, (N, d) = len(col.lengths), col.X.shape
    api.beagle_reserve(P, int(col.lengths.sum()))
    plain = torch.empty(P, dtype=torch.float32, device="cuda")
    api.beagle_eval(g, l, P, c, len(col.consts), X, y, N, d, col.tax, plain, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    out = torch.zeros(P, dtype=torch.float32, device="cuda")
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        api.beagle_eval(g, l, P, c, len(col.consts), X, y, N, d, col.tax, out, torch.cuda.current_stream().cuda_stream)
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    assert np.array_equal(_bits(out.cpu().numpy()), _bits(plain.cpu().numpy()))
    y.add_(1.0)                                                # same buffers, new targets: the graph reads them at replay
    graph.replay()
    api.beagle_eval(g, l, P, c, len(col.consts), X, y, N, d, col.tax, plain, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(_bits(out.cpu().numpy()), _bits(plain.cpu().numpy()))
