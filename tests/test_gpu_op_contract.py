"""-m gpu: the CUDA path's per-command accuracy contract, measured.

The oracle's running error bound E_p is only a bound if every command implementation on the GPU
obeys the contract that bound assumes (`orc_default_contract(1)`). Here each command is run alone,
through beagle_debug_outputs, on swept inputs, and its error against the fp64 definition (numpy,
written out here independently of oracle/ and of csrc/) is checked against the contract's formula.
Also pins the protected-operator edge table (D2) on the GPU, bit for bit.
"""
import numpy as np
import pytest

from paper_2607_06731_b200.colonies import OP, token

pytestmark = pytest.mark.gpu

U = 2.0 ** -24
EPS = float(np.float32(1e-6))
FLT_MIN = float(np.finfo(np.float32).tiny)


def _unary(op, a):
    from tests.gpu_util import gpu_outputs
    a = np.asarray(a, np.float32)
    n = len(a)
    out = np.empty(n, np.float32)
    prog = np.array([token(OP["LOAD"], 0), token(OP[op])], np.int32)
    for s in range(0, n, 1024):
        X = a[s:s + 1024].reshape(-1, 1)
        out[s:s + 1024] = gpu_outputs(prog, np.array([2], np.int32), np.zeros(0, np.float32), X)[0]
    return out


def _binary(op, a, b):
    from tests.gpu_util import gpu_outputs
    a = np.asarray(a, np.float32); b = np.asarray(b, np.float32)
    n = len(a)
    out = np.empty(n, np.float32)
    prog = np.array([token(OP["LOAD"], 0), token(OP["LOAD"], 1), token(OP[op])], np.int32)
    for s in range(0, n, 1024):
        X = np.stack([a[s:s + 1024], b[s:s + 1024]], axis=1)
        out[s:s + 1024] = gpu_outputs(prog, np.array([3], np.int32), np.zeros(0, np.float32), X)[0]
    return out


def _sweep(rng, lo_exp, hi_exp, n, signed=True):
    """log-uniform magnitudes 2^lo..2^hi, random signs."""
    m = np.exp2(rng.uniform(lo_exp, hi_exp, n))
    if signed:
        m *= rng.choice([-1.0, 1.0], n)
    return m.astype(np.float32)


def _contract(oracle):
    return oracle.contract(oracle.CONTRACT_B200)


def test_add_sub_mul_correctly_rounded():
    rng = np.random.default_rng(1)
    a = np.concatenate([_sweep(rng, -60, 60, 20000), _sweep(rng, -140, -120, 2000)])
    b = np.concatenate([_sweep(rng, -60, 60, 20000), _sweep(rng, -20, 20, 2000)])
    for op, f in (("ADD", np.add), ("SUB", np.subtract), ("MUL", np.multiply)):
        got = _binary(op, a, b)
        with np.errstate(all="ignore"):
            want = f(a.astype(np.float64), b.astype(np.float64)).astype(np.float32)
        assert np.array_equal(got.view(np.uint32), want.view(np.uint32)), op


def test_div_contract(oracle):
    c = _contract(oracle)
    rng = np.random.default_rng(2)
    a = np.concatenate([_sweep(rng, -40, 40, 40000), _sweep(rng, -100, 100, 10000)])
    b = np.concatenate([_sweep(rng, -19.5, 40, 40000), _sweep(rng, -19, 127.9, 10000)])
    got = _binary("DIV", a, b).astype(np.float64)
    a64, b64 = a.astype(np.float64), b.astype(np.float64)
    prot = np.abs(b64) < EPS
    with np.errstate(all="ignore"):
        want = np.where(prot, 1.0, a64 / b64)
    fin = np.abs(want) < 3.0e38
    bound = c.c_div * U * np.abs(want) + c.abs_floor + np.where(np.abs(b64) > 2.0 ** 126, np.abs(a64) * c.div_bigb_abs, 0.0)
    err = np.abs(got - want)
    assert np.all(err[fin] <= bound[fin]), (np.max(err[fin] / bound[fin]))
    assert np.all(got[prot] == 1.0)
    print("DIV max err/u|v|:", np.max((err / (U * np.abs(want) + 1e-300))[fin & (np.abs(want) > 1e-30) & (np.abs(b64) < 2.0 ** 126)]))


def test_sqrt_contract(oracle):
    c = _contract(oracle)
    rng = np.random.default_rng(3)
    a = np.concatenate([_sweep(rng, -126, 127.9, 60000), _sweep(rng, -149, -126, 2000)])
    got = _unary("SQRT", a).astype(np.float64)
    want = np.sqrt(np.abs(a.astype(np.float64)))
    err = np.abs(got - want)
    bound = c.c_sqrt * U * want + c.abs_sqrt + c.abs_floor
    assert np.all(err <= bound), np.max(err / bound)
    print("SQRT max err/u|v|:", np.max((err / (U * want))[want > 1e-18]))


def test_exp_contract(oracle):
    c = _contract(oracle)
    rng = np.random.default_rng(4)
    a = np.concatenate([rng.uniform(-110, 90, 60000), _sweep(rng, -30, 3, 10000)]).astype(np.float32)
    got = _unary("EXP", a).astype(np.float64)
    t = np.minimum(a.astype(np.float64), 80.0)
    want = np.exp(t)
    err = np.abs(got - want)
    bound = (c.c_exp + c.c_exp_arg * np.abs(t)) * U * want + c.abs_floor
    assert np.all(err <= bound), np.max(err / bound)
    print("EXP max err/((1+|t|)u v):", np.max((err / ((1 + np.abs(t)) * U * want))[want > 1e-37]))


def test_log_contract(oracle):
    c = _contract(oracle)
    rng = np.random.default_rng(5)
    a = np.concatenate([_sweep(rng, -19.9, 127.9, 60000), (1.0 + rng.uniform(-0.01, 0.01, 10000)).astype(np.float32),
                        _sweep(rng, -30, -19.95, 2000)])
    got = _unary("LOG", a).astype(np.float64)
    aa = np.abs(a.astype(np.float64))
    prot = aa < EPS
    with np.errstate(all="ignore"):
        want = np.where(prot, 0.0, np.log(aa))
    err = np.abs(got - want)
    bound = c.c_log_rel * U * np.abs(want) + c.c_log_abs * U + c.abs_floor
    assert np.all(err <= bound), np.max(err / bound)
    assert np.all(got[prot] == 0.0)
    print("LOG max err/(u(1+|v|)):", np.max(err / (U * (1 + np.abs(want)))))


def test_sin_cos_contract(oracle):
    c = _contract(oracle)
    rng = np.random.default_rng(6)
    a = np.concatenate([rng.uniform(-8, 8, 40000), rng.uniform(-700, 700, 20000),
                        _sweep(rng, -30, 22, 20000), _sweep(rng, 22, 60, 5000)]).astype(np.float32)
    for op, f in (("SIN", np.sin), ("COS", np.cos)):
        got = _unary(op, a).astype(np.float64)
        want = f(a.astype(np.float64))
        err = np.abs(got - want)
        bound = np.minimum((c.c_sin_abs + c.c_sin_arg * np.abs(a.astype(np.float64))) * U + c.abs_floor, 2.000001)
        assert np.all(np.abs(got) <= 1.0 + 1e-6), op
        assert np.all(err <= bound), (op, np.max(err / bound), a[np.argmax(err / bound)])
        small = np.abs(a) < 8
        print(op, "max abs err / u on |a|<8:", np.max(err[small]) / U,
              " max err/(|a|u) on |a|>=8:", np.max((err / (np.abs(a.astype(np.float64)) * U))[~small]))


def test_protected_edge_table_bitwise():
    """DESIGN.md D2 consequences (pin P7), on the GPU."""
    inf, nan = np.float32(np.inf), np.float32(np.nan)
    e80 = np.float32(np.exp(80.0))

    def b(x):
        return np.asarray(x, np.float32).view(np.uint32)

    # DIV
    a = np.array([3.0, 0.0, nan, 1.0, 1.0, inf, 5.0, 5.0, nan, 2.0, -0.0], np.float32)
    d = np.array([0.0, 0.0, 0.0, inf, -inf, inf, 9.9e-7, -9.9e-7, 1.0, nan, 1.0], np.float32)
    got = _binary("DIV", a, d)
    assert got[0] == 1 and got[1] == 1 and got[2] == 1
    assert b(got[3]) == b(0.0) and b(got[4]) == b(-0.0)
    assert np.isnan(got[5]) and got[6] == 1 and got[7] == 1 and np.isnan(got[8]) and np.isnan(got[9])
    thr = np.float32(1e-6)
    got = _binary("DIV", np.array([7.0, 7.0], np.float32), np.array([thr, np.nextafter(thr, np.float32(0))], np.float32))
    assert abs(got[0] / (7.0 / 1e-6) - 1) < 1e-6 and got[1] == 1      # the test is strict '<'
    # LOG
    got = _unary("LOG", np.array([0.0, -0.0, -np.e, inf, -inf, nan, 9.9e-7, 1.0], np.float32))
    assert got[0] == 0 and got[1] == 0 and abs(got[2] - 1) < 1e-6 and got[3] == inf and got[4] == inf
    assert np.isnan(got[5]) and got[6] == 0 and got[7] == 0
    # SQRT
    got = _unary("SQRT", np.array([-4.0, 0.0, -0.0, inf, -inf, nan], np.float32))
    assert abs(got[0] - 2) < 1e-6 and got[1] == 0 and got[2] == 0 and got[3] == inf and got[4] == inf and np.isnan(got[5])
    # EXP
    got = _unary("EXP", np.array([81.0, inf, 80.0, -inf, nan, 0.0, 1e30], np.float32))
    assert np.all(np.abs(got[[0, 1, 2, 6]] / e80 - 1) < 1e-4) and got[3] == 0 and np.isnan(got[4]) and got[5] == 1
    # SIN / COS
    assert np.all(np.isnan(_unary("SIN", np.array([inf, -inf, nan], np.float32))))
    assert np.all(np.isnan(_unary("COS", np.array([inf, -inf, nan], np.float32))))
    assert _unary("SIN", np.array([0.0], np.float32))[0] == 0 and _unary("COS", np.array([0.0], np.float32))[0] == 1


def test_f1_exact_commands_bit_exact():
    """SIGN SQUARE CUBE: exact / correctly rounded products, bit for bit on swept inputs."""
    rng = np.random.default_rng(11)
    a = np.concatenate([_sweep(rng, -60, 60, 20000), _sweep(rng, -140, -100, 2000), np.array([0.0, -0.0, np.inf, -np.inf], np.float32)])
    a64 = a.astype(np.float64)
    with np.errstate(all="ignore"):
        want = {"SIGN": (-a64).astype(np.float32), "SQUARE": (a64 * a64).astype(np.float32),
                "CUBE": ((a64 * a64).astype(np.float32).astype(np.float64) * a64).astype(np.float32)}
    for op, w in want.items():
        got = _unary(op, a)
        assert np.array_equal(got.view(np.uint32), w.view(np.uint32)), op


def test_f1_function_contract(oracle):
    """CBRT TAN ARCSIN ARCCOS ARCTAN TANH on swept inputs against numpy in fp64: relative error within the
    contract the oracle's bound assumes (c_fun), domain behaviour (NaN outside [-1, 1]) exact."""
    c = _contract(oracle)
    rng = np.random.default_rng(12)
    wide = np.concatenate([_sweep(rng, -100, 100, 40000), _sweep(rng, -4, 4, 40000)])
    unit = np.concatenate([rng.uniform(-1, 1, 40000).astype(np.float32), np.array([1.0, -1.0, 0.0], np.float32)])
    ang = np.concatenate([rng.uniform(-100, 100, 40000).astype(np.float32), _sweep(rng, -30, 0, 10000)])
    fns = [("CBRT", wide, np.cbrt, 0), ("TAN", ang, np.tan, 1), ("ARCSIN", unit, np.arcsin, 2), ("ARCCOS", unit, np.arccos, 3),
           ("ARCTAN", wide, np.arctan, 4), ("TANH", wide, np.tanh, 5)]
    for op, a, f, k in fns:
        got = _unary(op, a).astype(np.float64)
        want = f(a.astype(np.float64))
        err = np.abs(got - want)
        bound = c.c_fun[k] * U * np.abs(want) + c.abs_floor
        assert np.all(err <= bound), (op, float(np.max(err / bound)))
    out = np.array([1.0000001, -1.5, 3.0, np.inf], np.float32)
    assert np.all(np.isnan(_unary("ARCSIN", out))) and np.all(np.isnan(_unary("ARCCOS", out)))
    assert np.all(np.isnan(_unary("TAN", np.array([np.inf, -np.inf, np.nan], np.float32))))


def test_pow_contract(oracle):
    """POW = the C pow function against numpy in fp64: relative error within the contract the oracle's
    bound assumes (c_pow), the special cases of the C function exact."""
    c = _contract(oracle)
    rng = np.random.default_rng(13)
    a = np.concatenate([_sweep(rng, -20, 20, 60000, signed=False), rng.uniform(0.5, 2.0, 20000).astype(np.float32)])
    b = np.concatenate([rng.uniform(-6, 6, 60000), rng.uniform(-40, 40, 20000)]).astype(np.float32)
    got = _binary("POW", a, b).astype(np.float64)
    with np.errstate(all="ignore"):
        want = np.power(a.astype(np.float64), b.astype(np.float64))
    fin = (np.abs(want) < 1e38) & (np.abs(want) > 1e-37)
    err = np.abs(got - want)[fin]
    bound = (c.c_pow * U * np.abs(want) + c.abs_floor)[fin]
    assert fin.sum() > 60000 and np.all(err <= bound), float(np.max(err / bound))
    an = -_sweep(rng, -6, 6, 4000, signed=False)
    bn = rng.integers(-7, 8, 4000).astype(np.float32)
    got = _binary("POW", an, bn).astype(np.float64)
    want = np.power(an.astype(np.float64), bn.astype(np.float64))
    assert np.all(np.abs(got - want) <= c.c_pow * U * np.abs(want) + c.abs_floor)
    sa = np.array([-8.0, 3.0, 0.0, 0.0, 1.0, -1.0, np.nan, 2.0, 0.5], np.float32)
    sb = np.array([0.5, 0.0, -1.0, 2.0, np.nan, np.inf, 0.0, np.inf, np.inf], np.float32)
    got = _binary("POW", sa, sb)
    with np.errstate(all="ignore"):
        want = np.power(sa.astype(np.float64), sb.astype(np.float64)).astype(np.float32)
    assert np.array_equal(np.isnan(got), np.isnan(want)) and np.array_equal(got[~np.isnan(got)], want[~np.isnan(want)])
