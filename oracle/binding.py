"""ctypes binding of oracle/beagle_oracle.c — TEST INFRASTRUCTURE, not the product.

`build()` compiles the C file with gcc into oracle/libbeagle_oracle.so (building the checker is not
using it). `evaluate()` marshals numpy arrays and calls `orc_eval`; it does no arithmetic of its
own. `evaluate_parallel()` fans individual ranges out over host threads for wall time only
(SURVEY.md §8(d) "CPU baseline"): each range is the same single-threaded C call.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "beagle_oracle.c")
_LIB = os.path.join(_HERE, "libbeagle_oracle.so")

FLAG_MALFORMED = 1
FLAG_UNSTABLE = 2
FLAG_CLASS_UNSTABLE = 4

CONTRACT_IEEE = 0
CONTRACT_B200 = 1


class Contract(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in (
        "c_add", "c_mul", "c_div", "div_bigb_abs", "c_sqrt", "abs_sqrt", "c_exp", "c_exp_arg",
        "c_log_rel", "c_log_abs", "c_sin_abs", "c_sin_arg", "abs_floor", "sum_per_case",
        "sum_const")] + [("c_fun", ctypes.c_double * 6), ("c_pow", ctypes.c_double)]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fno-fast-math",
                               "-ffp-contract=off", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_eval.restype = ctypes.c_int
        _lib.orc_eval.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                                  ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p,
                                  ctypes.c_int32, ctypes.c_int32, ctypes.c_float,
                                  ctypes.POINTER(Contract), ctypes.c_int,
                                  ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                  ctypes.c_void_p]
        _lib.orc_default_contract.restype = None
        _lib.orc_eval_corr.restype = ctypes.c_int
        _lib.orc_eval_corr.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64,
                                       ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32,
                                       ctypes.c_float, ctypes.c_float, ctypes.POINTER(Contract),
                                       ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        _lib.orc_eval_std.restype = ctypes.c_int
        _lib.orc_eval_std.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64,
                                      ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                      ctypes.c_float, ctypes.c_float, ctypes.POINTER(Contract), ctypes.c_int,
                                      ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        _lib.orc_default_contract.argtypes = [ctypes.c_int, ctypes.POINTER(Contract)]
    return _lib


def contract(which: int = CONTRACT_B200) -> Contract:
    c = Contract()
    lib().orc_default_contract(which, ctypes.byref(c))
    return c


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def evaluate(genomes, lengths, consts, X, y, tax, *, contract_=None, mode=0, want_outputs=False):
    """Returns dict(fitness f32[P], bound f64[P], flags i32[P], depth i32[P], outputs f64[P,N]|None)."""
    genomes = np.ascontiguousarray(genomes, dtype=np.int32)
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    consts = np.ascontiguousarray(consts, dtype=np.float32)
    X = np.ascontiguousarray(X, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    P = int(lengths.shape[0])
    N, d = int(X.shape[0]), int(X.shape[1])
    assert y.shape[0] == N
    c = contract_ if contract_ is not None else contract(CONTRACT_B200)
    fit = np.empty(P, np.float32)
    bound = np.empty(P, np.float64)
    flags = np.empty(P, np.int32)
    depth = np.empty(P, np.int32)
    outs = np.empty((P, N), np.float64) if want_outputs else None
    rc = lib().orc_eval(_ptr(genomes), _ptr(lengths), P, _ptr(consts), int(consts.shape[0]),
                        _ptr(X), _ptr(y), N, d, float(tax), ctypes.byref(c), int(mode),
                        _ptr(fit), _ptr(bound), _ptr(flags), _ptr(depth), _ptr(outs))
    if rc != 0:
        raise ValueError("orc_eval: bad arguments")
    return dict(fitness=fit, bound=bound, flags=flags, depth=depth, outputs=outs)


def evaluate_corr(genomes, lengths, consts, X, y, M, tax, *, contract_=None):
    """The correlation fitness (Eq. 1-2): dict(fitness, bound, flags, depth, stats f64[P,4] = r^2, valid, c1, c2)."""
    genomes = np.ascontiguousarray(genomes, dtype=np.int32)
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    consts = np.ascontiguousarray(consts, dtype=np.float32)
    X = np.ascontiguousarray(X, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    P = int(lengths.shape[0])
    N, d = int(X.shape[0]), int(X.shape[1])
    assert y.shape[0] == N
    c = contract_ if contract_ is not None else contract(CONTRACT_B200)
    fit = np.empty(P, np.float32)
    bound = np.empty(P, np.float64)
    flags = np.empty(P, np.int32)
    depth = np.empty(P, np.int32)
    stats = np.empty((P, 4), np.float64)
    rc = lib().orc_eval_corr(_ptr(genomes), _ptr(lengths), P, _ptr(consts), int(consts.shape[0]),
                             _ptr(X), _ptr(y), N, d, float(M), float(tax), ctypes.byref(c),
                             _ptr(fit), _ptr(bound), _ptr(flags), _ptr(depth), _ptr(stats))
    if rc != 0:
        raise ValueError("orc_eval_corr: bad arguments")
    return dict(fitness=fit, bound=bound, flags=flags, depth=depth, stats=stats)


def evaluate_std(genomes, lengths, consts, X, y, power, M, tax, *, contract_=None, mode=0):
    """The Std integer-reward family (Eq. 5; power 1, 2, 3, 8): dict(fitness, bound, flags, depth)."""
    genomes = np.ascontiguousarray(genomes, dtype=np.int32)
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    consts = np.ascontiguousarray(consts, dtype=np.float32)
    X = np.ascontiguousarray(X, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    P = int(lengths.shape[0])
    N, d = int(X.shape[0]), int(X.shape[1])
    assert y.shape[0] == N
    c = contract_ if contract_ is not None else contract(CONTRACT_B200)
    fit = np.empty(P, np.float32)
    bound = np.empty(P, np.float64)
    flags = np.empty(P, np.int32)
    depth = np.empty(P, np.int32)
    rc = lib().orc_eval_std(_ptr(genomes), _ptr(lengths), P, _ptr(consts), int(consts.shape[0]),
                            _ptr(X), _ptr(y), N, d, int(power), float(M), float(tax), ctypes.byref(c), int(mode),
                            _ptr(fit), _ptr(bound), _ptr(flags), _ptr(depth))
    if rc != 0:
        raise ValueError("orc_eval_std: bad arguments")
    return dict(fitness=fit, bound=bound, flags=flags, depth=depth)


def evaluate_parallel(genomes, lengths, consts, X, y, tax, *, threads=None, contract_=None, mode=0):
    """Same call fanned out over host threads by individual ranges (wall time only)."""
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    genomes = np.ascontiguousarray(genomes, dtype=np.int32)
    P = int(lengths.shape[0])
    threads = threads or os.cpu_count() or 1
    if P == 0 or threads <= 1:
        return evaluate(genomes, lengths, consts, X, y, tax, contract_=contract_, mode=mode)
    inr = (lengths >= 1) & (lengths <= 512)
    off = np.concatenate([[0], np.cumsum(np.where(inr, lengths, 0), dtype=np.int64)])
    # ranges of roughly equal token count
    n_parts = min(P, threads * 8)
    targets = (off[-1] * np.arange(1, n_parts)) // n_parts
    cuts = np.unique(np.concatenate([[0], np.searchsorted(off[:-1], targets), [P]]))
    parts = [(int(a), int(b)) for a, b in zip(cuts[:-1], cuts[1:]) if b > a]

    def run(ab):
        a, b = ab
        return evaluate(genomes[off[a]:off[b]], lengths[a:b], consts, X, y, tax,
                        contract_=contract_, mode=mode)

    with ThreadPoolExecutor(max_workers=threads) as ex:
        res = list(ex.map(run, parts))
    return {k: np.concatenate([r[k] for r in res]) for k in ("fitness", "bound", "flags", "depth")}
