"""Seeded synthetic colonies shaped like BASELINE.json's five configs (host harness, not product).

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's
arithmetic: gen.c draws program shapes and packs tokens; this file draws the fitness cases with
plain numpy. Recipe and the list of what stands in for what: DESIGN.md §5.
The paper's own workloads (its QuadraticEq setup, and the Feynman suite it refers to,
PAPER.md:22) are not reproduced; these colonies stand in for their shapes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libcolony_gen.so")

OP = dict(CONST=1, LOAD=2, ADD=3, SUB=4, MUL=5, DIV=6, SIN=7, COS=8, LOG=9, SQRT=10, EXP=11,
          DUP=0x10, SWAP=0x11, DEL=0x12, SIGN=0x14, SQUARE=0x15, CUBE=0x16,
          CBRT=0x17, TAN=0x18, ARCSIN=0x19, ARCCOS=0x1A, ARCTAN=0x1B, TANH=0x1C,
          POW=0x13, COPY=0x1D, PASTE=0x1E)
OP_NAME = {v: k for k, v in OP.items()}


def token(op: int, arg: int = 0) -> int:
    """Pack {opcode:8, arg:24} as a signed int32 (R2)."""
    w = ((arg & 0xFFFFFF) << 8) | (op & 0xFF)
    return w - (1 << 32) if w >= (1 << 31) else w


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def _gen():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.colony_generate.restype = ctypes.c_int
        _lib.colony_generate.argtypes = [
            ctypes.c_int, ctypes.c_uint64, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_double,
            ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)]
    return _lib


# ------------------------------------------------------------------------------------------------
@dataclass
class ColonyConfig:
    number: int
    name: str
    P: int
    N: int
    d: int
    kind: int                 # 0 = G-tree, 1 = G-len
    dmin: int
    dmax: int
    lcap: int
    unary: tuple
    binary: tuple
    q_u: float
    clo: float
    chi: float
    tax: float = 1e-3
    designed_invalid: bool = False
    budget_bytes: int = 0     # > 0: chunked streaming with this device budget


_U2 = (OP["SIN"], OP["COS"])
_U5 = (OP["SIN"], OP["COS"], OP["LOG"], OP["SQRT"], OP["EXP"])
_B4 = (OP["ADD"], OP["SUB"], OP["MUL"], OP["DIV"])

CONFIGS = {
    1: ColonyConfig(1, "tiny", 1024, 512, 2, 0, 2, 4, 32, _U2, _B4, 0.2, -5.0, 5.0),
    2: ColonyConfig(2, "mid", 65536, 1024, 3, 0, 2, 6, 64, _U5, _B4, 0.2, -10.0, 10.0),
    3: ColonyConfig(3, "paper-scale", 1048576, 512, 5, 0, 2, 8, 128, _U5, _B4, 0.2, -10.0, 10.0),
    4: ColonyConfig(4, "physics-shaped", 1048576, 1024, 9, 0, 2, 10, 255, _U5, _B4, 0.4, -10.0, 10.0),
    5: ColonyConfig(5, "chunked-stress", 4194304, 1024, 9, 1, 0, 0, 512, _U5, _B4, 0.0, -10.0, 10.0,
                    designed_invalid=True, budget_bytes=1 << 30),
}


@dataclass
class Colony:
    cfg: ColonyConfig
    genomes: np.ndarray       # int32[T]
    lengths: np.ndarray       # int32[P]
    consts: np.ndarray        # float32[C]
    X: np.ndarray             # float32[N, d]
    y: np.ndarray             # float32[N]
    tax: float
    y_expr: str = ""
    stats: dict = field(default_factory=dict)

    @property
    def P(self):
        return int(self.lengths.shape[0])

    @property
    def T(self):
        return int(self.genomes.shape[0])

    @property
    def gp_ops(self):
        """GP operations of one evaluation = tokens x fitness cases (BASELINE.json metric)."""
        return self.T * int(self.X.shape[0])


# ------------------------------------------------------------------------------------------------
class _SplitMix64:
    def __init__(self, seed):
        self.s = seed & 0xFFFFFFFFFFFFFFFF

    def next(self):
        self.s = (self.s + 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & 0xFFFFFFFFFFFFFFFF
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & 0xFFFFFFFFFFFFFFFF
        return z ^ (z >> 31)

    def u(self):
        return (self.next() >> 11) * (1.0 / 9007199254740992.0)

    def normal(self):
        u1, u2 = self.u(), self.u()
        return float(np.sqrt(-2.0 * np.log(max(u1, 1e-300))) * np.cos(2.0 * np.pi * u2))


def _random_y_expr(rng, d):
    """A seeded random closed-form expression of 6..12 nodes over the inputs (configs 4-5),
    as a (text, numpy function) pair. Plain numpy arithmetic on positive inputs in [1,5]."""
    target = 6 + int(rng.u() * 7)
    un = [("sin", np.sin), ("cos", np.cos), ("log", lambda a: np.log(np.abs(a))),
          ("sqrt", lambda a: np.sqrt(np.abs(a))), ("exp", np.exp)]
    bn = [("+", np.add), ("-", np.subtract), ("*", np.multiply), ("/", np.divide)]

    def build(budget):
        if budget < 2:
            j = int(rng.u() * d)
            return 1, f"x{j}", (lambda X, j=j: X[:, j])
        if budget < 3 or rng.u() < 0.4:
            name, f = un[int(rng.u() * len(un))]
            n, s, g = build(budget - 1)
            return n + 1, f"{name}({s})", (lambda X, f=f, g=g: f(g(X)))
        name, f = bn[int(rng.u() * len(bn))]
        lb = min((budget - 1 + 1) // 2, budget - 2)
        n1, s1, g1 = build(lb)
        n2, s2, g2 = build(budget - 1 - n1)
        return n1 + n2 + 1, f"({s1} {name} {s2})", (lambda X, f=f, g1=g1, g2=g2: f(g1(X), g2(X)))

    n, s, g = build(target)
    return n, s, g


def make_dataset(cfg: ColonyConfig):
    """X float32[N,d], y float32[N]; computed in fp64 and rounded once."""
    rng = _SplitMix64(0xDA7A0000 + cfg.number)
    N, d = cfg.N, cfg.d
    U = np.array([[rng.u() for _ in range(d)] for _ in range(N)], dtype=np.float64)
    expr = ""
    with np.errstate(all="ignore"):
        if cfg.number == 1:
            X = -1.0 + 2.0 * U
            y = X[:, 0] ** 2 + np.sin(X[:, 1]); expr = "x0^2 + sin(x1)"
        elif cfg.number == 2:
            X = -3.0 + 6.0 * U
            noise = np.array([rng.normal() for _ in range(N)])
            y = X[:, 0] * X[:, 1] / (1.0 + X[:, 2] ** 2) + 0.01 * noise
            expr = "x0*x1/(1+x2^2) + 0.01*N(0,1)"
        elif cfg.number == 3:
            X = 1.0 + 4.0 * U
            y = X[:, 0] * X[:, 1] * np.exp(-X[:, 2] / X[:, 3]) + X[:, 4]
            expr = "x0*x1*exp(-x2/x3) + x4"
        else:
            X = np.exp(U * np.log(5.0))
            while True:
                n, expr, f = _random_y_expr(rng, d)
                y = np.asarray(f(X), dtype=np.float64)
                y32 = y.astype(np.float32)
                if 6 <= n <= 12 and np.all(np.isfinite(y32)) and float(np.ptp(y32)) > 1e-3:
                    break
    return X.astype(np.float32), y.astype(np.float32), expr


_F1_UNARY = (OP["SIGN"], OP["SQUARE"], OP["CUBE"])


def generate_programs(cfg: ColonyConfig, P: int | None = None, seed_offset: int = 0, gcl_mix: str = "hot"):
    """tokens int32[T], lengths int32[P], consts float32[C] for the first P individuals of cfg.
    seed_offset != 0 draws a different colony of the same shape (bench.py: one per rank).
    gcl_mix = "f1" (G-tree configs): SIGN SQUARE CUBE join the unary commands and DUP SWAP DEL are woven into the
    trees (gen.c "f1 mix"): the colony then speaks the part of the paper's language the interpreter runs."""
    P = cfg.P if P is None else int(P)
    seed = 0xBEA61E00 + cfg.number + int(seed_offset)
    f1 = gcl_mix == "f1"
    if f1 and cfg.kind != 0:
        raise ValueError("the f1 mix is defined for the tree-generated configs 1-4")
    unary = tuple(cfg.unary) + (_F1_UNARY if f1 else ())
    un = (ctypes.c_int * len(unary))(*unary)
    bn = (ctypes.c_int * len(cfg.binary))(*cfg.binary)
    lengths = np.empty(P, np.int32)
    T = ctypes.c_int64(0)
    C = ctypes.c_int64(0)
    g = _gen()

    def call(tok, con):
        g.colony_generate(cfg.kind, seed, P, cfg.dmin, cfg.dmax, cfg.lcap, un, len(unary),
                          bn, len(cfg.binary), cfg.q_u, cfg.d, cfg.clo, cfg.chi,
                          int(cfg.designed_invalid), int(f1), lengths.ctypes.data_as(ctypes.c_void_p),
                          None if tok is None else tok.ctypes.data_as(ctypes.c_void_p),
                          None if con is None else con.ctypes.data_as(ctypes.c_void_p),
                          ctypes.byref(T), ctypes.byref(C))

    call(None, None)
    tokens = np.empty(T.value, np.int32)
    consts = np.zeros(max(1, min(C.value, 1 << 24)), np.float32)
    call(tokens, consts)
    return tokens, lengths, consts


def colony_stats(tokens, lengths):
    ops = (tokens & 0xFF).astype(np.int64)
    hist = np.bincount(ops, minlength=32)[:32]
    T = int(tokens.shape[0])
    chk = int(np.bitwise_xor.reduce(
        (tokens.astype(np.uint32).astype(np.uint64) + np.arange(T, dtype=np.uint64))
        * np.uint64(0x9E3779B97F4A7C15))) if T else 0
    return dict(P=int(lengths.shape[0]), T=T,
                mean_len=float(lengths.mean()) if len(lengths) else 0.0,
                median_len=float(np.median(lengths)) if len(lengths) else 0.0,
                max_len=int(lengths.max()) if len(lengths) else 0,
                token_hist={OP_NAME[i]: int(hist[i]) for i in OP_NAME},
                checksum=f"{chk:016x}")


def make_colony(number: int, P: int | None = None) -> Colony:
    """The colony of BASELINE.json config `number` (or its first P individuals)."""
    cfg = CONFIGS[number]
    tokens, lengths, consts = generate_programs(cfg, P)
    X, y, expr = make_dataset(cfg)
    col = Colony(cfg, tokens, lengths, consts, X, y, cfg.tax, expr)
    col.stats = colony_stats(tokens, lengths)
    return col
