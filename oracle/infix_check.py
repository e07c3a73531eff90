"""infix_check.py — TEST INFRASTRUCTURE: an independent evaluator used only to pin the oracle.

Structurally different from oracle/beagle_oracle.c on purpose: it first rebuilds an expression
TREE from the postfix tokens, then evaluates that tree recursively with Python's `math` (fp64),
one case at a time, from named nodes ("add", "div", ...) rather than opcode numbers. It takes
symbolic tokens — ("x", j), ("c", value), "add", "sub", "mul", "div", "sin", "cos", "log",
"sqrt", "exp" — so it does not share the binary encoding either.

Semantics follow the same passages: PAPER.md:184 (RPN), PAPER.md:231/238 (operand order),
DESIGN.md D2 (protected forms), D4 (fp32 range), D5 (fitness).
"""
from __future__ import annotations

import math

FLT_MAX = 3.4028234663852886e38
EPS = 9.999999974752427e-07  # float32(1e-6) written out


def _sat(v):
    if v != v:
        return v
    if v > FLT_MAX:
        return math.inf
    if v < -FLT_MAX:
        return -math.inf
    return v


def to_tree(tokens):
    """Postfix list -> nested tuples; the last complete subtree is the program's value (D3)."""
    st = []
    for t in tokens:
        if isinstance(t, tuple):
            st.append(t)
        elif t in ("add", "sub", "mul", "div"):
            right = st.pop()
            left = st.pop()
            st.append((t, left, right))
        else:
            st.append((t, st.pop()))
    return st[-1]


def _mul(a, b):
    if (math.isinf(a) and b == 0) or (math.isinf(b) and a == 0):
        return math.nan
    return a * b


def _div(a, b):
    if b != b:
        return math.nan
    if abs(b) < EPS:
        return 1.0
    if math.isinf(b):
        return math.nan if (math.isinf(a) or a != a) else 0.0
    if a != a:
        return math.nan
    return a / b


def _exp(a):
    if a != a:
        return a
    return math.exp(80.0 if a > 80.0 else a) if a != -math.inf else 0.0


def _log(a):
    if a != a:
        return a
    if abs(a) < EPS:
        return 0.0
    return math.inf if math.isinf(a) else math.log(abs(a))


def _trig(f, a):
    if a != a or math.isinf(a):
        return math.nan
    return f(a)


def value(node, x):
    kind = node[0]
    if kind == "x":
        return float(x[node[1]])
    if kind == "c":
        return float(node[1])
    if len(node) == 3:
        a, b = value(node[1], x), value(node[2], x)
        if kind == "add":
            r = a + b
        elif kind == "sub":
            r = a - b
        elif kind == "mul":
            r = _mul(a, b)
        else:
            r = _div(a, b)
        return _sat(r)
    a = value(node[1], x)
    if kind == "sin":
        r = _trig(math.sin, a)
    elif kind == "cos":
        r = _trig(math.cos, a)
    elif kind == "log":
        r = _log(a)
    elif kind == "sqrt":
        r = math.sqrt(abs(a)) if a == a else a
    else:
        r = _exp(a)
    return _sat(r)


def fitness(tokens, X, y, tax):
    """MSE + tax * len(tokens), with the overflow rules of D5 (sum saturates, then / N)."""
    tree = to_tree(tokens)
    s = 0.0
    for xi, yi in zip(X, y):
        r = _sat(value(tree, xi) - float(yi))
        q = _sat(r * r) if not math.isinf(r) else math.inf
        s = s + q
    if s == s and s > FLT_MAX:
        s = math.inf
    return s / len(y) + float(tax) * len(tokens)
