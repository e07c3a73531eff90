"""Test helpers: a tiny assembler from text to packed tokens (encoding only, no arithmetic)."""
import numpy as np

from paper_2607_06731_b200.colonies import OP, token

_NAMES = {"ADD": "add", "SUB": "sub", "MUL": "mul", "DIV": "div", "SIN": "sin", "COS": "cos",
          "LOG": "log", "SQRT": "sqrt", "EXP": "exp"}


def asm(text, consts=None, const_base=0):
    """'x0 x1 ADD 2.5 MUL' -> (tokens int32[], consts float32[]). Numbers become CONST entries
    appended to `consts` (a list that is extended in place if given)."""
    cl = [] if consts is None else consts
    toks = []
    for w in text.replace(";", " ").split():
        u = w.upper()
        if u.startswith(("COPY@", "PASTE@")):                   # GCL's variables: COPY@2, PASTE@2
            toks.append(token(OP[u.split("@")[0]], int(u.split("@")[1])))
        elif u in OP and u not in ("CONST", "LOAD"):
            toks.append(token(OP[u]))
        elif u.startswith("X") and u[1:].isdigit():
            toks.append(token(OP["LOAD"], int(u[1:])))
        else:
            cl.append(np.float32(float(w)))
            toks.append(token(OP["CONST"], const_base + len(cl) - 1))
    return np.array(toks, np.int32), np.array(cl, np.float32)


def symbolic(tokens, consts):
    """Packed tokens -> the symbolic form oracle/infix_check.py takes."""
    out = []
    inv = {v: k for k, v in OP.items()}
    for w in np.asarray(tokens).astype(np.uint32):
        op, arg = int(w & 0xFF), int(w >> 8)
        if op == OP["CONST"]:
            out.append(("c", float(consts[arg])))
        elif op == OP["LOAD"]:
            out.append(("x", arg))
        else:
            out.append(_NAMES[inv[op]])
    return out


def pack(programs, consts):
    """list of token arrays -> (genomes, lengths, consts)."""
    lengths = np.array([len(p) for p in programs], np.int32)
    genomes = np.concatenate(programs).astype(np.int32) if programs else np.zeros(0, np.int32)
    return genomes, lengths, np.asarray(consts, np.float32)


def random_gcl_programs(rng, n_prog, d, names):
    """Seeded random postfix programs as text over the commands in `names` (plus terminals x0..x{d-1} and constants):
    a command is taken when the stack holds its operands, else a terminal is pushed; kept when something is left on
    the stack. Shapes only, no arithmetic."""
    progs_text = []
    while len(progs_text) < n_prog:
        toks, depth = [], 0
        for _ in range(int(rng.integers(3, 60))):
            nm = names[int(rng.integers(len(names)))]
            need = 2 if nm in ("ADD", "SUB", "MUL", "DIV", "SWAP", "POW") else 1
            if depth < need or (nm == "DUP" and depth >= 30) or rng.random() < 0.35:
                toks.append(f"x{int(rng.integers(d))}" if rng.random() < 0.8 else f"{rng.uniform(-3, 3):.4f}"); depth += 1
            else:
                toks.append(nm); depth += {"DUP": 1, "DEL": -1}.get(nm, -1 if need == 2 and nm != "SWAP" else 0)
        if depth >= 1:
            progs_text.append(" ".join(toks))
    return progs_text
