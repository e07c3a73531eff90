"""Mutation check of the oracle's pins (test infrastructure; run by hand, not collected by pytest).

Each entry is one plausible mistake in oracle/beagle_oracle.c (a transposed operand, a wrong sign, index, limit or constant, a
dropped term of a value or of a bound). The script plants them one at a time in a copy of the repository under /tmp, rebuilds the
oracle there and runs the CPU pins (tests/test_oracle_pins.py) against it: a mutant that passes every pin points at a missing pin.
DESIGN.md section 4 records the outcome.

    python tests/mutate_oracle.py [first] [last]            # the value / structure mutants
    MUT_SET=2 python tests/mutate_oracle.py                 # the error-bound mutants
"""
import os, shutil, subprocess, sys, time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
WORK = "/tmp/mut"
M = [
    # (name, old, new): old must occur exactly once in the source
    ("const index", "st[sp].v = (double)consts[arg];", "st[sp].v = (double)consts[0];"),
    ("load index", "st[sp].v = (double)x[arg];", "st[sp].v = (double)x[0];"),
    ("add/sub swapped", "(op == OP_ADD) ? a.v + b.v : a.v - b.v", "(op == OP_ADD) ? a.v - b.v : a.v + b.v"),
    ("sub transposed", "(op == OP_ADD) ? a.v + b.v : a.v - b.v", "(op == OP_ADD) ? a.v + b.v : b.v - a.v"),
    ("mul -> add", "double v = a.v * b.v;", "double v = a.v + b.v;"),
    ("dup copies second", "case OP_DUP:  st[sp] = st[sp - 1]; sp++; break;", "case OP_DUP:  st[sp] = st[sp > 1 ? sp - 2 : sp - 1]; sp++; break;"),
    ("swap is a no-op", "case OP_SWAP: { pair b = st[sp - 1]; st[sp - 1] = st[sp - 2]; st[sp - 2] = b; break; }", "case OP_SWAP: { break; }"),
    ("del is a no-op", "case OP_DEL:  sp--; break;", "case OP_DEL:  break;"),
    ("sign dropped", "st[sp - 1].v = -st[sp - 1].v; break;", "st[sp - 1].v = st[sp - 1].v; break;"),
    ("sign -> abs", "st[sp - 1].v = -st[sp - 1].v; break;", "st[sp - 1].v = fabs(st[sp - 1].v); break;"),
    ("square -> identity", "case OP_SQUARE: st[sp - 1] = mul_pair(st[sp - 1], st[sp - 1], c, mirror, flags); break;", "case OP_SQUARE: break;"),
    ("cube -> square", "st[sp - 1] = mul_pair(mul_pair(a, a, c, mirror, flags), a, c, mirror, flags);", "st[sp - 1] = mul_pair(a, a, c, mirror, flags);"),
    ("copy index", "case OP_COPY:  var[arg] = st[sp - 1]; break;", "case OP_COPY:  var[0] = st[sp - 1]; break;"),
    ("paste index", "case OP_PASTE: st[sp] = var[arg]; sp++; break;", "case OP_PASTE: st[sp] = var[0]; sp++; break;"),
    ("copy pops", "case OP_COPY:  var[arg] = st[sp - 1]; break;", "case OP_COPY:  var[arg] = st[sp - 1]; if (sp > 1) sp--; break;"),
    ("pow transposed", "double v = pow(a.v, b.v), e = 0.0;", "double v = pow(b.v, a.v), e = 0.0;"),
    ("div transposed", "                v = a.v / b.v;\n                if (!isnan(a.v) && !isinf(a.v)) {", "                v = b.v / a.v;\n                if (!isnan(a.v) && !isinf(a.v)) {"),
    ("div protected value", "else if (ab + b.e < EPS_PROT) v = 1.0;", "else if (ab + b.e < EPS_PROT) v = 0.0;"),
    ("div protection not strict", "else if (ab + b.e < EPS_PROT) v = 1.0;", "else if (ab + b.e <= EPS_PROT) v = 1.0;"),
    ("eps", "#define EPS_PROT ((double)1e-6f)", "#define EPS_PROT ((double)1e-5f)"),
    ("eps as double", "#define EPS_PROT ((double)1e-6f)", "#define EPS_PROT (1e-6)"),
    ("div nan/inf divisor", "if (isnan(b.v) || isinf(b.v)) v = a.v / b.v;", "if (isnan(b.v) || isinf(b.v)) v = 1.0;"),
    ("sin/cos swapped", "double v = (op == OP_SIN) ? sin(a.v) : cos(a.v);", "double v = (op == OP_SIN) ? cos(a.v) : sin(a.v);"),
    ("log without abs", "                v = log(aa);\n", "                v = log(a.v);\n"),
    ("log protected value", "else if (aa + a.e < EPS_PROT) v = 0.0;", "else if (aa + a.e < EPS_PROT) v = 1.0;"),
    ("log of inf", "else if (isinf(a.v)) v = INFINITY;", "else if (isinf(a.v)) v = -INFINITY;"),
    ("log10", "                v = log(aa);\n", "                v = log10(aa);\n"),
    ("sqrt without abs", "double aa = fabs(a.v), v = sqrt(aa), e = 0.0;", "double aa = fabs(a.v), v = sqrt(a.v), e = 0.0;"),
    ("exp clamp 88", "double t = a.v > 80.0 ? 80.0 : a.v;", "double t = a.v > 88.0 ? 88.0 : a.v;"),
    ("exp clamp by fmin", "double t = a.v > 80.0 ? 80.0 : a.v;", "double t = fmin(a.v, 80.0);"),
    ("exp clamp below too", "double t = a.v > 80.0 ? 80.0 : a.v;", "double t = a.v > 80.0 ? 80.0 : (a.v < -80.0 ? -80.0 : a.v);"),
    ("exp2", "double v = exp(t), e = 0.0;", "double v = exp2(t), e = 0.0;"),
    ("asin/acos swapped", "case OP_ARCSIN: return asin(a);\n    case OP_ARCCOS: return acos(a);", "case OP_ARCSIN: return acos(a);\n    case OP_ARCCOS: return asin(a);"),
    ("tan -> tanh", "case OP_TAN: return tan(a);", "case OP_TAN: return tanh(a);"),
    ("tanh -> atan", "default: return tanh(a);", "default: return atan(a);"),
    ("cbrt -> sqrt", "case OP_CBRT: return cbrt(a);", "case OP_CBRT: return sqrt(fabs(a));"),
    ("result = bottom of stack", "return st[sp - 1]; /* D3: output = top of stack */", "return st[0]; /* D3: output = top of stack */"),
    ("residual sign irrelevant -> abs error", "double q0 = r.v * r.v;", "double q0 = fabs(r.v);"),
    ("mean over N-1", "double fit = S / (double)N + (double)tax * (double)L;", "double fit = S / (double)(N > 1 ? N - 1 : N) + (double)tax * (double)L;"),
    ("sum not mean", "double fit = S / (double)N + (double)tax * (double)L;", "double fit = S + (double)tax * (double)L;"),
    ("tax subtracted", "double fit = S / (double)N + (double)tax * (double)L;", "double fit = S / (double)N - (double)tax * (double)L;"),
    ("tax on L+1", "double fit = S / (double)N + (double)tax * (double)L;", "double fit = S / (double)N + (double)tax * (double)(L + 1);"),
    ("tax dropped", "double fit = S / (double)N + (double)tax * (double)L;", "double fit = S / (double)N;"),
    ("overflow on the mean", "if (S > FMAX) S = INFINITY;", "if (S / (double)N > FMAX) S = INFINITY;"),
    ("residual saturation dropped", "pair r = finish(r0, o.e + U32 * (fabs(r0) + o.e) + c->abs_floor, mirror, &flags);", "pair r; r.v = r0; r.e = o.e + U32 * (fabs(r0) + o.e) + c->abs_floor;"),
    ("x row stride", "pair o = run_case(tok, L, consts, X + (size_t)i * d, c, mirror, &flags);", "pair o = run_case(tok, L, consts, X + (size_t)i, c, mirror, &flags);"),
    ("out-of-range lengths count words", "        if (inrange) off += L;            /* out-of-range lengths count as 0 words */", "        if (L > 0) off += L;"),
    ("stack limit 31", "if (sp > ORC_MAX_STACK) return -1;", "if (sp >= ORC_MAX_STACK) return -1;"),
    ("stack limit 33", "if (sp > ORC_MAX_STACK) return -1;", "if (sp > ORC_MAX_STACK + 1) return -1;"),
    ("const index bound", "case OP_CONST: if ((int64_t)arg >= n_consts) return -1; sp++; break;", "case OP_CONST: if ((int64_t)arg > n_consts) return -1; sp++; break;"),
    ("load index bound", "case OP_LOAD:  if ((int64_t)arg >= (int64_t)d) return -1; sp++; break;", "case OP_LOAD:  if ((int64_t)arg > (int64_t)d) return -1; sp++; break;"),
    ("operator arg ignored", "if (arg != 0 || sp < 2) return -1; sp--; break;", "if (sp < 2) return -1; sp--; break;"),
    ("unary arg ignored", "            if (arg != 0 || sp < 1) return -1; break;\n", "            if (sp < 1) return -1; break;\n"),
    ("binary needs one", "if (arg != 0 || sp < 2) return -1; sp--; break;", "if (arg != 0 || sp < 1) return -1; sp--; break;"),
    ("final depth exactly one", "return (sp >= 1 && live == 0) ? mx : -1;", "return (sp == 1 && live == 0) ? mx : -1;"),
    ("unpaired copy allowed", "return (sp >= 1 && live == 0) ? mx : -1;", "return (sp >= 1) ? mx : -1;"),
    ("paste keeps the variable", "live &= ~(1u << arg); sp++; break;", "sp++; break;"),
    ("depth = final depth", "if (sp > mx) mx = sp;", "mx = sp;"),
    ("max length 511", "int inrange = (L >= 1 && L <= ORC_MAX_LEN);\n        int depth = inrange ? check_program(tok, L, n_consts, d) : -1;\n        if (inrange) off += L;            /*", "int inrange = (L >= 1 && L < ORC_MAX_LEN);\n        int depth = inrange ? check_program(tok, L, n_consts, d) : -1;\n        if (inrange) off += L;            /*"),
    ("fp32 overflow -> inf dropped", "else if (a > FMAX) v = v > 0 ? INFINITY : -INFINITY;", "else if (a > FMAX) v = v;"),
    ("mirror rounding dropped", "if (mirror) v = (double)(float)v;", "if (mirror) v = v;"),
    # correlation
    ("corr: r2 not squared again", "const double r4 = r2 * r2, dr4", "const double r4 = r2, dr4"),
    ("corr: c1 - c2 sign", "- (double)M * (double)(c1 - c2);      /* Eq. 2 */", "- (double)M * (double)(c2 - c1);      /* Eq. 2 */"),
    ("corr: c1 + c2", "- (double)M * (double)(c1 - c2);      /* Eq. 2 */", "- (double)M * (double)(c1 + c2);      /* Eq. 2 */"),
    ("corr: times N not nv", "const double score = (double)M * r4 * (double)nv", "const double score = (double)M * r4 * (double)N"),
    ("corr: tax added", "const double fit = score - (double)tax * (double)L;\n        fitness_out[p] = (float)fit;\n        if (bound_out) bound_out[p] = (double)M * nv", "const double fit = score + (double)tax * (double)L;\n        fitness_out[p] = (float)fit;\n        if (bound_out) bound_out[p] = (double)M * nv"),
    ("corr: means over N", "const double mf = sf / nv, my = sy / nv;", "const double mf = sf / N, my = sy / N;"),
    ("corr: c1/c2 classes swapped", "if (vf && vy) ++nv; else if (vf != vy) ++c1; else ++c2;", "if (vf && vy) ++nv; else if (vf != vy) ++c2; else ++c1;"),
    ("corr: one valid pair is enough", "if (nv >= 2) {", "if (nv >= 1) {"),
    ("corr: covariance not squared", "r2 = (Sfy * Sfy) / (Sff * Syy);", "r2 = fabs(Sfy) / sqrt(Sff * Syy);"),
    # std
    ("std: penalty M/10", "const float pen = M / 11.0f;", "const float pen = M / 10.0f;"),
    ("std: both zero scores 0", "            if (mx == 0.0f) {\n                score += (double)M;", "            if (mx == 0.0f) {\n                score += 0.0;"),
    ("std: ratio inverted", "const float q = mn / mx;", "const float q = mx / mn;"),
    ("std: cube = square", "else if (power == 3) qp = (q * q) * q;", "else if (power == 3) qp = (q * q);"),
    ("std: hyper = fourth power", "else if (power == 8) { qp = q * q; qp = qp * qp; qp = qp * qp; }", "else if (power == 8) { qp = q * q; qp = qp * qp; }"),
    ("std: opposite sign ignored", "if (opposite) t = t - pen;", "if (0) t = t - pen;"),
    ("std: penalty after rounding", "if (opposite) t = t - pen;\n            score += (double)rintf(t);", "score += (double)rintf(t) - (opposite ? (double)rintf(pen) : 0.0); if (0)\n            score += (double)rintf(t);"),
    ("std: round half away", "score += (double)rintf(t);", "score += (double)roundf(t);"),
    ("std: truncation", "score += (double)rintf(t);", "score += (double)truncf(t);"),
    ("std: one-sided invalid scores +M", "score += (vf != vy) ? -(double)M : (double)M; continue;", "score += (vf != vy) ? (double)M : -(double)M; continue;"),
    ("std: tax added", "const double fit = score - (double)tax * (double)L;\n        fitness_out[p] = (float)fit;\n        if (bound_out) bound_out[p] = E +", "const double fit = score + (double)tax * (double)L;\n        fitness_out[p] = (float)fit;\n        if (bound_out) bound_out[p] = E +"),
    ("std: power applied to M q", "float t = M * qp;", "float t = powf(M * q, (float)power) / powf(M, (float)(power - 1));"),
]

M2 = [
    ("bound add: b.e dropped", "double e1 = a.e + b.e;", "double e1 = a.e;"),
    ("bound add: rounding dropped", "st[sp - 2] = finish(v, e1 + c->c_add * U32 * (fabs(v) + e1) + fl, mirror, flags);", "st[sp - 2] = finish(v, e1 + fl, mirror, flags);"),
    ("bound mul: a.e term dropped", "double e1 = fabs(a.v) * b.e + fabs(b.v) * a.e + a.e * b.e;", "double e1 = fabs(a.v) * b.e + a.e * b.e;"),
    ("bound mul: rounding dropped", "return finish(v, e1 + c->c_mul * U32 * (fabs(v) + e1) + c->abs_floor, mirror, flags);", "return finish(v, e1 + c->abs_floor, mirror, flags);"),
    ("bound div: divisor term dropped", "double e1 = (a.e + fabs(v) * b.e) / (ab - b.e);", "double e1 = (a.e) / (ab - b.e);"),
    ("bound div: rounding dropped", "e = e1 + c->c_div * U32 * (fabs(v) + e1) + fl;", "e = e1 + fl;"),
    ("bound sin: input dropped", "double e = fmin(a.e, 2.0) + (c->c_sin_abs", "double e = 0.0 + (c->c_sin_abs"),
    ("bound sin: contract dropped", "double e = fmin(a.e, 2.0) + (c->c_sin_abs + c->c_sin_arg * (fabs(a.v) + a.e)) * U32 + fl;", "double e = fmin(a.e, 2.0) + fl;"),
    ("bound log: input dropped", "double e1 = -log1p(-a.e / aa);", "double e1 = 0.0;"),
    ("bound sqrt: input dropped", "double e1 = fmax(v - lo, hi - v);", "double e1 = 0.0;"),
    ("bound exp: input dropped", "double e1 = v * expm1(dt);", "double e1 = 0.0;"),
    ("bound exp: contract dropped", "e = e1 + (c->c_exp + c->c_exp_arg * (fabs(t) + dt)) * U32 * (v + e1) + fl;", "e = e1 + fl;"),
    ("bound fun: input dropped", "double e1 = fmax(fabs(fun_eval(op, lo) - v), fabs(fun_eval(op, hi) - v));", "double e1 = 0.0;"),
    ("bound pow: one corner only", "for (int ia = -1; ia <= 1 && !unstable; ia += 2)", "for (int ia = 1; ia <= 1 && !unstable; ia += 2)"),
    ("bound residual: output dropped", "pair r = finish(r0, o.e + U32 * (fabs(r0) + o.e) + c->abs_floor, mirror, &flags);", "pair r = finish(r0, U32 * (fabs(r0)) + c->abs_floor, mirror, &flags);"),
    ("bound square: factor 2 dropped", "double eq1 = 2.0 * fabs(r.v) * r.e + r.e * r.e;", "double eq1 = fabs(r.v) * r.e + r.e * r.e;"),
    ("bound sum: cases not added", "            ES += q.e;\n", "            ES = q.e;\n"),
    ("bound sum: summation dropped", "double E = ES + (c->sum_per_case * (double)N + c->sum_const) * U32 * (S + ES);", "double E = ES;"),
    ("bound final: not divided", ": ES / (double)N + 4.0 * U32 * fabs(fit) + c->abs_floor;", ": ES + 4.0 * U32 * fabs(fit) + c->abs_floor;"),
    ("bound final: dropped", ": ES / (double)N + 4.0 * U32 * fabs(fit) + c->abs_floor;", ": 4.0 * U32 * fabs(fit) + c->abs_floor;"),
    ("bound x10", ": ES / (double)N + 4.0 * U32 * fabs(fit) + c->abs_floor;", ": 10.0 * ES / (double)N + 4.0 * U32 * fabs(fit) + c->abs_floor;"),
    ("unstable div never flagged", "} else { *flags |= ORC_FLAG_UNSTABLE; v = (ab < EPS_PROT) ? 1.0 : a.v / b.v; }", "} else { v = (ab < EPS_PROT) ? 1.0 : a.v / b.v; }"),
    ("unstable log never flagged", "} else { *flags |= ORC_FLAG_UNSTABLE; v = (aa < EPS_PROT) ? 0.0 : log(aa); }", "} else { v = (aa < EPS_PROT) ? 0.0 : log(aa); }"),
    ("class-unstable never flagged", "else if (a - e <= FMAX && a + e >= FMAX) *flags |= ORC_FLAG_CLASS_UNSTABLE;", "else if (0) *flags |= ORC_FLAG_CLASS_UNSTABLE;"),
    ("corr bound: A dropped", "A += fabs(dy) * e[i]; B +=", "A += 0.0; B +="),
    ("corr bound: B dropped", "B += 2.0 * fabs(df) * e[i] + e[i] * e[i];", "B += 0.0;"),
    ("corr bound: dr4 dropped", "bound_out[p] = (double)M * nv * dr4 + 4.0 * U32", "bound_out[p] = 0.0 * dr4 + 4.0 * U32"),
    ("std bound: boundary cases dropped", "if (o.e > 0.0 && dist <= dt) E += dt + 1.0;", "if (0) E += dt + 1.0;"),
    ("std bound: dq halved", "const double dq = 2.0 * e / (double)mx;", "const double dq = 0.1 * e / (double)mx;"),
    ("contract: div 3.5 -> 1", "c->c_div = 3.5;", "c->c_div = 1.0;"),
    ("contract: sin 12 -> 1", "c->c_sin_abs = 12.0; c->c_sin_arg = 3.0;", "c->c_sin_abs = 1.0; c->c_sin_arg = 0.0;"),
]


def setup():
    if os.path.exists(WORK):
        shutil.rmtree(WORK)
    os.makedirs(WORK)
    for d in ("oracle", "tests", "paper_2607_06731_b200", "include"):
        shutil.copytree(os.path.join(ROOT, d), os.path.join(WORK, d), ignore=shutil.ignore_patterns("__pycache__", "libbeagle_oracle.so"))
    for f in ("BASELINE.json",):
        if os.path.exists(os.path.join(ROOT, f)):
            shutil.copy(os.path.join(ROOT, f), WORK)


def run(i, name, old, new, src):
    n = src.count(old)
    if n != 1:
        return f"{i:3d} {name}: PATTERN x{n}"
    open(os.path.join(WORK, "oracle", "beagle_oracle.c"), "w").write(src.replace(old, new))
    lib = os.path.join(WORK, "oracle", "libbeagle_oracle.so")
    if os.path.exists(lib):
        os.remove(lib)
    t0 = time.time()
    r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_oracle_pins.py", "-x", "-q", "-p", "no:cacheprovider"], cwd=WORK,
                       capture_output=True, text=True)
    tail = [l for l in r.stdout.splitlines() if l.startswith("FAILED") or "passed" in l or "error" in l.lower()]
    killed = r.returncode != 0
    return f"{i:3d} {name}: {'killed' if killed else 'SURVIVED'} ({time.time() - t0:.0f}s) {tail[0][:110] if tail else ''}"


if __name__ == "__main__":
    setup()
    src = open(os.path.join(ROOT, "oracle", "beagle_oracle.c")).read()
    if os.environ.get("MUT_SET") == "2":
        M = M2
    a = int(sys.argv[1]) if len(sys.argv) > 1 else 0
    b = int(sys.argv[2]) if len(sys.argv) > 2 else len(M)
    for i, (name, old, new) in enumerate(M[a:b], start=a):
        print(run(i, name, old, new, src), flush=True)
