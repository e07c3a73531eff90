/* beagle_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded CPU evaluator of what the Beagle scoring path computes, written
 * from the paper and DESIGN.md's readings, in fp64. It shares no code, header, table or constant
 * generator with the CUDA path (paper_2607_06731_b200/csrc); the opcode numbers below are retyped
 * from DESIGN.md D2, not included. Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.
 *
 * What it follows
 *   - PAPER.md:184 (§3.2): RPN stack machine; unary commands replace the top of the stack, binary
 *     commands replace the top two with the result.
 *   - PAPER.md:190: the stack holds 32 entries.
 *   - PAPER.md:200-294 (Table 3): command meanings; operand order SUB = second-top - top
 *     (PAPER.md:231), DIV = second-top / top.
 *   - PAPER.md:314: length = the number of GCL commands (terminals included).
 *   - PAPER.md:63: one aggregated value per individual for the whole batch of fitness cases.
 *   - north_star (BASELINE.json) where the paper is silent: fitness = MSE + tax*length, protected
 *     div/log/sqrt/exp, {opcode:8,arg:24} tokens, constants in a side fp32 table. Exact forms:
 *     DESIGN.md D1-D6.
 *
 * The method is an exact evaluation, so the oracle is the definition written out: for every
 * individual, for every case, run the tokens in order on a stack; square the residual; sum; divide
 * by N; add tax*L. No blocking, fusion or reordering.
 *
 * Beside the value v the stack carries e >= |v_gpu - v|, a running bound on how far an fp32
 * evaluator whose per-op accuracy obeys `orc_contract` can be from v (DESIGN.md §4 "error bound").
 * The bound never changes v; it only tells the parity test which tolerance class an individual is
 * in (STRICT / CONDITIONED / UNSTABLE).
 *
 * Pins (tests/test_oracle_pins.py, all CPU): P1 printed lengths, P2 closed forms of the paper's
 * printed genomes, P3 x0*x0 vs x0^2, P4 CONST/LOAD reduce to numpy, P5 identity insertion,
 * P6 commutativity/antisymmetry, P7 protected-operator edge table, P8 brute force of all programs
 * of <= 3 tokens against an independent recursive evaluator (oracle/infix_check.py), P9 power-of-two
 * scaling, P10 overflow semantics, P11 the bound is a bound (fp32 mirror), P12 case duplication.
 * P13-P18 the rest of Table 3 (P17b: the corner bound of POW is a bound), P19 the correlation fitness (orc_eval_corr),
 * P21 / P21b the Std family (orc_eval_std: Eq. 5 by hand; its bound E is a bound).
 * Parity unpinned: nothing (every value and every bound the parity rule uses has a pin of its own).
 */
#include <float.h>
#include <math.h>
#include <stdint.h>
#include <stddef.h>

/* DESIGN.md D2 (numbers retyped, not shared) */
enum { OP_CONST = 1, OP_LOAD = 2, OP_ADD = 3, OP_SUB = 4, OP_MUL = 5, OP_DIV = 6,
       OP_SIN = 7, OP_COS = 8, OP_LOG = 9, OP_SQRT = 10, OP_EXP = 11,
       /* the rest of Table 3 in its own order from 0x10 (D2); built so far: the three
        * stack commands, the three exact unary ones, six more unary functions, POW and the COPY / PASTE variables. */
       OP_DUP = 0x10, OP_SWAP = 0x11, OP_DEL = 0x12, OP_SIGN = 0x14, OP_SQUARE = 0x15, OP_CUBE = 0x16,
       /* unprotected, as the paper's are: plain mathematical functions, NaN outside their domain */
       OP_CBRT = 0x17, OP_TAN = 0x18, OP_ARCSIN = 0x19, OP_ARCCOS = 0x1A, OP_ARCTAN = 0x1B, OP_TANH = 0x1C,
       OP_POW = 0x13,    /* second-top to the power of top, the C pow function: NaN for a negative base with a
                            non-integer exponent */
       OP_COPY = 0x1D,   /* top of stack -> variable @arg, stack unchanged                              */
       OP_PASTE = 0x1E };/* variable @arg -> pushed; the variable is destroyed                                      */
#define ORC_MAX_VARS 32  /* variable identifiers @0 .. @31 (D2 extension)                                  */

#define ORC_MAX_LEN   512
#define ORC_MAX_STACK 32
#define ORC_MAX_N     1024

#define ORC_FLAG_MALFORMED      1 /* DESIGN.md D3 / R9                                        */
#define ORC_FLAG_UNSTABLE       2 /* an input interval straddles a protected-op threshold     */
#define ORC_FLAG_CLASS_UNSTABLE 4 /* an interval straddles the fp32 overflow edge, or the sign
                                     of an infinity depends on an uncertain zero              */

/* Accuracy contract of the evaluator being checked, in units of u = 2^-24 unless said otherwise.
 * The test passes the CUDA path's published contract or the IEEE contract
 * (all c = 1, abs terms 0) for the fp32 mirror.                                               */
typedef struct {
    double c_add;        /* ADD, SUB: relative                                                */
    double c_mul;        /* MUL: relative                                                     */
    double c_div;        /* DIV: relative                                                     */
    double div_bigb_abs; /* DIV: extra absolute error |a| * this when |b| can exceed 2^126    */
    double c_sqrt;       /* SQRT: relative                                                    */
    double abs_sqrt;     /* SQRT: absolute (denormal inputs flushed)                          */
    double c_exp;        /* EXP: relative, constant part                                      */
    double c_exp_arg;    /* EXP: relative, per unit of |argument|                             */
    double c_log_rel;    /* LOG: relative                                                     */
    double c_log_abs;    /* LOG: absolute                                                     */
    double c_sin_abs;    /* SIN, COS: absolute, constant part                                 */
    double c_sin_arg;    /* SIN, COS: absolute, per unit of |argument|                        */
    double abs_floor;    /* every computed op: absolute (denormal results flushed), NOT in u  */
    double sum_per_case; /* summation: the fp32 sum of N squares is off by at most            */
    double sum_const;    /*   (sum_per_case * N + sum_const) * u * S  (depth of the add tree) */
    double c_fun[6];     /* CBRT TAN ARCSIN ARCCOS ARCTAN TANH: relative                      */
    double c_pow;        /* POW: relative                                                     */
} orc_contract;

static const double U32 = 5.9604644775390625e-08; /* 2^-24 */
static const double FMAX = 3.4028234663852886e+38; /* FLT_MAX */
#define EPS_PROT ((double)1e-6f)                   /* DESIGN.md D2: EPS = 1e-6f               */

typedef struct { double v, e; } pair;

/* D4: fp32 range semantics in an fp64 carrier; mirror mode rounds to fp32 instead. Also applies
 * the overflow-edge test of DESIGN.md §4 (last row of the propagation table).                  */
static inline pair finish(double v, double e, int mirror, int* flags) {
    pair r;
    if (isnan(v)) { r.v = v; r.e = 0.0; return r; }
    if (isinf(v)) { r.v = v; r.e = 0.0; return r; }
    double a = fabs(v);
    if (!(e < INFINITY)) { *flags |= ORC_FLAG_CLASS_UNSTABLE; e = 0.0; }
    else if (a - e <= FMAX && a + e >= FMAX) *flags |= ORC_FLAG_CLASS_UNSTABLE;
    if (mirror) v = (double)(float)v;
    else if (a > FMAX) v = v > 0 ? INFINITY : -INFINITY;
    r.v = v; r.e = isinf(v) ? 0.0 : e;
    return r;
}

/* Static well-formedness (D3): returns the maximum stack depth, or -1 if malformed. */
static int check_program(const uint32_t* tok, int L, int64_t n_consts, int d) {
    if (L < 1 || L > ORC_MAX_LEN) return -1;
    int sp = 0, mx = 0;
    uint32_t live = 0;   /* variables that hold a value: COPY and PASTE come in pairs */
    for (int t = 0; t < L; ++t) {
        uint32_t op = tok[t] & 0xFFu, arg = tok[t] >> 8;
        switch (op) {
        case OP_COPY:  if (arg >= ORC_MAX_VARS || sp < 1 || ((live >> arg) & 1u)) return -1; live |= 1u << arg; break;
        case OP_PASTE: if (arg >= ORC_MAX_VARS || !((live >> arg) & 1u)) return -1; live &= ~(1u << arg); sp++; break;
        case OP_CONST: if ((int64_t)arg >= n_consts) return -1; sp++; break;
        case OP_LOAD:  if ((int64_t)arg >= (int64_t)d) return -1; sp++; break;
        case OP_ADD: case OP_SUB: case OP_MUL: case OP_DIV: case OP_POW:
            if (arg != 0 || sp < 2) return -1; sp--; break;
        case OP_SIN: case OP_COS: case OP_LOG: case OP_SQRT: case OP_EXP:
        case OP_SIGN: case OP_SQUARE: case OP_CUBE:
        case OP_CBRT: case OP_TAN: case OP_ARCSIN: case OP_ARCCOS: case OP_ARCTAN: case OP_TANH:
            if (arg != 0 || sp < 1) return -1; break;
        case OP_DUP:  if (arg != 0 || sp < 1) return -1; sp++; break;
        case OP_SWAP: if (arg != 0 || sp < 2) return -1; break;
        case OP_DEL:  if (arg != 0 || sp < 1) return -1; sp--; break;
        default: return -1;
        }
        if (sp > ORC_MAX_STACK) return -1;
        if (sp > mx) mx = sp;
    }
    return (sp >= 1 && live == 0) ? mx : -1;   /* a COPY without its PASTE is not a valid program */
}

/* a * b with its bound; also the two products of CUBE and the one of SQUARE. */
static pair mul_pair(pair a, pair b, const orc_contract* c, int mirror, int* flags) {
    double v = a.v * b.v;
    if ((isinf(a.v) && !isnan(b.v) && !isinf(b.v) && fabs(b.v) <= b.e) ||
        (isinf(b.v) && !isnan(a.v) && !isinf(a.v) && fabs(a.v) <= a.e))
        *flags |= ORC_FLAG_CLASS_UNSTABLE;     /* inf * (maybe zero, sign unknown) */
    double e1 = fabs(a.v) * b.e + fabs(b.v) * a.e + a.e * b.e;
    if (isnan(e1)) e1 = 0.0;                   /* inf * 0 inside the bound only    */
    return finish(v, e1 + c->c_mul * U32 * (fabs(v) + e1) + c->abs_floor, mirror, flags);
}

/* CBRT TAN ARCSIN ARCCOS ARCTAN TANH: the plain function; each is monotone on every interval of
 * its domain, so the input's uncertainty maps to max |f(a +- e) - f(a)|. An interval that reaches past the domain of
 * ARCSIN / ARCCOS, or across a pole of TAN, makes the individual UNSTABLE.                                          */
static double fun_eval(uint32_t op, double a) {
    switch (op) {
    case OP_CBRT: return cbrt(a);
    case OP_TAN: return tan(a);
    case OP_ARCSIN: return asin(a);
    case OP_ARCCOS: return acos(a);
    case OP_ARCTAN: return atan(a);
    default: return tanh(a);
    }
}
static pair fun_pair(uint32_t op, pair a, const orc_contract* c, int mirror, int* flags) {
    double v = fun_eval(op, a.v), e = 0.0;
    if (!isnan(a.v) && !isinf(a.v) && !isnan(v)) {
        double lo = a.v - a.e, hi = a.v + a.e;
        if (op == OP_ARCSIN || op == OP_ARCCOS) {
            if (lo < -1.0 || hi > 1.0) { *flags |= ORC_FLAG_UNSTABLE; lo = fmax(lo, -1.0); hi = fmin(hi, 1.0); }
        } else if (op == OP_TAN) {
            const double pi = 3.14159265358979323846;
            if (floor(lo / pi + 0.5) != floor(hi / pi + 0.5)) { *flags |= ORC_FLAG_UNSTABLE; lo = hi = a.v; }
        }
        double e1 = fmax(fabs(fun_eval(op, lo) - v), fabs(fun_eval(op, hi) - v));
        if (isnan(e1)) e1 = 0.0;
        e = e1 + c->c_fun[op - OP_CBRT] * U32 * (fabs(v) + e1) + c->abs_floor;
    } else if (isnan(v) && !isnan(a.v) && (fabs(a.v) - a.e <= 1.0) && (op == OP_ARCSIN || op == OP_ARCCOS))
        *flags |= ORC_FLAG_UNSTABLE;           /* outside the domain, but the interval reaches into it */
    return finish(v, e, mirror, flags);
}

/* One program on one case: PAPER.md:184 stack semantics, Table 3 operand order, D2 values. */
static pair run_case(const uint32_t* tok, int L, const float* consts, const float* x,
                     const orc_contract* c, int mirror, int* flags) {
    pair st[ORC_MAX_STACK], var[ORC_MAX_VARS];
    int sp = 0;
    const double fl = c->abs_floor;
    for (int t = 0; t < L; ++t) {
        uint32_t op = tok[t] & 0xFFu, arg = tok[t] >> 8;
        switch (op) {
        case OP_CONST: st[sp].v = (double)consts[arg]; st[sp].e = 0.0; sp++; break;
        case OP_LOAD:  st[sp].v = (double)x[arg];      st[sp].e = 0.0; sp++; break;
        case OP_ADD: case OP_SUB: {
            pair a = st[sp - 2], b = st[sp - 1];
            double v = (op == OP_ADD) ? a.v + b.v : a.v - b.v;
            double e1 = a.e + b.e;
            st[sp - 2] = finish(v, e1 + c->c_add * U32 * (fabs(v) + e1) + fl, mirror, flags);
            sp--; break; }
        case OP_MUL:
            st[sp - 2] = mul_pair(st[sp - 2], st[sp - 1], c, mirror, flags);
            sp--; break;
        case OP_DUP:  st[sp] = st[sp - 1]; sp++; break;                    /* the two top-most are identical */
        case OP_SWAP: { pair b = st[sp - 1]; st[sp - 1] = st[sp - 2]; st[sp - 2] = b; break; }
        case OP_DEL:  sp--; break;                                         /* pops the stack */
        case OP_SIGN: st[sp - 1].v = -st[sp - 1].v; break;                 /* changes the sign; exact */
        case OP_SQUARE: st[sp - 1] = mul_pair(st[sp - 1], st[sp - 1], c, mirror, flags); break;   /* a * a */
        case OP_CBRT: case OP_TAN: case OP_ARCSIN: case OP_ARCCOS: case OP_ARCTAN: case OP_TANH:
            st[sp - 1] = fun_pair(op, st[sp - 1], c, mirror, flags); break;
        case OP_COPY:  var[arg] = st[sp - 1]; break;                       /* no change to the stack */
        case OP_PASTE: st[sp] = var[arg]; sp++; break;                     /* pushes the variable    */
        case OP_POW: {                         /* second-top ^ top. Bound: the corners of the input box */
            pair a = st[sp - 2], b = st[sp - 1];
            double v = pow(a.v, b.v), e = 0.0;
            if (!isnan(v) && !isinf(v) && !isnan(a.v) && !isinf(a.v) && !isnan(b.v) && !isinf(b.v)) {
                double e1 = 0.0;
                int unstable = 0;
                if (a.v < 0.0 && b.e > 0.0) unstable = 1;                  /* a non-integer exponent nearby: NaN */
                if (fabs(a.v) <= a.e && (a.e > 0.0 || b.v <= 0.0)) unstable = 1;   /* the base may be zero or change sign */
                for (int ia = -1; ia <= 1 && !unstable; ia += 2)
                    for (int ib = -1; ib <= 1; ib += 2) {
                        double w = pow(a.v + ia * a.e, b.v + ib * b.e);
                        if (isnan(w)) { unstable = 1; break; }
                        e1 = fmax(e1, fabs(w - v));
                    }
                if (unstable) { *flags |= ORC_FLAG_UNSTABLE; e1 = 0.0; }
                e = e1 + c->c_pow * U32 * (fabs(v) + e1) + fl;
            }
            st[sp - 2] = finish(v, e, mirror, flags);
            sp--; break; }
        case OP_CUBE: {                                                    /* (a * a) * a, two products */
            pair a = st[sp - 1];
            st[sp - 1] = mul_pair(mul_pair(a, a, c, mirror, flags), a, c, mirror, flags);
            break; }
        case OP_DIV: {                         /* P:238; protected form D2: |b|<EPS ? 1 : a/b */
            pair a = st[sp - 2], b = st[sp - 1];
            double ab = fabs(b.v), v, e = 0.0;
            if (isnan(b.v) || isinf(b.v)) v = a.v / b.v;
            else if (ab + b.e < EPS_PROT) v = 1.0;
            else if (ab - b.e >= EPS_PROT) {
                v = a.v / b.v;
                if (!isnan(a.v) && !isinf(a.v)) {
                    double e1 = (a.e + fabs(v) * b.e) / (ab - b.e);
                    e = e1 + c->c_div * U32 * (fabs(v) + e1) + fl;
                    if (ab + b.e > 8.507059173023462e+37) /* 2^126 */
                        e += (fabs(a.v) + a.e) * c->div_bigb_abs;
                }
            } else { *flags |= ORC_FLAG_UNSTABLE; v = (ab < EPS_PROT) ? 1.0 : a.v / b.v; }
            st[sp - 2] = finish(v, e, mirror, flags);
            sp--; break; }
        case OP_SIN: case OP_COS: {
            pair a = st[sp - 1];
            double v = (op == OP_SIN) ? sin(a.v) : cos(a.v);  /* sin(+-inf) = NaN */
            double e = fmin(a.e, 2.0) + (c->c_sin_abs + c->c_sin_arg * (fabs(a.v) + a.e)) * U32 + fl;
            if (!(e < 2.000001)) e = 2.000001;
            st[sp - 1] = finish(v, e, mirror, flags);
            break; }
        case OP_LOG: {                         /* P:253; protected: |a|<EPS ? 0 : ln|a|      */
            pair a = st[sp - 1];
            double aa = fabs(a.v), v, e = 0.0;
            if (isnan(a.v)) v = a.v;
            else if (isinf(a.v)) v = INFINITY;
            else if (aa + a.e < EPS_PROT) v = 0.0;
            else if (aa - a.e >= EPS_PROT) {
                v = log(aa);
                double e1 = -log1p(-a.e / aa);
                e = e1 + c->c_log_rel * U32 * (fabs(v) + e1) + c->c_log_abs * U32 + fl;
            } else { *flags |= ORC_FLAG_UNSTABLE; v = (aa < EPS_PROT) ? 0.0 : log(aa); }
            st[sp - 1] = finish(v, e, mirror, flags);
            break; }
        case OP_SQRT: {                        /* P:249; protected: sqrt|a|                  */
            pair a = st[sp - 1];
            double aa = fabs(a.v), v = sqrt(aa), e = 0.0;
            if (!isnan(a.v) && !isinf(a.v)) {
                double lo = aa > a.e ? sqrt(aa - a.e) : 0.0, hi = sqrt(aa + a.e);
                double e1 = fmax(v - lo, hi - v);
                e = e1 + c->c_sqrt * U32 * (v + e1) + c->abs_sqrt + fl;
            }
            st[sp - 1] = finish(v, e, mirror, flags);
            break; }
        case OP_EXP: {                         /* P:275; clamped: exp(a > 80 ? 80 : a)       */
            pair a = st[sp - 1];
            double t = a.v > 80.0 ? 80.0 : a.v;  /* ternary so NaN passes (R5) */
            double v = exp(t), e = 0.0;
            if (!isnan(a.v) && !isinf(a.v)) {
                double up = fmin(a.v + a.e, 80.0) - t, dn = t - fmin(a.v - a.e, 80.0);
                double dt = fmax(up, dn);
                double e1 = v * expm1(dt);
                e = e1 + (c->c_exp + c->c_exp_arg * (fabs(t) + dt)) * U32 * (v + e1) + fl;
            }
            st[sp - 1] = finish(v, e, mirror, flags);
            break; }
        default: break; /* unreachable: check_program ran first */
        }
    }
    return st[sp - 1]; /* D3: output = top of stack */
}

/* orc_eval — the whole colony (D5-D6).
 *   genomes/lengths/consts/X/y as in include/beagle.h (host pointers); mode 0 = truth (fp64
 *   carrier with fp32 range), 1 = mirror (every op result rounded to fp32).
 *   fitness_out[P] float; bound_out[P] double (E_p) or NULL; flags_out[P] int32 or NULL;
 *   depth_out[P] int32 (max stack depth, 0 if malformed) or NULL;
 *   outputs P*N doubles (per-case outputs, NaN rows for malformed) or NULL.
 * Returns 0, or -1 on bad arguments.                                                          */
int orc_eval(const int32_t* genomes, const int32_t* lengths, int64_t P,
             const float* consts, int64_t n_consts,
             const float* X, const float* y, int32_t N, int32_t d, float tax,
             const orc_contract* c, int mode,
             float* fitness_out, double* bound_out, int32_t* flags_out, int32_t* depth_out,
             double* outputs) {
    if (P < 0 || N < 1 || N > ORC_MAX_N || d < 1 || !c) return -1;
    const int mirror = (mode == 1);
    int64_t off = 0;
    for (int64_t p = 0; p < P; ++p) {
        int L = lengths[p];
        const uint32_t* tok = (const uint32_t*)genomes + off;
        int inrange = (L >= 1 && L <= ORC_MAX_LEN);
        int depth = inrange ? check_program(tok, L, n_consts, d) : -1;
        if (inrange) off += L;            /* out-of-range lengths count as 0 words */
        int flags = 0;
        if (depth < 0) {
            union { uint32_t u; float f; } qn; qn.u = 0x7FC00000u;
            fitness_out[p] = qn.f;
            if (bound_out) bound_out[p] = 0.0;
            if (flags_out) flags_out[p] = ORC_FLAG_MALFORMED;
            if (depth_out) depth_out[p] = 0;
            if (outputs) for (int i = 0; i < N; ++i) outputs[p * (int64_t)N + i] = NAN;
            continue;
        }
        double S = 0.0, ES = 0.0;
        for (int i = 0; i < N; ++i) {
            pair o = run_case(tok, L, consts, X + (size_t)i * d, c, mirror, &flags);
            if (outputs) outputs[p * (int64_t)N + i] = o.v;
            /* D5: r = sat32(out - y), q = sat32(r^2) */
            double r0 = o.v - (double)y[i];
            pair r = finish(r0, o.e + U32 * (fabs(r0) + o.e) + c->abs_floor, mirror, &flags);
            double q0 = r.v * r.v;
            double eq1 = 2.0 * fabs(r.v) * r.e + r.e * r.e;
            if (isnan(eq1)) eq1 = 0.0;
            pair q = finish(q0, eq1 + U32 * (q0 + eq1) + c->abs_floor, mirror, &flags);
            S += q.v;              /* fp64 sum; NaN and +inf propagate by IEEE rules */
            ES += q.e;
        }
        if (!isnan(S) && !isinf(S)) {
            double E = ES + (c->sum_per_case * (double)N + c->sum_const) * U32 * (S + ES);
            if (S - E <= FMAX && S + E >= FMAX) flags |= ORC_FLAG_CLASS_UNSTABLE;
            if (S > FMAX) S = INFINITY;   /* D5: overflow is decided on the sum, not the mean */
            ES = E;
        } else ES = 0.0;
        double fit = S / (double)N + (double)tax * (double)L;
        fitness_out[p] = (float)fit;
        if (bound_out) bound_out[p] = (isnan(fit) || isinf(fit)) ? 0.0
                                     : ES / (double)N + 4.0 * U32 * fabs(fit) + c->abs_floor;
        if (flags_out) flags_out[p] = flags;
        if (depth_out) depth_out[p] = depth;
    }
    return 0;
}

/* orc_eval_corr — the paper's default objective, the correlation fitness (Eq. 1-2, printed again
 * as Eq. 3-4 at P:494-501; D7). For every individual:
 *   a case is a VALID pair when both the model output f_i and the target y_i are finite ("NaN, Inf, etc.");
 *   c1 = number of valid/invalid pairs (exactly one side finite), c2 = number of invalid/invalid pairs;
 *   r  = Pearson correlation of f and y over the valid pairs, means taken over the valid pairs (Eq. 1);
 *   score = M r^4 (N - (c1 + c2)) - M (c1 - c2)                                                  (Eq. 2);
 *   fitness = score - tax * L   (maximised; the length tax is a rate per command taken off the score).
 * Readings (R23): r = 0 when fewer than two valid pairs are left or either side has zero variance there.
 * Written as the definition: the textbook two-pass sums in fp64, nothing reordered.
 * The bound follows the perturbation of r^2 = Sfy^2 / (Sff Syy) under |f_gpu,i - f_i| <= e_i plus the rounding of an
 * fp32 two-pass summation in the contract's order (means of values shifted by one of them); it never changes a value.
 * stats (NULL or P*4 doubles): r^2, valid pairs, c1, c2.                                                          */
int orc_eval_corr(const int32_t* genomes, const int32_t* lengths, int64_t P,
                  const float* consts, int64_t n_consts,
                  const float* X, const float* y, int32_t N, int32_t d, float M, float tax,
                  const orc_contract* c,
                  float* fitness_out, double* bound_out, int32_t* flags_out, int32_t* depth_out, double* stats) {
    if (P < 0 || N < 1 || N > ORC_MAX_N || d < 1 || !c) return -1;
    double f[ORC_MAX_N], e[ORC_MAX_N];
    int64_t off = 0;
    for (int64_t p = 0; p < P; ++p) {
        int L = lengths[p];
        const uint32_t* tok = (const uint32_t*)genomes + off;
        int inrange = (L >= 1 && L <= ORC_MAX_LEN);
        int depth = inrange ? check_program(tok, L, n_consts, d) : -1;
        if (inrange) off += L;
        int flags = 0;
        if (depth < 0) {
            union { uint32_t u; float f; } qn; qn.u = 0x7FC00000u;
            fitness_out[p] = qn.f;
            if (bound_out) bound_out[p] = 0.0;
            if (flags_out) flags_out[p] = ORC_FLAG_MALFORMED;
            if (depth_out) depth_out[p] = 0;
            if (stats) for (int k = 0; k < 4; ++k) stats[4 * p + k] = NAN;
            continue;
        }
        int nv = 0, c1 = 0, c2 = 0;
        for (int i = 0; i < N; ++i) {
            pair o = run_case(tok, L, consts, X + (size_t)i * d, c, 0, &flags);
            f[i] = o.v; e[i] = o.e;
            int vf = isfinite(o.v), vy = isfinite((double)y[i]);
            if (vf && vy) ++nv; else if (vf != vy) ++c1; else ++c2;
        }
        double r2 = 0.0, dr2 = 0.0;
        if (nv >= 2) {
            double sf = 0.0, sy = 0.0;
            for (int i = 0; i < N; ++i) if (isfinite(f[i]) && isfinite((double)y[i])) { sf += f[i]; sy += (double)y[i]; }
            const double mf = sf / nv, my = sy / nv;                       /* Eq. 1: the two means */
            double Sff = 0.0, Syy = 0.0, Sfy = 0.0, A = 0.0, B = 0.0, Df = 0.0, Dy = 0.0;
            for (int i = 0; i < N; ++i) if (isfinite(f[i]) && isfinite((double)y[i])) {
                const double df = f[i] - mf, dy = (double)y[i] - my;
                Sfy += dy * df; Sff += df * df; Syy += dy * dy;           /* Eq. 1: numerator, the two sums under the root */
                A += fabs(dy) * e[i]; B += 2.0 * fabs(df) * e[i] + e[i] * e[i];
                Df = fmax(Df, fabs(df)); Dy = fmax(Dy, fabs(dy));
            }
            const double g = (c->sum_per_case * (double)N + c->sum_const + 4.0) * U32;
            const double dSfy = A + g * sqrt(Sff * Syy) + nv * g * g * 4.0 * Df * Dy + c->abs_floor;
            const double dSff = B + g * Sff + nv * g * g * 4.0 * Df * Df;
            const double dSyy = g * Syy + nv * g * g * 4.0 * Dy * Dy;
            if (!(Sff <= FMAX && Syy <= FMAX && fabs(Sfy) <= FMAX) || Df * Df > FMAX || Dy * Dy > FMAX)
                flags |= ORC_FLAG_CLASS_UNSTABLE;                        /* fp32 sums of squares overflow           */
            if (Sff > 0.0 && Syy > 0.0) {
                r2 = (Sfy * Sfy) / (Sff * Syy);                           /* "the r value is then squared"    */
                if (dSff > 0.5 * Sff || dSyy > 0.5 * Syy) flags |= ORC_FLAG_UNSTABLE;    /* variance within its own error */
                else {
                    const double hi = (Sfy * Sfy + 2.0 * fabs(Sfy) * dSfy + dSfy * dSfy) / ((Sff - dSff) * (Syy - dSyy));
                    const double lo = fmax(0.0, Sfy * Sfy - 2.0 * fabs(Sfy) * dSfy) / ((Sff + dSff) * (Syy + dSyy));
                    dr2 = fmax(hi - r2, r2 - lo) + 4.0 * U32 * r2;
                }
            } else if (dSff > 0.0 && Syy > 0.0) flags |= ORC_FLAG_UNSTABLE;  /* zero variance here, maybe not in fp32 */
        }
        const double r4 = r2 * r2, dr4 = 2.0 * r2 * dr2 + dr2 * dr2;
        const double score = (double)M * r4 * (double)nv - (double)M * (double)(c1 - c2);      /* Eq. 2 */
        const double fit = score - (double)tax * (double)L;
        fitness_out[p] = (float)fit;
        if (bound_out) bound_out[p] = (double)M * nv * dr4 + 4.0 * U32 * (fabs((double)M * r4 * nv) + fabs((double)M * (c1 - c2)) + fabs(fit)) + c->abs_floor;
        if (flags_out) flags_out[p] = flags;
        if (depth_out) depth_out[p] = depth;
        if (stats) { stats[4 * p] = r2; stats[4 * p + 1] = nv; stats[4 * p + 2] = c1; stats[4 * p + 3] = c2; }
    }
    return 0;
}

/* orc_eval_std — the point-to-point integer-reward family StdFitFunc / StdSquareFitFunc / StdCubeFitFunc /
 * StdHyperFitFunc (PAPER.md:490 and Eq. 5 at P:503-506; D9). For every valid pair (both sides finite):
 *     M                                       if max(|f|, |y|) = 0
 *     round(M q^p - M/11)                      if f y < 0          q = min(|f|, |y|) / max(|f|, |y|)
 *     round(M q^p)                             otherwise
 * with p = 1 (Eq. 5 as printed), 2, 3, 8 for the Square, Cube and Hyper variants; a pair with exactly one side finite
 * scores -M, a pair with neither +M (the convention of Eq. 2; FitFunctionIfInvalid's values are not printed);
 * score = sum over the cases; fitness = score - tax * L, maximised.
 * Readings (R25): `round` is round-half-to-even (the default of the paper's implementation language); the
 * powers apply to the ratio q before scaling by M (applied to the integer reward they would turn the penalty of an
 * opposite sign into a bonus); "f y < 0" is decided on the signs (no underflow of the product).
 * The reward is an integer decided by floating point, so it is taken in the paper's precision, fp32, on both sides:
 * the arithmetic below is fp32, in the order |.|, min/max, one division, the power by squarings, * M, - M/11, rintf.
 * The bound: a case can differ from the device's by |dt| + 1 when its unrounded value t is within dt of a rounding
 * boundary, where dt follows from the output bound e; otherwise by nothing.
 * mode as in orc_eval: 0 = outputs in fp64, 1 = mirror (every command's result rounded to fp32).                   */
int orc_eval_std(const int32_t* genomes, const int32_t* lengths, int64_t P,
                 const float* consts, int64_t n_consts,
                 const float* X, const float* y, int32_t N, int32_t d, int32_t power, float M, float tax,
                 const orc_contract* c, int mode,
                 float* fitness_out, double* bound_out, int32_t* flags_out, int32_t* depth_out) {
    if (P < 0 || N < 1 || N > ORC_MAX_N || d < 1 || !c) return -1;
    if (power != 1 && power != 2 && power != 3 && power != 8) return -1;
    int64_t off = 0;
    const float pen = M / 11.0f;
    for (int64_t p = 0; p < P; ++p) {
        int L = lengths[p];
        const uint32_t* tok = (const uint32_t*)genomes + off;
        int inrange = (L >= 1 && L <= ORC_MAX_LEN);
        int depth = inrange ? check_program(tok, L, n_consts, d) : -1;
        if (inrange) off += L;
        int flags = 0;
        if (depth < 0) {
            union { uint32_t u; float f; } qn; qn.u = 0x7FC00000u;
            fitness_out[p] = qn.f;
            if (bound_out) bound_out[p] = 0.0;
            if (flags_out) flags_out[p] = ORC_FLAG_MALFORMED;
            if (depth_out) depth_out[p] = 0;
            continue;
        }
        double score = 0.0, E = 0.0;
        for (int i = 0; i < N; ++i) {
            pair o = run_case(tok, L, consts, X + (size_t)i * d, c, mode == 1, &flags);
            const int vf = isfinite(o.v), vy = isfinite((double)y[i]);
            if (!(vf && vy)) { score += (vf != vy) ? -(double)M : (double)M; continue; }
            const float f = (float)o.v, yy = y[i];
            const float a = fabsf(f), b = fabsf(yy);
            const float mx = fmaxf(a, b), mn = fminf(a, b);
            if (mx == 0.0f) {
                score += (double)M;
                if (o.e > 0.0) E += (double)M;              /* the device's output may be non-zero */
                continue;
            }
            const float q = mn / mx;
            float qp = q;
            if (power == 2) qp = q * q;
            else if (power == 3) qp = (q * q) * q;
            else if (power == 8) { qp = q * q; qp = qp * qp; qp = qp * qp; }
            const int opposite = (f < 0.0f && yy > 0.0f) || (f > 0.0f && yy < 0.0f);
            float t = M * qp;
            if (opposite) t = t - pen;
            score += (double)rintf(t);
            /* how far the device's t can be: dq <= 2 e / mx (q <= 1), d(q^p) <= p q^(p-1) dq, plus fp32 roundings */
            const double e = o.e + U32 * fabs(o.v);
            const double dq = 2.0 * e / (double)mx;
            double dt = (double)M * (double)power * pow((double)q, (double)(power - 1)) * dq + 8.0 * U32 * (double)M;
            if (fabs(o.v) <= e && yy != 0.0f) dt += (double)pen;          /* the sign of the output is not certain */
            const double fr = (double)t - floor((double)t);
            const double dist = fabs(fr - 0.5);                            /* distance to the rounding boundary */
            if (o.e > 0.0 && dist <= dt) E += dt + 1.0;
        }
        const double fit = score - (double)tax * (double)L;
        fitness_out[p] = (float)fit;
        if (bound_out) bound_out[p] = E + 4.0 * U32 * fabs(fit);
        if (flags_out) flags_out[p] = flags;
        if (depth_out) depth_out[p] = depth;
    }
    return 0;
}

/* The two contracts the tests use most, so that Python does not have to retype 13 doubles.
 * which = 0: IEEE (every op correctly rounded: c = 1, a little slack for libm, no abs terms);
 * which = 1: the CUDA path's published contract, DESIGN.md §6 (numbers retyped from there).   */
void orc_default_contract(int which, orc_contract* c) {
    if (which == 0) {
        c->c_add = 1.0; c->c_mul = 1.0; c->c_div = 1.0; c->div_bigb_abs = 0.0;
        c->c_sqrt = 1.0; c->abs_sqrt = 0.0; c->c_exp = 1.001; c->c_exp_arg = 0.0;
        c->c_log_rel = 1.001; c->c_log_abs = 0.0; c->c_sin_abs = 1.001; c->c_sin_arg = 0.0;
        c->abs_floor = 1.5e-45;
        c->sum_per_case = 1.0; c->sum_const = 0.0;   /* any summation order */
        for (int k = 0; k < 6; ++k) c->c_fun[k] = 1.001;
        c->c_pow = 1.001;
    } else {
        c->c_add = 1.0; c->c_mul = 1.0;
        c->c_div = 3.5; c->div_bigb_abs = 1.1754943508222875e-38;
        c->c_sqrt = 3.0; c->abs_sqrt = 1.1e-19;
        c->c_exp = 6.0; c->c_exp_arg = 2.5;
        c->c_log_rel = 5.0; c->c_log_abs = 4.0;
        c->c_sin_abs = 12.0; c->c_sin_arg = 3.0;
        c->abs_floor = 1.1754943508222875e-38;
        c->sum_per_case = 1.0 / 32.0; c->sum_const = 5.0; /* per-lane chain + 5 shuffle levels */
        /* CUDA math library cbrtf tanf asinf acosf atanf tanhf: documented 1 4 2 2 2 2 ulp, + 1 for the rounding of the input side */
        c->c_fun[0] = 3.0; c->c_fun[1] = 6.0; c->c_fun[2] = 4.0; c->c_fun[3] = 4.0; c->c_fun[4] = 4.0; c->c_fun[5] = 4.0;
        c->c_pow = 10.0;                                   /* powf: documented 4 ulp (older toolkits 8) */
    }
}
