/* gen.c — seeded synthetic colonies (host harness; serves both the CUDA path and the oracle).
 *
 * Holds NONE of the method's arithmetic: it only draws random program SHAPES and packs them as
 * {opcode:8,arg:24} postfix tokens (R2). Recipe: DESIGN.md §5.
 *   RNG      SplitMix64, one stream per individual: state0 = seed ^ ((p+1) * 0x9E3779B97F4A7C15),
 *            u = (next >> 11) * 2^-53.
 *   G-tree   ramped half-and-half trees (configs 1-4), emitted in postfix.
 *   G-len    exact-length linear sampler with Zipf(1) lengths on 1..512 (config 5), plus the four
 *            designed-invalid suffixes.
 *   f1 mix   (bench.py --gcl-mix f1) G-tree with the paper's stack commands woven in (Table 3): a binary node
 *            becomes `A DUP op` (both operands the same subtree) with probability 0.15 or gets a SWAP in front of its
 *            command with probability 0.15; a terminal becomes `t t' DEL` with probability 0.05. Programs stay
 *            well-formed and within the token cap. SIGN SQUARE CUBE come in through the caller's unary set.
 * Constants: the k-th CONST token in population order gets index k mod 2^24 of the side table.
 */
#include <stdint.h>
#include <string.h>
#include <math.h>

enum { OP_CONST = 1, OP_LOAD = 2, OP_ADD = 3, OP_SUB = 4, OP_MUL = 5, OP_DIV = 6,
       OP_SIN = 7, OP_COS = 8, OP_LOG = 9, OP_SQRT = 10, OP_EXP = 11, OP_DUP = 0x10, OP_SWAP = 0x11, OP_DEL = 0x12 };
#define TOK(op, arg) ((int32_t)(((uint32_t)(arg) << 8) | (uint32_t)(op)))
#define MAXC (1 << 24)

typedef struct { uint64_t s; } rng_t;
static inline uint64_t rng_next(rng_t* r) {
    uint64_t z = (r->s += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
static inline double rng_u(rng_t* r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }
static inline int rng_int(rng_t* r, int n) { int k = (int)(rng_u(r) * n); return k < n ? k : n - 1; }

typedef struct {
    int n_un, n_bin, d, f1;
    int un[16], bin[8];
    double q_u, clo, chi;
} opset_t;

typedef struct {
    int32_t tok[520];
    float   cval[520];   /* value of the j-th CONST token of this individual */
    int     n, nc;
} prog_t;

static void emit_terminal(prog_t* g, rng_t* r, const opset_t* o) {
    int k = rng_int(r, o->d + 1);
    if (k < o->d) g->tok[g->n++] = TOK(OP_LOAD, k);
    else {
        double c = o->clo + (o->chi - o->clo) * rng_u(r);
        g->cval[g->nc++] = (float)c;
        g->tok[g->n++] = TOK(OP_CONST, 0); /* index patched by the caller */
    }
}
static void emit_const(prog_t* g, float c) { g->cval[g->nc++] = c; g->tok[g->n++] = TOK(OP_CONST, 0); }

/* returns the number of tokens emitted for this subtree */
static int gen_tree(prog_t* g, rng_t* r, const opset_t* o, int depth_left, int budget, int grow, int root) {
    int start = g->n;
    if (depth_left == 0 || budget < 2 || (grow && !root && rng_u(r) < 0.3)) {
        emit_terminal(g, r, o);
        if (o->f1 && budget >= 3 && rng_u(r) < 0.05) { emit_terminal(g, r, o); g->tok[g->n++] = TOK(OP_DEL, 0); }
        return g->n - start;
    }
    int unary = (budget < 3) ? 1 : (rng_u(r) < o->q_u);
    if (unary) {
        int op = o->un[rng_int(r, o->n_un)];
        gen_tree(g, r, o, depth_left - 1, budget - 1, grow, 0);
        g->tok[g->n++] = TOK(op, 0);
    } else {
        int op = o->bin[rng_int(r, o->n_bin)];
        int lb = (budget - 1 + 1) / 2;           /* ceil((budget-1)/2) */
        if (lb > budget - 2) lb = budget - 2;
        double f = o->f1 ? rng_u(r) : 1.0;
        if (f < 0.15) {                          /* A DUP op */
            gen_tree(g, r, o, depth_left - 1, lb, grow, 0);
            g->tok[g->n++] = TOK(OP_DUP, 0);
        } else if (f < 0.30 && budget >= 4) {    /* A B SWAP op */
            if (lb > budget - 3) lb = budget - 3;
            int ls = gen_tree(g, r, o, depth_left - 1, lb, grow, 0);
            gen_tree(g, r, o, depth_left - 1, budget - 2 - ls, grow, 0);
            g->tok[g->n++] = TOK(OP_SWAP, 0);
        } else {
            int ls = gen_tree(g, r, o, depth_left - 1, lb, grow, 0);
            gen_tree(g, r, o, depth_left - 1, budget - 1 - ls, grow, 0);
        }
        g->tok[g->n++] = TOK(op, 0);
    }
    return g->n - start;
}

/* exact-length linear sampler: classes {terminal .375, unary .25, binary .375} restricted to the
 * feasible ones (depth in [1,32] after the token, and the remaining tokens can bring it to 1). */
static void gen_len(prog_t* g, rng_t* r, const opset_t* o, int L) {
    int s = 0;
    for (int t = 0; t < L; ++t) {
        int rem = L - t - 1;
        double wt = (s + 1 <= 32 && s <= rem) ? 0.375 : 0.0;
        double wu = (s >= 1 && s - 1 <= rem) ? 0.25 : 0.0;
        double wb = (s >= 2) ? 0.375 : 0.0;
        double x = rng_u(r) * (wt + wu + wb);
        if (x < wt) { emit_terminal(g, r, o); s++; }
        else if (x < wt + wu) g->tok[g->n++] = TOK(o->un[rng_int(r, o->n_un)], 0);
        else { g->tok[g->n++] = TOK(o->bin[rng_int(r, o->n_bin)], 0); s--; }
    }
}

static void emit_B(prog_t* g) { /* C100 EXP C100 EXP MUL = +inf in fp32 range */
    emit_const(g, 100.0f); g->tok[g->n++] = TOK(OP_EXP, 0);
    emit_const(g, 100.0f); g->tok[g->n++] = TOK(OP_EXP, 0);
    g->tok[g->n++] = TOK(OP_MUL, 0);
}

static int zipf_len(rng_t* r, const double* cdf, int n) {
    double u = rng_u(r) * cdf[n - 1];
    int lo = 0, hi = n - 1;
    while (lo < hi) { int m = (lo + hi) / 2; if (cdf[m] > u) hi = m; else lo = m + 1; }
    return lo + 1;
}

/* colony_generate — kind 0 = G-tree, 1 = G-len.
 * First call with tokens == NULL to get lengths[P] and the totals (*T_out, *C_out); then call
 * again with tokens (T words) and consts (min(C, 2^24) floats). Returns 0.                    */
int colony_generate(int kind, uint64_t seed, int64_t P, int dmin, int dmax, int lcap,
                    const int* un, int n_un, const int* bin, int n_bin, double q_u,
                    int d, double clo, double chi, int designed_invalid, int f1_mix,
                    int32_t* lengths, int32_t* tokens, float* consts,
                    int64_t* T_out, int64_t* C_out) {
    opset_t o; memset(&o, 0, sizeof o);
    o.n_un = n_un; o.n_bin = n_bin; o.d = d; o.q_u = q_u; o.clo = clo; o.chi = chi; o.f1 = f1_mix;
    for (int i = 0; i < n_un; ++i) o.un[i] = un[i];
    for (int i = 0; i < n_bin; ++i) o.bin[i] = bin[i];
    double cdf[512]; double acc = 0.0;
    for (int k = 1; k <= 512; ++k) { acc += 1.0 / k; cdf[k - 1] = acc; }
    int R = dmax - dmin + 1;
    int64_t T = 0, C = 0;
    prog_t g;
    for (int64_t p = 0; p < P; ++p) {
        rng_t r; r.s = seed ^ ((uint64_t)(p + 1) * 0x9E3779B97F4A7C15ull);
        g.n = 0; g.nc = 0;
        if (kind == 0) {
            int depth = dmin + (int)(p % R);
            int grow = (int)((p / R) & 1);
            gen_tree(&g, &r, &o, depth, lcap, grow, 1);
        } else {
            int L = zipf_len(&r, cdf, lcap < 512 ? lcap : 512);
            if (designed_invalid && (p % 20) == 0 && L >= 16) {
                int which = (int)((p / 20) & 3);
                static const int suf[4] = { 6, 12, 3, 10 };
                gen_len(&g, &r, &o, L - suf[which]);
                if (which == 0) { emit_B(&g); g.tok[g.n++] = TOK(OP_ADD, 0); }
                else if (which == 1) { emit_B(&g); emit_B(&g); g.tok[g.n++] = TOK(OP_SUB, 0);
                                       g.tok[g.n++] = TOK(OP_ADD, 0); }
                else if (which == 2) { emit_const(&g, 69.0f); g.tok[g.n++] = TOK(OP_EXP, 0);
                                       g.tok[g.n++] = TOK(OP_ADD, 0); }
                else {
                    g.tok[g.n++] = TOK(OP_LOAD, rng_int(&r, d));
                    emit_const(&g, 2.0f); g.tok[g.n++] = TOK(OP_SUB, 0);
                    emit_const(&g, 1.0e4f); g.tok[g.n++] = TOK(OP_MUL, 0);
                    g.tok[g.n++] = TOK(OP_EXP, 0);
                    emit_const(&g, 100.0f); g.tok[g.n++] = TOK(OP_EXP, 0);
                    g.tok[g.n++] = TOK(OP_MUL, 0); g.tok[g.n++] = TOK(OP_ADD, 0);
                }
            } else gen_len(&g, &r, &o, L);
        }
        lengths[p] = g.n;
        if (tokens) {
            int j = 0;
            for (int t = 0; t < g.n; ++t) {
                int32_t w = g.tok[t];
                if ((w & 0xFF) == OP_CONST) {
                    int64_t k = C + j;
                    if (k < MAXC) consts[k] = g.cval[j];
                    w = TOK(OP_CONST, (uint32_t)(k % MAXC));
                    j++;
                }
                tokens[T + t] = w;
            }
        }
        T += g.n; C += g.nc;
    }
    *T_out = T; *C_out = C;
    return 0;
}
