"""The seeded synthetic colonies are what DESIGN.md §5 says they are (-m "not gpu"): every program of every config is a program
(well-formed by the oracle's static check, final depth 1 for the tree configs), lengths stay under the config's cap, the realised
sizes are the ones BASELINE.md / bench.py quote, and the f1 mix really speaks the paper's extra commands."""
import numpy as np
import pytest

from paper_2607_06731_b200 import colonies as C


def _depth_walk(tokens, lengths):
    """Stack effect of every program, vectorised per program (plain Python: small samples only)."""
    delta = np.zeros(256, np.int64)
    for n in ("CONST", "LOAD", "DUP", "PASTE"):
        delta[C.OP[n]] = 1
    for n in ("ADD", "SUB", "MUL", "DIV", "POW", "DEL"):
        delta[C.OP[n]] = -1
    ops = tokens.view(np.uint32) & 0xFF
    off = np.concatenate(([0], np.cumsum(lengths)))
    final, deepest = [], []
    for p in range(len(lengths)):
        run = np.cumsum(delta[ops[off[p]:off[p + 1]]])
        final.append(int(run[-1])); deepest.append(int(run.max()))
    return np.array(final), np.array(deepest)


@pytest.mark.parametrize("number", [1, 2, 3, 4, 5])
def test_every_generated_program_is_a_program(oracle, number):
    cfg = C.CONFIGS[number]
    P = min(cfg.P, 3000)
    tokens, lengths, consts = C.generate_programs(cfg, P)
    assert lengths.min() >= 1 and lengths.max() <= cfg.lcap and tokens.shape[0] == lengths.sum()
    X, y, _ = C.make_dataset(cfg)
    assert X.shape == (cfg.N, cfg.d) and y.shape == (cfg.N,) and X.dtype == np.float32
    r = oracle.evaluate(tokens, lengths, consts, X[:4], y[:4], cfg.tax)          # 4 cases: the static check is what is wanted
    assert not np.any(r["flags"] & oracle.FLAG_MALFORMED)
    final, deepest = _depth_walk(tokens, lengths)
    assert np.array_equal(deepest, r["depth"]) and deepest.max() <= 32
    if cfg.kind == 0:
        assert np.all(final == 1)                                # trees leave exactly their root
    else:
        assert np.all(final >= 1)
    # only the commands the config names, and terminals
    ops = set(np.unique(tokens.view(np.uint32) & 0xFF).tolist())
    assert ops <= set(cfg.unary) | set(cfg.binary) | {C.OP["CONST"], C.OP["LOAD"]}
    args = tokens.view(np.uint32) >> 8
    is_load = (tokens.view(np.uint32) & 0xFF) == C.OP["LOAD"]
    is_const = (tokens.view(np.uint32) & 0xFF) == C.OP["CONST"]
    assert args[is_load].max() < cfg.d and args[is_const].max() < len(consts) and not args[~is_load & ~is_const].any()
    # (config 5 plants overflowing suffixes on every 20th long program: their constants 69, 100, 10000 are not drawn)
    drawn = consts[~np.isin(consts, [69.0, 100.0, 10000.0])] if cfg.designed_invalid else consts
    assert np.all((drawn >= cfg.clo) & (drawn <= cfg.chi))


def test_config3_is_the_workload_the_bench_line_names():
    cfg = C.CONFIGS[3]
    tokens, lengths, consts = C.generate_programs(cfg)
    assert lengths.shape[0] == 1_048_576 and tokens.shape[0] == 38_607_086          # bench.py: config.tokens; BASELINE.md §4
    assert tokens.shape[0] * cfg.N == 19_766_828_032                                # gp_ops_per_step
    assert abs(lengths.mean() - 36.8) < 0.05 and lengths.max() <= 128
    st = C.colony_stats(tokens, lengths)
    assert st


def test_f1_mix_speaks_the_papers_extra_commands(oracle):
    cfg = C.CONFIGS[3]
    P = 20000
    tokens, lengths, consts = C.generate_programs(cfg, P, gcl_mix="f1")
    hot_tokens, hot_lengths, _ = C.generate_programs(cfg, P)
    ops = tokens.view(np.uint32) & 0xFF
    f1 = np.isin(ops, [C.OP[n] for n in ("DUP", "SWAP", "DEL", "SIGN", "SQUARE", "CUBE")])
    assert 0.12 < f1.mean() < 0.22                                                  # 17 % of the tokens
    off = np.concatenate(([0], np.cumsum(lengths)))
    uses = np.add.reduceat(f1.astype(np.int64), off[:-1]) > 0
    assert uses.mean() > 0.8                                                        # 88 % of the programs use at least one
    assert lengths.max() <= cfg.lcap
    X, y, _ = C.make_dataset(cfg)
    r = oracle.evaluate(tokens, lengths, consts, X[:4], y[:4], cfg.tax)
    assert not np.any(r["flags"] & oracle.FLAG_MALFORMED)
    # the hot colony of the same seed is untouched by the option
    again, again_l, _ = C.generate_programs(cfg, P)
    assert np.array_equal(again, hot_tokens) and np.array_equal(again_l, hot_lengths)


def _tree_depths(tokens, lengths, cfg):
    """Depth of the expression tree a postfix program spells (root = depth 0, R17). Plain Python: small samples only."""
    ops = tokens.view(np.uint32) & 0xFF
    un, bi = set(cfg.unary), set(cfg.binary)
    off = np.concatenate(([0], np.cumsum(lengths)))
    out = []
    for p in range(len(lengths)):
        st = []
        for o in ops[off[p]:off[p + 1]].tolist():
            if o in un:
                st[-1] += 1
            elif o in bi:
                b = st.pop(); a = st.pop(); st.append(max(a, b) + 1)
            else:
                st.append(0)
        out.append(st[-1])
    return np.array(out)


@pytest.mark.parametrize("number,q_lo,q_hi", [(1, 0.17, 0.23), (2, 0.19, 0.26), (3, 0.20, 0.27), (4, 0.39, 0.46)])
def test_tree_configs_are_ramped_half_and_half_with_the_stated_mix(number, q_lo, q_hi):
    """SURVEY.md §8(d) / DESIGN.md §5: individual p gets depth Dmin + (p mod R), 'full' when floor(p / R) is even, else 'grow';
    a function node is unary with probability q_u (forced when two tokens are left, hence a little above it); a terminal is
    uniform over the d variables and 'a constant'."""
    cfg = C.CONFIGS[number]
    P = 6000
    tokens, lengths, _ = C.generate_programs(cfg, P)
    depth = _tree_depths(tokens, lengths, cfg)
    R = cfg.dmax - cfg.dmin + 1
    p = np.arange(P)
    assigned = cfg.dmin + p % R
    full = (p // R) % 2 == 0
    assert np.all(depth <= assigned)
    assert np.mean(depth[full] == assigned[full]) > 0.99          # (the token budget cuts a handful of the deepest full trees short)
    assert 0.6 < np.mean(depth[~full] / assigned[~full]) < 0.95   # grow: terminals come early with probability 0.3 per node
    ops = tokens.view(np.uint32) & 0xFF
    isu, isb = np.isin(ops, list(cfg.unary)), np.isin(ops, list(cfg.binary))
    assert q_lo < isu.sum() / (isu.sum() + isb.sum()) < q_hi
    n_const, n_load = int((ops == C.OP["CONST"]).sum()), int((ops == C.OP["LOAD"]).sum())
    assert abs(n_const / (n_const + n_load) - 1.0 / (cfg.d + 1)) < 0.01
    loads = (tokens.view(np.uint32) >> 8)[ops == C.OP["LOAD"]]
    share = np.bincount(loads, minlength=cfg.d) / len(loads)
    assert np.all(np.abs(share - 1.0 / cfg.d) < 0.02)             # every variable equally often


def test_config5_lengths_follow_the_zipf_law_and_its_designed_invalid_programs_are_invalid(oracle):
    """Config 5 (BASELINE.json: 'heavy-tailed lengths 1-512 tokens (Zipf-like)', '5 % are designed to produce NaN/inf'):
    P(L = k) proportional to 1 / k on 1..512 (mean 512 / H_512 = 75.1 tokens: what makes 4 M programs 1.26 GB and a 1 GB budget
    force chunking); every 20th individual, if it has 16 tokens or more, ends in an overflowing suffix."""
    cfg = C.CONFIGS[5]
    P = 200_000
    tokens, lengths, consts = C.generate_programs(cfg, P)
    H = np.sum(1.0 / np.arange(1, 513))
    assert abs(lengths.mean() - 512.0 / H) < 1.0
    assert abs(np.mean(lengths == 1) - 1.0 / H) < 0.004
    assert abs(np.mean(lengths >= 256) - np.sum(1.0 / np.arange(256, 513)) / H) < 0.004
    assert lengths.min() == 1 and lengths.max() == 512
    ops = tokens.view(np.uint32) & 0xFF
    isu, isb = np.isin(ops, list(cfg.unary)).mean(), np.isin(ops, list(cfg.binary)).mean()
    assert abs(isu - 0.25) < 0.02 and abs(isb - 0.375) < 0.02     # classes {terminal .375, unary .25, binary .375}, feasibility-restricted
    # the designed-invalid ones: the oracle calls every one of them non-finite on the config's own cases, and they are
    # 5 % of the long-enough programs
    n = 40_000
    off = np.concatenate(([0], np.cumsum(lengths[:n], dtype=np.int64)))
    sel = np.array([p for p in range(0, n, 20) if lengths[p] >= 16])
    assert abs(len(sel) / np.count_nonzero(lengths[:n] >= 16) - 0.05) < 0.005
    g = np.concatenate([tokens[off[p]:off[p + 1]] for p in sel])
    X, y, _ = C.make_dataset(cfg)
    r = oracle.evaluate_parallel(g, lengths[sel], consts, X, y, cfg.tax)
    assert not np.any(r["flags"] & oracle.FLAG_MALFORMED)
    assert not np.any(np.isfinite(r["fitness"])), int(np.isfinite(r["fitness"]).sum())


def test_datasets_are_the_distributions_baseline_json_names():
    """x ranges and targets of the five configs (BASELINE.json 'configs'), recomputed from the rounded inputs."""
    X, y, _ = C.make_dataset(C.CONFIGS[1])
    assert X.min() >= -1 and X.max() <= 1 and abs(X.mean()) < 0.05
    assert np.allclose(y, X[:, 0].astype(np.float64) ** 2 + np.sin(X[:, 1].astype(np.float64)), rtol=0, atol=1e-6)
    X, y, _ = C.make_dataset(C.CONFIGS[2])
    assert X.min() >= -3 and X.max() <= 3 and abs(X.mean()) < 0.1
    X64 = X.astype(np.float64)
    noise = y - X64[:, 0] * X64[:, 1] / (1.0 + X64[:, 2] ** 2)
    assert abs(noise.mean()) < 0.002 and 0.008 < noise.std() < 0.012              # + 0.01 N(0, 1)
    X, y, _ = C.make_dataset(C.CONFIGS[3])
    assert X.min() >= 1 and X.max() <= 5 and abs(X.mean() - 3.0) < 0.05
    X64 = X.astype(np.float64)
    assert np.allclose(y, X64[:, 0] * X64[:, 1] * np.exp(-X64[:, 2] / X64[:, 3]) + X64[:, 4], rtol=1e-5, atol=0)
    for number in (4, 5):
        X, y, expr = C.make_dataset(C.CONFIGS[number])
        assert X.shape == (1024, 9) and X.min() >= 1 and X.max() <= 5
        assert abs(np.log(X.astype(np.float64)).mean() - np.log(5.0) / 2) < 0.03  # log-uniform in [1, 5]
        assert np.all(np.isfinite(y)) and np.ptp(y) > 1e-3                         # finite on all cases and not constant
        nodes = len([w for w in expr.replace("(", " ").replace(")", " ").split() if w])
        assert 6 <= nodes <= 12, (expr, nodes)                                     # 'a seeded random 6-12-node closed-form expression'
