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
