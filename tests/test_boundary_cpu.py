"""CPU-only checks of the boundary and of the host logic (no compute calls, no GPU):
- the C-ABI library builds, loads, and exports every symbol include/beagle.h declares;
- the binding declares the same set; the calls that need no device behave (limits, status strings,
  synchronous argument errors);
- token packing round-trips, including arg = 2^24 - 1;
- bench.py's multi-rank plumbing (sum of units / max time over ranks) on a world_size-2 gloo group.
"""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2607_06731_b200 import api, colonies

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "beagle.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(beagle_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = _declared()
    assert "beagle_eval" in names and "beagle_eval_chunked" in names
    l = ctypes.CDLL(api._build.build())
    for n in names:
        assert hasattr(l, n), f"{n} declared in include/beagle.h but not exported"
    assert sorted(api.EXPORTS) == names, "binding and header disagree"


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "beagle.h"\nint main(void){return BEAGLE_TOKEN(BEAGLE_OP_LOAD,3)==0x302?0:1;}\n')
    exe = tmp_path / "t"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    assert subprocess.call([str(exe)]) == 0


def test_limits_and_status_strings_without_device():
    assert api.beagle_limits() == dict(max_len=512, max_stack=32, max_n=1024, max_d=32)
    for s in (0, -1, -2, -3, -4, -99):
        assert isinstance(api.beagle_status_string(s), str) and api.beagle_status_string(s)


def test_argument_errors_are_synchronous_without_device():
    l = api.lib()
    one = ctypes.c_int32(0)
    p = ctypes.addressof(one)
    # P < 0, N out of range, d out of range, consts NULL with n_consts > 0, NULL data with P > 0
    assert l.beagle_eval(p, p, -1, None, 0, p, p, 4, 1, 0.0, p, None) == api.ERR_INVALID_ARG
    assert l.beagle_eval(p, p, 1, None, 0, p, p, 0, 1, 0.0, p, None) == api.ERR_INVALID_ARG
    assert l.beagle_eval(p, p, 1, None, 0, p, p, 1025, 1, 0.0, p, None) == api.ERR_INVALID_ARG
    assert l.beagle_eval(p, p, 1, None, 0, p, p, 4, 33, 0.0, p, None) == api.ERR_INVALID_ARG
    assert l.beagle_eval(p, p, 1, None, 1, p, p, 4, 1, 0.0, p, None) == api.ERR_INVALID_ARG
    assert l.beagle_eval(None, p, 1, None, 0, p, p, 4, 1, 0.0, p, None) == api.ERR_INVALID_ARG
    assert l.beagle_eval_chunked(p, p, 1, None, 0, p, p, 4, 1, 0.0, p, 100, None) == api.ERR_INVALID_ARG
    assert l.beagle_reserve(-1, 0) == api.ERR_INVALID_ARG
    # P == 0 is OK and enqueues nothing, device or not
    assert l.beagle_eval(None, None, 0, None, 0, None, None, 4, 1, 0.0, None, None) == api.OK
    assert api.beagle_last_launch_count() == 0


def test_token_round_trip():
    for op in colonies.OP.values():
        for arg in (0, 1, 255, 256, 65535, (1 << 24) - 1):
            w = np.array([colonies.token(op, arg)], np.int32).view(np.uint32)[0]
            assert int(w & 0xFF) == op and int(w >> 8) == arg


def test_seed_offset_gives_a_different_colony_of_the_same_shape():
    cfg = colonies.CONFIGS[3]
    a = colonies.generate_programs(cfg, 2000)
    b = colonies.generate_programs(cfg, 2000, seed_offset=0x10000)
    a2 = colonies.generate_programs(cfg, 2000)
    assert np.array_equal(a[0], a2[0]) and np.array_equal(a[1], a2[1])
    assert not np.array_equal(a[1], b[1])
    assert abs(a[1].mean() - b[1].mean()) < 0.15 * a[1].mean()


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import bench
rank, local_rank, world = bench.dist_init("gloo")
units = 1000 * (rank + 1)                 # rank 0: 1000 units/step, rank 1: 2000
ms = 10.0 if rank == 0 else 40.0          # the slower rank decides
value, ms_max = bench.job_throughput(units, 4, ms, world)
bench.dist_barrier(world)
assert world == 2 and ms_max == 40.0, (world, ms_max)
assert abs(value - (4 * 3000) / 0.040) < 1e-6, value
assert bench.rank_seed_offset(rank) == 0x10000 * rank
print("ok", rank)
"""


def test_bench_multi_rank_plumbing_gloo(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=ROOT))
    port = 29600 + (os.getpid() % 300)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for p in procs:
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0, out
        assert "ok" in out


def test_bench_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def _c_constants(path, pattern):
    """name -> int for every `NAME = value` / `#define NAME value` in a C source that matches `pattern` (comments stripped)."""
    text = re.sub(r"/\*.*?\*/", "", open(path).read(), flags=re.S)
    out = {}
    for name, val in re.findall(pattern, text):
        out[name] = int(val, 0)
    return out


def test_retyped_constants_agree_everywhere():
    """The opcode numbers, limits, status codes and fitness selectors are typed out in several places that must not share code
    (the header, the binding, the input generators, the oracle: 'numbers retyped, not shared'): they have to stay the same numbers."""
    hdr = os.path.join(ROOT, "include", "beagle.h")
    ops_h = {k[len("BEAGLE_OP_"):]: v for k, v in _c_constants(hdr, r"#define\s+(BEAGLE_OP_[A-Z]+)\s+(0x[0-9A-Fa-f]+|\d+)").items()}
    assert len(ops_h) == 26 and ops_h == colonies.OP                                     # header == generators / test assembler
    ops_o = {k[len("OP_"):]: v for k, v in _c_constants(os.path.join(ROOT, "oracle", "beagle_oracle.c"),
                                                        r"\b(OP_[A-Z]+)\s*=\s*(0x[0-9A-Fa-f]+|\d+)").items()}
    assert ops_o == ops_h                                                                # == the oracle's own enum
    ops_g = {k[len("OP_"):]: v for k, v in _c_constants(os.path.join(ROOT, "paper_2607_06731_b200", "colonies", "gen.c"),
                                                        r"\b(OP_[A-Z]+)\s*=\s*(0x[0-9A-Fa-f]+|\d+)").items()}
    assert ops_g and all(ops_h[k] == v for k, v in ops_g.items())                        # the C generator names a subset
    lim = _c_constants(hdr, r"#define\s+(BEAGLE_MAX_[A-Z]+)\s+(\d+)")
    assert (lim["BEAGLE_MAX_LEN"], lim["BEAGLE_MAX_STACK"], lim["BEAGLE_MAX_N"], lim["BEAGLE_MAX_D"], lim["BEAGLE_MAX_VARS"]) == (512, 32, 1024, 32, 32)
    olim = _c_constants(os.path.join(ROOT, "oracle", "beagle_oracle.c"), r"#define\s+(ORC_MAX_[A-Z]+)\s+(\d+)")
    assert (olim["ORC_MAX_LEN"], olim["ORC_MAX_STACK"], olim["ORC_MAX_N"], olim["ORC_MAX_VARS"]) == (512, 32, 1024, 32)
    st = _c_constants(hdr, r"\b(BEAGLE_(?:OK|ERR_[A-Z_]+))\s*=\s*(-?\d+)")
    assert st == dict(BEAGLE_OK=api.OK, BEAGLE_ERR_INVALID_ARG=api.ERR_INVALID_ARG, BEAGLE_ERR_UNSUPPORTED=api.ERR_UNSUPPORTED,
                      BEAGLE_ERR_CUDA=api.ERR_CUDA, BEAGLE_ERR_NOMEM=api.ERR_NOMEM, BEAGLE_ERR_NOT_RESERVED=api.ERR_NOT_RESERVED)
    for s in st.values():
        assert api.beagle_status_string(s) != "unknown status"
    fit = _c_constants(hdr, r"#define\s+(BEAGLE_FIT_[A-Z_]+)\s+(\d+)")
    assert fit == dict(BEAGLE_FIT_MSE=api.FIT_MSE, BEAGLE_FIT_CORRELATION=api.FIT_CORRELATION, BEAGLE_FIT_STD=api.FIT_STD,
                       BEAGLE_FIT_STD_SQUARE=api.FIT_STD_SQUARE, BEAGLE_FIT_STD_CUBE=api.FIT_STD_CUBE, BEAGLE_FIT_STD_HYPER=api.FIT_STD_HYPER)
    # Table 2, typed out in the header, the binding and the ranking oracle
    m = re.search(r"BEAGLE_TABLE2\[10\]\s*=\s*\{([^}]*)\}", open(hdr).read())
    table_h = tuple(float(x.strip().rstrip("f")) for x in m.group(1).split(","))
    from oracle import ranking
    assert table_h == api.TABLE2 == tuple(float(x) for x in ranking.EXPECTED_CHILDREN)
    assert abs(sum(table_h) / 10 - 1.0) < 1e-12                                          # the paper's table averages one child
