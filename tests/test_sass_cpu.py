"""CPU-only: the built library is what DESIGN.md section 7 says it is, read from its SASS (cuobjdump, no GPU needed).

The interpreter's operands and operand stack live in tensor memory (LDTM / STTM = tcgen05.ld / st, UTCATOMSWS = tcgen05.alloc /
dealloc), its micro-op records arrive by TMA bulk copies (UBLKCP) on mbarriers (SYNCS), and a micro-op is dispatched by ONE indexed
branch on the uniform datapath (BRXU). A build that lost one of these (a compiler change, an edit that makes ptxas fall back to a
per-thread branch or to local memory) would still pass parity and only show up as a slower bench: this test names it.
profiles/r2_sass_static.md is the table these counts come from.
"""
import collections
import re
import shutil
import subprocess

import pytest

from paper_2607_06731_b200 import api


@pytest.fixture(scope="module")
def sass():
    if shutil.which("cuobjdump") is None or shutil.which("c++filt") is None:
        pytest.skip("cuobjdump / c++filt not on PATH")
    lib = api._build.build()
    text = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    res = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    kernels = {}
    for f in text.split("\t\tFunction : ")[1:]:
        mangled = f.split("\n")[0].strip()
        name = subprocess.run(["c++filt", mangled], capture_output=True, text=True).stdout.strip()
        name = name.split("(")[0].replace("void ", "").replace("beagle::", "")
        ins = re.findall(r"^\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_]+)", f, flags=re.M)
        m = re.search(r"Function %s:\n\s+REG:(\d+) STACK:(\d+) SHARED:(\d+)" % re.escape(mangled), res)
        kernels[name] = dict(count=collections.Counter(ins), total=len(ins), reg=int(m.group(1)), stack=int(m.group(2)))
    return kernels


def test_every_interpreter_instantiation_uses_tensor_memory_tma_and_one_uniform_dispatch(sass):
    evals = {k: v for k, v in sass.items() if k.startswith("k_eval<")}
    assert len(evals) == 6, sorted(evals)          # MSE (plain, grouped x 3 pass modes), correlation, Std
    for name, k in evals.items():
        c = k["count"]
        assert c["LDTM"] >= 20 and c["STTM"] >= 20, (name, c["LDTM"], c["STTM"])       # operands and slots in tensor memory
        assert c["UTCATOMSWS"] >= 2, name                                              # tcgen05.alloc and dealloc
        assert c["UBLKCP"] == 1, (name, c["UBLKCP"])                                   # one bulk-copy site: the group fetch
        assert c["SYNCS"] >= 3, name                                                   # mbarrier init / expect_tx / try_wait
        assert c["BRXU"] == 1 and c["BRX"] == 0, (name, c["BRXU"], c["BRX"])           # one dispatch site, on the uniform datapath
        assert c["WARPSYNC"] <= 1, (name, c["WARPSYNC"])                               # the tcgen05 operations are known warp-uniform
        assert k["reg"] <= 64, (name, k["reg"])                                        # 1024 threads per block fit
        assert k["stack"] <= 2048, (name, k["stack"])                                  # the 31 memory slots (1984 bytes) and nothing else


def test_the_compiler_walk_stays_within_its_register_budget(sass):
    for name in ("k_compile<false>", "k_compile<true>"):
        k = sass[name]
        assert k["reg"] <= 80, (name, k["reg"])                                        # 6 blocks of 128 threads per SM
        assert k["stack"] <= 32, (name, k["stack"])                                    # a few words spilled outside the loop, no more
        assert k["count"]["BRX"] == 0 and k["count"]["BRXU"] == 0, name               # table-driven: no indexed branch in the walk
    assert sass["k_compile<true>"]["total"] > sass["k_compile<false>"]["total"]        # the f1 branch is only in the one instantiation


def test_the_prior_art_kernel_uses_neither(sass):
    c = sass["k_eval_blockwise"]["count"]
    assert c["LDTM"] == 0 and c["STTM"] == 0 and c["UBLKCP"] == 0
