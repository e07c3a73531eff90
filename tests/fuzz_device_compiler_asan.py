"""Fuzz of the device's two program compilers on the host under AddressSanitizer (test infrastructure; run by hand, not collected).

compute-sanitizer is refused on this GPU pool, so the memory safety of the compile step (the code that writes variable-length records
into a shared workspace on the device) is checked where it can be: compile_general and the body of k_compile's walk are compiled for the
host too (beagle_debug_compile, beagle_debug_walk: the same source as the kernels), the host build is instrumented by ASan, and random
token streams go through both: uniformly random words, plausible programs of all 26 commands with stray arguments and opcodes, every
length 1..512, random plans (slot rows 0..31, reciprocal and staged rows 0..d), record buffers exactly as large as the documented bound
(len + 1, len + 8 records). Properties asserted beside ASan's own: records <= tokens, depth in 1..32 for what is compiled.
DESIGN.md section 4 records the outcome.

    python tests/fuzz_device_compiler_asan.py [seed] [seconds]
"""
import ctypes
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
LIB = "/tmp/beagle_asan/libbeagle_asan.so"


def build():
    os.makedirs(os.path.dirname(LIB), exist_ok=True)
    subprocess.check_call(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O1", "-g", "-std=c++17", "--fmad=false", "-shared",
                           "-Xcompiler", "-fPIC,-fsanitize=address,-fno-omit-frame-pointer", "-o", LIB,
                           os.path.join(ROOT, "paper_2607_06731_b200", "csrc", "beagle.cu")])


def main():
    import numpy as np
    seed = int(sys.argv[1]) if len(sys.argv) > 1 else 1
    budget = float(sys.argv[2]) if len(sys.argv) > 2 else 60.0
    lib = ctypes.CDLL(LIB)
    i32, i64, vp, u32 = ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p, ctypes.c_uint32
    lib.beagle_debug_walk.argtypes = [vp, i32, vp, i64, i32, i32, i32, i32, i32, u32, i32, vp] + [ctypes.POINTER(i32)] * 4
    lib.beagle_debug_compile.argtypes = [vp, i32, vp, i64, i32, i32, i32, i32, i32, u32, vp] + [ctypes.POINTER(i32)] * 3
    rng = np.random.default_rng(seed)
    ops_valid = np.array([1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11] + list(range(0x10, 0x1F)), np.uint32)
    consts = rng.uniform(-3, 3, 64).astype(np.float32)
    consts[:4] = [0, 1e-7, np.inf, np.nan]
    n_calls = n_taken = n_ok = 0
    t0 = time.time()
    while time.time() - t0 < budget:
        L = int(rng.choice([1, 2, 3, 5, 8, 13, 40, 100, 255, 511, 512])) if rng.random() < 0.5 else int(rng.integers(1, 513))
        mode = rng.random()
        if mode < 0.25:                            # uniformly random words
            tok = rng.integers(0, 2**32, L, dtype=np.uint64).astype(np.uint32)
        else:                                      # plausible programs that mostly stay well-formed
            tok = np.empty(L, np.uint32)
            depth = 0
            for t in range(L):
                if depth < 2 or rng.random() < 0.45:
                    op = 1 if rng.random() < 0.3 else 2
                    arg = int(rng.integers(0, 64 if op == 1 else 8))
                    depth += 1
                else:
                    op = int(rng.choice(ops_valid))
                    arg = 0 if rng.random() < 0.97 else int(rng.integers(0, 40))
                    depth += {3: -1, 4: -1, 5: -1, 6: -1, 0x13: -1, 0x12: -1, 0x10: 1, 0x1E: 1}.get(op, 0)
                if mode > 0.9 and rng.random() < 0.02:
                    op = int(rng.integers(0, 256))
                tok[t] = (arg << 8) | op
        tok = np.ascontiguousarray(tok.view(np.int32))
        d = int(rng.integers(1, 33))
        S_T, k_rcp, k_un = int(rng.integers(0, 32)), int(rng.integers(0, d + 1)), int(rng.integers(0, d + 1))
        n, dep, a, b = i32(), i32(), i32(), i32()
        rec = np.zeros((L + 8, 2), np.uint32)      # the binding's sizes: an overrun is ASan's to find
        for f1 in (0, 1):
            st = lib.beagle_debug_walk(tok.ctypes.data, L, consts.ctypes.data, 64, d, S_T, k_rcp, k_un, 2048, int(rng.integers(0, 2**32)),
                                       f1, rec.ctypes.data, ctypes.byref(n), ctypes.byref(dep), ctypes.byref(a), ctypes.byref(b))
            assert st == 0
            if a.value:
                n_taken += 1
                assert n.value <= L and 1 <= dep.value <= 32, (n.value, L, dep.value)
        rec2 = np.zeros((L + 1, 2), np.uint32)
        st = lib.beagle_debug_compile(tok.ctypes.data, L, consts.ctypes.data, 64, d, S_T, k_rcp, k_un, 2048, int(rng.integers(0, 2**32)),
                                      rec2.ctypes.data, ctypes.byref(n), ctypes.byref(dep), ctypes.byref(a))
        assert st == 0 and n.value <= L and 0 <= dep.value <= 32
        n_ok += dep.value > 0
        n_calls += 1
    print(f"seed {seed}: {n_calls} programs, {n_taken} compiled by the walk, {n_ok} well-formed by the general compiler: no finding")


if __name__ == "__main__":
    if os.environ.get("BEAGLE_ASAN_CHILD") != "1":
        build()
        asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
        env = dict(os.environ, BEAGLE_ASAN_CHILD="1", LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0")
        sys.exit(subprocess.call([sys.executable] + sys.argv, env=env))
    main()
