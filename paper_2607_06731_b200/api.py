"""Thin ctypes binding of libbeagle_b200.so (include/beagle.h) — argument marshalling only.

Every function has the name and argument order of its C entry point; tensors are passed as raw
pointers (`tensor.data_ptr()`), streams as `torch.cuda.current_stream().cuda_stream`. PyTorch
supplies device memory and streams, nothing else: every step of the path runs in the library's
kernels. There is no CPU fallback: if the library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

OK = 0
ERR_INVALID_ARG = -1
ERR_UNSUPPORTED = -2
ERR_CUDA = -3
ERR_NOMEM = -4
ERR_NOT_RESERVED = -5


class BeagleError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().beagle_status_string(status).decode()
        extra = f" (cudaError {lib().beagle_last_cuda_error()})" if status in (ERR_CUDA, ERR_NOMEM) else ""
        super().__init__(f"{where}: {msg}{extra}")


_lib = None
_i32, _i64, _f32, _vp = ctypes.c_int32, ctypes.c_int64, ctypes.c_float, ctypes.c_void_p

_SIGNATURES = {
    "beagle_eval": (_i32, [_vp, _vp, _i64, _vp, _i64, _vp, _vp, _i32, _i32, _f32, _vp, _vp]),
    "beagle_eval_fit": (_i32, [_vp, _vp, _i64, _vp, _i64, _vp, _vp, _i32, _i32, _i32, _f32, _f32, _vp, _vp]),
    "beagle_eval_chunked": (_i32, [_vp, _vp, _i64, _vp, _i64, _vp, _vp, _i32, _i32, _f32, _vp, _i64, _vp]),
    "beagle_eval_chunked_fit": (_i32, [_vp, _vp, _i64, _vp, _i64, _vp, _vp, _i32, _i32, _i32, _f32, _f32, _vp, _i64, _vp]),
    "beagle_rank": (_i32, [_vp, _i64, _vp, _i32, _i32, _vp, _vp, _vp]),
    "beagle_eval_blockwise": (_i32, [_vp, _vp, _i64, _vp, _i64, _vp, _vp, _i32, _i32, _f32, _vp, _vp]),
    "beagle_debug_outputs": (_i32, [_vp, _vp, _i64, _vp, _i64, _vp, _i32, _i32, _vp, _vp]),
    "beagle_debug_schedule": (_i32, [_i64, _vp, _vp, _vp, _vp]),
    "beagle_debug_counts": (_i32, [ctypes.POINTER(_i32)] * 4 + [_vp]),
    "beagle_debug_plan": (_i32, [_i32, _i32, _i32, _i32, _i32, ctypes.POINTER(_i32)]),
    "beagle_debug_chunk_plan": (_i32, [_vp, _i64, _i64, _vp, _i64, ctypes.POINTER(_i64), ctypes.POINTER(_i32), ctypes.POINTER(_i64)]),
    "beagle_debug_compile": (_i32, [_vp, _i32, _vp, _i64, _i32, _i32, _i32, _i32, _i32, ctypes.c_uint32, _vp,
                                    ctypes.POINTER(_i32), ctypes.POINTER(_i32), ctypes.POINTER(_i32)]),
    "beagle_debug_corr": (_i32, [_vp, _vp, _i32, _i32, _f32, _f32, _i32, ctypes.POINTER(_f32)]),
    "beagle_debug_rank": (_i32, [_vp, _i64, _vp, _i32, _i32, _i32, _vp, _vp]),
    "beagle_debug_prepass": (_i32, [_vp, _i64, _vp, _vp, _i32, _i32, _i32, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "beagle_debug_queue": (_i32, [_vp, _i32, _i32, _i32, _i32, _i32, _i32, ctypes.c_uint32, ctypes.c_uint32, _vp, _i32,
                                  ctypes.POINTER(_i32), ctypes.POINTER(_i32)]),
    "beagle_debug_walk": (_i32, [_vp, _i32, _vp, _i64, _i32, _i32, _i32, _i32, _i32, ctypes.c_uint32, _i32, _vp,
                                 ctypes.POINTER(_i32), ctypes.POINTER(_i32), ctypes.POINTER(_i32), ctypes.POINTER(_i32)]),
    "beagle_debug_std_reward": (_i32, [_vp, _vp, _i64, _i32, _f32, _vp]),
    "beagle_debug_walk_tables": (None, [ctypes.POINTER(ctypes.c_uint32), ctypes.POINTER(ctypes.c_uint32)]),
    "beagle_limits": (None, [ctypes.POINTER(_i32)] * 4),
    "beagle_status_string": (ctypes.c_char_p, [_i32]),
    "beagle_last_cuda_error": (_i32, []),
    "beagle_reserve": (_i32, [_i64, _i64]),
    "beagle_reserve_chunked": (_i32, [_i64]),
    "beagle_release": (None, []),
    "beagle_last_launch_count": (_i32, []),
    "beagle_set_chunk_target": (None, [_i64]),
    "beagle_chunk_buffers": (_i32, []),
    "beagle_set_profiling": (None, [_i32]),
    "beagle_profiled_eval_kernel_ms": (_f32, [ctypes.POINTER(_i32)]),
    "beagle_profiled_prepass_ms": (_f32, [ctypes.POINTER(_i32)]),
}
EXPORTS = tuple(_SIGNATURES)


def library_path() -> str:
    return _build.LIB


def lib():
    """Load (building first if the in-tree .so is missing or stale). Fails loudly."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if not os.path.exists(path) or os.environ.get("BEAGLE_REBUILD") == "1":
            path = _build.build()
        l = ctypes.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(l, name)       # AttributeError if a declared symbol is not exported
            fn.restype, fn.argtypes = res, args
        _lib = l
    return _lib


def _ptr(t):
    """torch tensor / numpy array / int / None -> address."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _check(status: int, where: str):
    if status != OK:
        raise BeagleError(status, where)


def beagle_eval(genomes, lengths, P, consts, n_consts, X, y, N, d, tax, fitness_out, stream=0):
    _check(lib().beagle_eval(_ptr(genomes), _ptr(lengths), int(P), _ptr(consts), int(n_consts),
                             _ptr(X), _ptr(y), int(N), int(d), float(tax), _ptr(fitness_out),
                             int(stream) or None), "beagle_eval")


FIT_MSE, FIT_CORRELATION, FIT_STD, FIT_STD_SQUARE, FIT_STD_CUBE, FIT_STD_HYPER = 0, 1, 2, 3, 4, 5


def beagle_eval_fit(genomes, lengths, P, consts, n_consts, X, y, N, d, fit, M, tax, fitness_out, stream=0):
    _check(lib().beagle_eval_fit(_ptr(genomes), _ptr(lengths), int(P), _ptr(consts), int(n_consts),
                                 _ptr(X), _ptr(y), int(N), int(d), int(fit), float(M), float(tax), _ptr(fitness_out),
                                 int(stream) or None), "beagle_eval_fit")


def beagle_eval_chunked(h_genomes, h_lengths, P, h_consts, n_consts, X, y, N, d, tax, fitness_out,
                        device_budget_bytes, stream=0):
    _check(lib().beagle_eval_chunked(_ptr(h_genomes), _ptr(h_lengths), int(P), _ptr(h_consts),
                                     int(n_consts), _ptr(X), _ptr(y), int(N), int(d), float(tax),
                                     _ptr(fitness_out), int(device_budget_bytes), int(stream) or None),
           "beagle_eval_chunked")


def beagle_eval_chunked_fit(h_genomes, h_lengths, P, h_consts, n_consts, X, y, N, d, fit, M, tax, fitness_out,
                            device_budget_bytes, stream=0):
    _check(lib().beagle_eval_chunked_fit(_ptr(h_genomes), _ptr(h_lengths), int(P), _ptr(h_consts), int(n_consts),
                                         _ptr(X), _ptr(y), int(N), int(d), int(fit), float(M), float(tax),
                                         _ptr(fitness_out), int(device_budget_bytes), int(stream) or None),
           "beagle_eval_chunked_fit")


TABLE2 = (0.01, 0.03, 0.06, 0.15, 0.25, 0.5, 1.0, 1.5, 2.5, 4.0)   # include/beagle.h BEAGLE_TABLE2 (Table 2)


def beagle_rank(fitness, P, sample_idx, n_sample, maximise, decile_out, hist_out=None, stream=0):
    _check(lib().beagle_rank(_ptr(fitness), int(P), _ptr(sample_idx), int(n_sample), int(bool(maximise)),
                             _ptr(decile_out), _ptr(hist_out), int(stream) or None), "beagle_rank")


def beagle_eval_blockwise(genomes, lengths, P, consts, n_consts, X, y, N, d, tax, fitness_out, stream=0):
    _check(lib().beagle_eval_blockwise(_ptr(genomes), _ptr(lengths), int(P), _ptr(consts),
                                       int(n_consts), _ptr(X), _ptr(y), int(N), int(d), float(tax),
                                       _ptr(fitness_out), int(stream) or None), "beagle_eval_blockwise")


def beagle_debug_outputs(genomes, lengths, P, consts, n_consts, X, N, d, out_PxN, stream=0):
    _check(lib().beagle_debug_outputs(_ptr(genomes), _ptr(lengths), int(P), _ptr(consts),
                                      int(n_consts), _ptr(X), int(N), int(d), _ptr(out_PxN),
                                      int(stream) or None), "beagle_debug_outputs")


def beagle_debug_schedule(P, off, depth, perm, stream=0):
    _check(lib().beagle_debug_schedule(int(P), _ptr(off), _ptr(depth), _ptr(perm), int(stream) or None),
           "beagle_debug_schedule")


def beagle_debug_counts(stream=0):
    v = [_i32() for _ in range(4)]
    _check(lib().beagle_debug_counts(*[ctypes.byref(x) for x in v], int(stream) or None), "beagle_debug_counts")
    return dict(n_sorted=v[0].value, n_general=v[1].value, n_slow=v[2].value, n_malformed=v[3].value)


def beagle_debug_compile(tokens, consts, d, tmem_slots, k_rcp, k_un, un_row_bytes, rcp_unsafe=0):
    """One program through the host build of the device's general compiler: (depth, slow, records uint32[n, 2]); numpy in, numpy out."""
    import numpy as np
    tokens = np.ascontiguousarray(tokens, np.int32)
    consts = np.ascontiguousarray(consts, np.float32)
    rec = np.zeros((len(tokens) + 1, 2), np.uint32)
    n, depth, slow = _i32(0), _i32(0), _i32(0)
    _check(lib().beagle_debug_compile(_ptr(tokens), len(tokens), _ptr(consts) if len(consts) else None, len(consts), int(d),
                                      int(tmem_slots), int(k_rcp), int(k_un), int(un_row_bytes), int(rcp_unsafe), _ptr(rec),
                                      ctypes.byref(n), ctypes.byref(depth), ctypes.byref(slow)), "beagle_debug_compile")
    return depth.value, bool(slow.value), rec[: n.value]


def beagle_debug_corr(f, y, length, M, tax, pre=False):
    """The correlation fitness of one individual from its per-case outputs, by the device's reduction on the host (emulated warp)."""
    import numpy as np
    f = np.ascontiguousarray(f, np.float32); y = np.ascontiguousarray(y, np.float32)
    out = _f32(0.0)
    _check(lib().beagle_debug_corr(_ptr(f), _ptr(y), len(f), int(length), float(M), float(tax), int(bool(pre)), ctypes.byref(out)),
           "beagle_debug_corr")
    return np.float32(out.value)


def beagle_debug_rank(fitness, sample_idx, maximise, grid=4):
    """k_rank on the host (SIMT emulator over the kernel's own source): (decile uint8[P], hist int64[10]); numpy in, numpy out."""
    import numpy as np
    fitness = np.ascontiguousarray(fitness, np.float32)
    sample_idx = np.ascontiguousarray(sample_idx, np.int64)
    dec = np.full(len(fitness), 255, np.uint8)
    hist = np.full(10, -1, np.int64)
    _check(lib().beagle_debug_rank(_ptr(fitness), len(fitness), _ptr(sample_idx), len(sample_idx), int(bool(maximise)), int(grid),
                                   _ptr(dec), _ptr(hist)), "beagle_debug_rank")
    return dec, hist


def beagle_debug_prepass(lengths, X, y, split=False):
    """The scheduling pre-pass on the host (SIMT emulator over the kernels' own source); numpy in, dict of numpy out."""
    import numpy as np
    lengths = np.ascontiguousarray(lengths, np.int32)
    X = np.ascontiguousarray(X, np.float32); y = np.ascontiguousarray(y, np.float32)
    P, (N, d) = len(lengths), X.shape
    npad = (N + 511) // 512 * 512
    out = dict(off=np.full(P, -1, np.int64), sched=np.full((P, 4), -1, np.int32), fitness=np.full(P, -12345.0, np.float32),
               depth=np.full(P, -7, np.int32), xt=np.full((d + 1, npad), -3.0, np.float32), hdr=np.zeros(6, np.int64),
               binstart=np.zeros(513, np.int32), binubase=np.zeros(513, np.int64))
    _check(lib().beagle_debug_prepass(_ptr(lengths), P, _ptr(X), _ptr(y), N, d, int(bool(split)), _ptr(out["off"]), _ptr(out["sched"]),
                                      _ptr(out["fitness"]), _ptr(out["depth"]), _ptr(out["xt"]), _ptr(out["hdr"]),
                                      _ptr(out["binstart"]), _ptr(out["binubase"])), "beagle_debug_prepass")
    return out


def beagle_debug_queue(meta4, max_len, ring_bytes, grid, threads, grouped, skip_seed=0, queue_start=0):
    """One warp of k_eval's scheduling loop on the host: (events int32[n, 4], (batch, stage_bytes, stages)); numpy in, numpy out."""
    import numpy as np
    meta4 = np.ascontiguousarray(meta4, np.int32).reshape(-1, 4)
    cap = 6 * len(meta4) + 64
    ev = np.zeros((cap, 4), np.int32)
    n = _i32(0)
    sizing = (_i32 * 3)()
    _check(lib().beagle_debug_queue(_ptr(meta4) if len(meta4) else None, len(meta4), int(max_len), int(ring_bytes), int(grid), int(threads),
                                    int(bool(grouped)), int(skip_seed), int(queue_start), _ptr(ev), cap, ctypes.byref(n), sizing),
           "beagle_debug_queue")
    assert n.value <= cap, "event buffer too small"
    return ev[: n.value], tuple(sizing)


def beagle_debug_walk(tokens, consts, d, tmem_slots, k_rcp, k_un, un_row_bytes, rcp_unsafe=0, f1=False):
    """One program through the host build of k_compile's walk: (taken, depth, used_f1, records uint32[n, 2]); numpy in, numpy out."""
    import numpy as np
    tokens = np.ascontiguousarray(tokens, np.int32)
    consts = np.ascontiguousarray(consts, np.float32)
    rec = np.zeros((len(tokens) + 8, 2), np.uint32)
    n, depth, taken, used = _i32(0), _i32(0), _i32(0), _i32(0)
    _check(lib().beagle_debug_walk(_ptr(tokens), len(tokens), _ptr(consts) if len(consts) else None, len(consts), int(d),
                                   int(tmem_slots), int(k_rcp), int(k_un), int(un_row_bytes), int(rcp_unsafe), int(f1), _ptr(rec),
                                   ctypes.byref(n), ctypes.byref(depth), ctypes.byref(taken), ctypes.byref(used)), "beagle_debug_walk")
    return bool(taken.value), depth.value, bool(used.value), rec[: n.value]


def beagle_debug_std_reward(f, y, fit, M):
    """Rewards of the pairs (f[i], y[i]) by the device's std_reward compiled for the host; numpy in, numpy out."""
    import numpy as np
    f = np.ascontiguousarray(f, np.float32); y = np.ascontiguousarray(y, np.float32)
    out = np.empty(len(f), np.float32)
    _check(lib().beagle_debug_std_reward(_ptr(f), _ptr(y), len(f), int(fit), float(M), _ptr(out)), "beagle_debug_std_reward")
    return out


def beagle_limits():
    v = [_i32() for _ in range(4)]
    lib().beagle_limits(*[ctypes.byref(x) for x in v])
    return dict(max_len=v[0].value, max_stack=v[1].value, max_n=v[2].value, max_d=v[3].value)


def beagle_status_string(status: int) -> str:
    return lib().beagle_status_string(int(status)).decode()


def beagle_last_cuda_error() -> int:
    return lib().beagle_last_cuda_error()


def beagle_reserve(P_max, T_max=0):
    _check(lib().beagle_reserve(int(P_max), int(T_max)), "beagle_reserve")


def beagle_reserve_chunked(device_budget_bytes):
    _check(lib().beagle_reserve_chunked(int(device_budget_bytes)), "beagle_reserve_chunked")


def beagle_release():
    lib().beagle_release()


def beagle_last_launch_count() -> int:
    return lib().beagle_last_launch_count()


def beagle_set_chunk_target(nbytes):
    lib().beagle_set_chunk_target(int(nbytes))


def beagle_chunk_buffers() -> int:
    return lib().beagle_chunk_buffers()


def beagle_set_profiling(on):
    """False / 0: off; True / 1: every call; n > 1: every n-th call."""
    lib().beagle_set_profiling(int(on))


def beagle_profiled_eval_kernel_ms():
    """(number of recorded calls, mean device ms of their evaluation kernels)."""
    n = _i32(0)
    ms = float(lib().beagle_profiled_eval_kernel_ms(ctypes.byref(n)))
    return n.value, ms


def beagle_profiled_prepass_ms():
    """(number of recorded calls, mean device ms of their pre-pass: scan, sort, compile)."""
    n = _i32(0)
    ms = float(lib().beagle_profiled_prepass_ms(ctypes.byref(n)))
    return n.value, ms


def raw_status(name: str, *args) -> int:
    """Call an entry point and return its status instead of raising (for the argument-error tests)."""
    return getattr(lib(), name)(*args)
