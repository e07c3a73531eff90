"""Helpers of the -m gpu tests: move numpy inputs to the device and call the C-ABI through the binding."""
import numpy as np
import torch

from paper_2607_06731_b200 import api


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a if dtype is None else np.asarray(a, dtype)))
    return t.cuda()


def gpu_eval(genomes, lengths, consts, X, y, tax, fn="beagle_eval"):
    """Returns float32[P] computed by the CUDA path."""
    P = int(len(lengths))
    N, d = int(X.shape[0]), int(X.shape[1])
    g, l = dev(genomes, np.int32), dev(lengths, np.int32)
    c = dev(consts, np.float32) if len(consts) else None
    Xd, yd = dev(X, np.float32), dev(y, np.float32)
    out = torch.full((max(P, 1),), -12345.0, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    getattr(api, fn)(g, l, P, c, len(consts), Xd, yd, N, d, tax, out, st)
    torch.cuda.synchronize()
    return out[:P].cpu().numpy()


def gpu_eval_fit(genomes, lengths, consts, X, y, fit, M, tax):
    """float32[P] through beagle_eval_fit."""
    P = int(len(lengths))
    N, d = int(X.shape[0]), int(X.shape[1])
    g, l = dev(genomes, np.int32), dev(lengths, np.int32)
    c = dev(consts, np.float32) if len(consts) else None
    Xd, yd = dev(X, np.float32), dev(y, np.float32)
    out = torch.full((max(P, 1),), -12345.0, dtype=torch.float32, device="cuda")
    api.beagle_eval_fit(g, l, P, c, len(consts), Xd, yd, N, d, fit, M, tax, out, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out[:P].cpu().numpy()


def gpu_eval_chunked(genomes, lengths, consts, X, y, tax, budget, pinned=True):
    P = int(len(lengths))
    N, d = int(X.shape[0]), int(X.shape[1])
    hg = torch.from_numpy(np.ascontiguousarray(genomes, np.int32))
    hl = torch.from_numpy(np.ascontiguousarray(lengths, np.int32))
    hc = torch.from_numpy(np.ascontiguousarray(consts, np.float32))
    if pinned:
        hg, hl, hc = hg.pin_memory(), hl.pin_memory(), hc.pin_memory()
    Xd, yd = dev(X, np.float32), dev(y, np.float32)
    out = torch.full((max(P, 1),), -12345.0, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    api.beagle_eval_chunked(hg, hl, P, hc if len(consts) else None, len(consts), Xd, yd, N, d, tax,
                            out, budget, st)
    torch.cuda.synchronize()
    return out[:P].cpu().numpy()


def gpu_outputs(genomes, lengths, consts, X):
    """Per-case outputs float32[P, N] through beagle_debug_outputs."""
    P = int(len(lengths))
    N, d = int(X.shape[0]), int(X.shape[1])
    g, l = dev(genomes, np.int32), dev(lengths, np.int32)
    c = dev(consts, np.float32) if len(consts) else None
    Xd = dev(X, np.float32)
    out = torch.full((max(P, 1), N), -12345.0, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    api.beagle_debug_outputs(g, l, P, c, len(consts), Xd, N, d, out, st)
    torch.cuda.synchronize()
    return out[:P].cpu().numpy()
