"""CPU-only: the scheduling pre-pass (a2-a3: offsets, length histogram and its scans, counting sort by length, start records; a4's
transpose) run on the host by a small SIMT emulator from the source the three kernels are compiled from (beagle_debug_prepass =
csrc/prepass_body.inc under csrc/simt_host.inc: one OS thread per CUDA thread, barriers for __syncthreads and the warp shuffles; the
library's SASS is unchanged by the arrangement). Checked against plain numpy: "integer work is bit-exact"."""
import numpy as np
import pytest

from paper_2607_06731_b200 import api


def stride(L):
    return (L + 3 + 1) & ~1


def check(lengths, X, y, split=False):
    lengths = np.asarray(lengths, np.int32)
    P = len(lengths)
    N, d = X.shape
    o = api.beagle_debug_prepass(lengths, X, y, split)
    inr = (lengths >= 1) & (lengths <= 512)
    cl = np.where(inr, lengths, 0).astype(np.int64)
    off = np.concatenate([[0], np.cumsum(cl)[:-1]])
    assert np.array_equal(o["off"], off)                                          # a2: exclusive prefix sum, out-of-range lengths count 0
    T, uent, n_sorted, max_len, unsafe, zeroed = o["hdr"].tolist()
    assert T == cl.sum() and n_sorted == inr.sum() and zeroed == 0
    assert max_len == (cl.max() if inr.any() else 0)
    assert uent == sum(stride(int(L)) for L in cl[inr])
    # out-of-range lengths: the canonical NaN and depth 0, in band; nothing else is touched here
    assert np.all(o["fitness"][~inr].view(np.uint32) == 0x7FC00000) and np.all(o["depth"][~inr] == 0)
    assert np.all(o["fitness"][inr] == np.float32(-12345.0)) and np.all(o["depth"][inr] == -7)
    # a3: the sorted order: a permutation of the in-range individuals, longest first; every start record says where its tokens and
    # its records are; record blocks follow one another in the sorted order
    s = o["sched"]
    assert np.all(s[n_sorted:] == -1)
    p = s[:n_sorted, 0]
    assert np.array_equal(np.sort(p), np.nonzero(inr)[0])
    w = s[:n_sorted, 3].astype(np.int64)
    L = w & 0x3FF
    assert np.array_equal(L, lengths[p]) and np.all(np.diff(L) <= 0)
    tok = ((w >> 10) & 0xFF) << 32 | (s[:n_sorted, 1].astype(np.int64) & 0xFFFFFFFF)
    assert np.array_equal(tok, off[p])
    ub = ((w >> 18) & 0xFF) << 32 | (s[:n_sorted, 2].astype(np.int64) & 0xFFFFFFFF)
    strides = (L + 4) & ~1
    assert np.array_equal(ub, np.concatenate([[0], np.cumsum(strides)[:-1]])[:n_sorted])
    # the bins: bin k holds length 512 - k; their exclusive scans
    cnt = np.bincount(512 - lengths[inr], minlength=513)[:513].astype(np.int64)
    assert np.array_equal(o["binstart"], np.concatenate([[0], np.cumsum(cnt)[:-1]]))
    bs = np.array([stride(512 - k) for k in range(513)], np.int64)
    assert np.array_equal(o["binubase"], np.concatenate([[0], np.cumsum(cnt * bs)[:-1]]))
    # a4: the cases variable-major, zero-padded, y as the last row; which variables have a protected case
    npad = (N + 511) // 512 * 512
    xt = np.zeros((d + 1, npad), np.float32)
    xt[:d, :N] = X.T
    xt[d, :N] = y
    assert np.array_equal(o["xt"].view(np.uint32), xt.view(np.uint32))
    assert unsafe == sum(1 << j for j in range(d) if np.any(np.abs(X[:, j]) < np.float32(1e-6)))
    return o


@pytest.mark.parametrize("P", [1, 31, 256, 2047, 2048, 2049, 5000, 20000])
def test_prepass_on_random_colonies(P):
    rng = np.random.default_rng(P)
    lengths = rng.integers(1, 513, P).astype(np.int32)
    bad = rng.random(P) < 0.03                       # out-of-range lengths sprinkled in: 0, negative, too long
    lengths[bad] = rng.choice([0, -5, 513, 100000, -2**31], int(bad.sum()))
    N, d = int(rng.integers(1, 1025)), int(rng.integers(1, 33))
    X = rng.uniform(-2, 2, (N, d)).astype(np.float32)
    X[rng.integers(N), rng.integers(d)] = 0.0       # a protected case in one variable
    y = rng.normal(size=N).astype(np.float32)
    check(lengths, X, y, split=bool(P % 2))


def test_prepass_shapes_of_the_configs():
    rng = np.random.default_rng(1)
    X = rng.uniform(1, 5, (512, 5)).astype(np.float32)
    y = X[:, 4].copy()
    # Zipf-like lengths (config 5), many equal lengths (one crowded bin), all of one length, nothing in range
    H = 1.0 / np.arange(1, 513)
    zipf = rng.choice(np.arange(1, 513), 30000, p=H / H.sum()).astype(np.int32)
    check(zipf, X, y)
    check(np.full(9000, 37, np.int32), X, y)
    check(rng.choice([1, 2, 512], 7000).astype(np.int32), X, y)
    o = check(np.array([0, 0, 700, -1], np.int32), X, y)
    assert o["hdr"][2] == 0 and o["hdr"][3] == 0
    # more than 32 blocks of 2048 programs: the scan of the block sums goes across warps of the one-block kernel
    big = rng.integers(1, 40, 150_000).astype(np.int32)
    big[::1000] = 0
    check(big, X, y)


def test_prepass_argument_errors():
    l = api.lib()
    one = np.zeros(1, np.int32)
    assert l.beagle_debug_prepass(one.ctypes.data, 0, one.ctypes.data, one.ctypes.data, 1, 1, 0, *([one.ctypes.data] * 8)) == api.ERR_INVALID_ARG
    assert l.beagle_debug_prepass(None, 1, one.ctypes.data, one.ctypes.data, 1, 1, 0, *([one.ctypes.data] * 8)) == api.ERR_INVALID_ARG
    assert l.beagle_debug_prepass(one.ctypes.data, (1 << 24) + 1, one.ctypes.data, one.ctypes.data, 1, 1, 0, *([one.ctypes.data] * 8)) == api.ERR_INVALID_ARG
    assert l.beagle_debug_prepass(one.ctypes.data, 1, one.ctypes.data, one.ctypes.data, 1025, 1, 0, *([one.ctypes.data] * 8)) == api.ERR_INVALID_ARG


# ---- k_rank the same way: the kernel's own source under the emulator, against oracle/ranking.py ------------------------
@pytest.mark.parametrize("P,n_sample,grid,seed", [(1000, 100, 1, 1), (5000, 100, 3, 2), (37, 100, 2, 3), (5000, 7, 4, 4), (3000, 1024, 2, 5), (1, 1, 1, 6)])
def test_rank_kernel_on_the_host_matches_the_ranking_oracle(P, n_sample, grid, seed):
    from oracle import ranking as R
    rng = np.random.default_rng(seed)
    f = (rng.standard_normal(P) * 100).astype(np.float32)
    f[rng.random(P) < 0.03] = np.nan                 # NaN is worse than every number (R24)
    f[rng.random(P) < 0.03] = np.inf
    if seed % 2:
        f = np.round(f, 0)                           # many ties: equal fitnesses are not strictly worse
    sample = rng.integers(0, P, n_sample)
    for maximise in (False, True):
        dec, hist = api.beagle_debug_rank(f, sample, maximise, grid)
        want, whist, _ = R.rank_deciles(f, sample, maximise)
        assert np.array_equal(dec, want) and np.array_equal(hist, whist)
        assert hist.sum() == P
