"""-m gpu: the parts of the path that are integer work or plumbing, checked bit for bit.

- the pre-pass's outputs (offsets, per-program scan, length-sorted schedule) through
  beagle_debug_schedule / beagle_debug_counts, against numpy and the oracle's depth;
- the chunk loop (a8) with K = 2, 3, 5 and 8 staging buffers, and config 5 as BASELINE.json configures it
  (P = 4,194,304, a 1 GiB device budget) against the resident call and a stratified sample of the oracle;
- the boundary's promises about blocking: a released workspace comes back, an un-reserved call inside a stream
  capture is refused with a status code instead of a hidden synchronisation.
"""
import numpy as np
import pytest

from paper_2607_06731_b200 import colonies
from tests import parity
from tests.util import asm, pack

pytestmark = pytest.mark.gpu

QNAN = np.uint32(0x7FC00000)


def _bits(a):
    return np.asarray(a, np.float32).view(np.uint32)


def _splice(col, extra_progs, extra_lengths_only, seed):
    """Insert hand-made programs (token arrays) and individuals that are a length only (out of range: 0 words) at seeded
    places of a colony. Returns genomes, lengths."""
    rng = np.random.default_rng(seed)
    off = np.concatenate([[0], np.cumsum(col.lengths, dtype=np.int64)])
    progs = [col.genomes[off[p]:off[p + 1]] for p in range(col.P)]
    lens = [int(l) for l in col.lengths]
    for e in extra_progs:
        k = int(rng.integers(0, len(progs) + 1))
        progs.insert(k, np.asarray(e, np.int32)); lens.insert(k, len(e))
    for l in extra_lengths_only:
        k = int(rng.integers(0, len(progs) + 1))
        progs.insert(k, np.zeros(0, np.int32)); lens.insert(k, int(l))
    return np.concatenate(progs).astype(np.int32), np.array(lens, np.int32)


def test_prepass_integer_outputs_bit_exact(oracle):
    """off[] = exclusive prefix sum of the clamped lengths, depth[] = the oracle's maximum stack depth (0 for malformed),
    perm[] = the in-range individuals, each once, by non-increasing length, then -1 (integer work is exact)."""
    import torch
    from paper_2607_06731_b200 import api
    from tests.gpu_util import dev
    col = colonies.make_colony(5, 50000)
    T = colonies.token
    OP = colonies.OP
    bad = [[T(OP["ADD"])], [T(OP["LOAD"], 0), T(OP["LOAD"], 1), T(0x3F)], [T(OP["LOAD"], 99)], [T(OP["CONST"], 1 << 23)],
           [T(OP["LOAD"], 0), T(OP["SIN"], 5)], [T(OP["LOAD"], 0)] * 33 + [T(OP["ADD"])] * 32, [T(OP["LOAD"], 0), T(OP["DEL"])]]
    f1 = [asm(t, [])[0] for t in ("x0 DUP MUL", "x0 x1 SWAP SUB", "x0 x1 ADD DUP DUP MUL MUL", "x0 x1 DEL SQUARE", "x0 SIN x1 COS SWAP DIV",
                                 "x0 x1 POW", "x0 COPY@3 DEL PASTE@3", "x0 TANH CUBE SIGN")]
    g, l = _splice(col, bad * 40 + f1 * 40, [0, -7, 513, 100000, -2147483648] * 30, seed=5)
    P = len(l)
    N, d = col.X.shape
    out = torch.empty(P, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    gd, ld, cd, Xd, yd = dev(g), dev(l), dev(col.consts), dev(col.X), dev(col.y)
    for _ in range(2):      # twice: the second call knows that the colony has stack commands and compiles them in k_compile's own walk
        api.beagle_eval(gd, ld, P, cd, len(col.consts), Xd, yd, N, d, col.tax, out, st)
        torch.cuda.synchronize()
    off = torch.empty(P, dtype=torch.int64, device="cuda"); depth = torch.empty(P, dtype=torch.int32, device="cuda")
    perm = torch.empty(P, dtype=torch.int32, device="cuda")
    api.beagle_debug_schedule(P, off, depth, perm, st)
    cnt = api.beagle_debug_counts(st)
    torch.cuda.synchronize()
    off, depth, perm = off.cpu().numpy(), depth.cpu().numpy(), perm.cpu().numpy()
    inr = (l >= 1) & (l <= 512)
    want_off = np.concatenate([[0], np.cumsum(np.where(inr, l, 0), dtype=np.int64)])[:-1]
    assert np.array_equal(off, want_off)
    orc = oracle.evaluate_parallel(g, l, col.consts, col.X[:2], col.y[:2], col.tax)     # two cases: only the static scan matters
    assert np.array_equal(depth, orc["depth"])
    n_sorted = int(inr.sum())
    assert cnt["n_sorted"] == n_sorted
    assert np.all(perm[n_sorted:] == -1)
    head = perm[:n_sorted]
    assert np.array_equal(np.sort(head), np.nonzero(inr)[0])                     # each in-range individual exactly once
    assert np.all(np.diff(l[head]) <= 0)                                         # longest first
    malformed = (orc["flags"] & 1) != 0
    assert cnt["n_malformed"] == int((malformed & inr).sum())
    assert np.all(_bits(out.cpu().numpy())[malformed] == QNAN)
    assert cnt["n_slow"] == 3 * 40                                               # POW, COPY / PASTE, TANH: the blockwise kernel
    # what k_compile's walk turns down: the malformed ones and the three programs with POW, a variable, a library function
    # (DUP SWAP DEL SIGN SQUARE CUBE are compiled by the walk itself)
    assert cnt["n_general"] == len(bad) * 40 + 3 * 40


@pytest.mark.parametrize("K", [2, 3, 5, 8])
def test_chunked_with_K_staging_buffers(K):
    """The chunk loop with K staging buffers (buffer c mod K, more chunks than buffers): bit-identical to the resident call."""
    import torch
    from paper_2607_06731_b200 import api
    from tests.gpu_util import gpu_eval, gpu_eval_chunked
    col = colonies.make_colony(5, 90000)
    ref = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    target = 1 << 20                                                             # 1 MiB buffers: the colony is about 27 MB
    api.beagle_set_chunk_target(target)
    try:
        out = gpu_eval_chunked(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, K * target + 4096)
        assert api.beagle_chunk_buffers() == K
        words = int(col.T) + col.P
        assert words * 4 > 2 * K * target                                        # more than 2 K chunks: every buffer is reused
        assert np.array_equal(_bits(out), _bits(ref))
        out2 = gpu_eval_chunked(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, K * target + 4096, pinned=False)
        assert np.array_equal(_bits(out2), _bits(ref))
    finally:
        api.beagle_set_chunk_target(0)
        torch.cuda.synchronize()


def test_config5_as_configured(oracle):
    """BASELINE.json configs[4] at its own size and in its own regime: P = 4,194,304 from pinned host memory through
    beagle_eval_chunked with a 1 GiB device budget (8 staging buffers, more chunks than buffers), bit-identical to
    beagle_eval on the resident colony; the oracle on a stratified sample: every designed-invalid
    individual of a stride, the 4096 longest, the 4096 deepest, a seeded 1/256 of the rest."""
    import torch
    from paper_2607_06731_b200 import api
    from tests.gpu_util import dev
    cfg = colonies.CONFIGS[5]
    col = colonies.make_colony(5)
    P = col.P
    assert P == 4194304 and cfg.budget_bytes == 1 << 30
    N, d = col.X.shape
    st = torch.cuda.current_stream().cuda_stream
    Xd, yd = dev(col.X), dev(col.y)
    hg = torch.from_numpy(col.genomes).pin_memory(); hl = torch.from_numpy(col.lengths).pin_memory()
    hc = torch.from_numpy(col.consts).pin_memory()
    out = torch.full((P,), -12345.0, dtype=torch.float32, device="cuda")
    api.beagle_eval_chunked(hg, hl, P, hc, len(col.consts), Xd, yd, N, d, col.tax, out, cfg.budget_bytes, st)
    torch.cuda.synchronize()
    K = api.beagle_chunk_buffers()
    n_chunks = -(-(int(col.T) + P) * 4 // ((cfg.budget_bytes // K) & ~255))
    print(f"config 5: T = {col.T}, {K} staging buffers, about {n_chunks} chunks")
    assert K == 8 and n_chunks > K
    fit = out.cpu().numpy()
    ref = torch.full((P,), -1.0, dtype=torch.float32, device="cuda")
    api.beagle_eval(dev(col.genomes), dev(col.lengths), P, dev(col.consts), len(col.consts), Xd, yd, N, d, col.tax, ref, st)
    torch.cuda.synchronize()
    assert np.array_equal(_bits(fit), _bits(ref.cpu().numpy()))                  # DESIGN.md R19
    api.beagle_release()                                                         # several GB of micro-ops: give them back
    rng = np.random.default_rng(55)
    depth = oracle.evaluate_parallel(col.genomes, col.lengths, col.consts, col.X[:1], col.y[:1], col.tax)["depth"]
    designed = np.arange(0, P, 20)[::16]                                         # p mod 20 == 0: the designed-invalid ones (L >= 16)
    longest = np.argsort(-col.lengths, kind="stable")[:4096]
    deepest = np.argsort(-depth, kind="stable")[:4096]
    rest = np.nonzero(rng.random(P) < 1.0 / 256)[0]
    sel = np.unique(np.concatenate([designed, longest, deepest, rest]))
    off = np.concatenate([[0], np.cumsum(col.lengths, dtype=np.int64)])
    g = np.concatenate([col.genomes[off[p]:off[p + 1]] for p in sel])
    orc = oracle.evaluate_parallel(g, col.lengths[sel], col.consts, col.X, col.y, col.tax)
    rep = parity.compare(fit[sel], orc)
    msg = parity.describe(rep, fit[sel], orc)
    print(f"config 5 as configured, {len(sel)} sampled: {msg}")
    assert len(rep["bad"]) == 0, msg
    assert rep["invalid"] > 1000                                                 # the designed-invalid programs are there
    assert rep["strict"] >= 0.60 * (rep["strict"] + rep["conditioned"]), msg
    assert not np.any(fit == np.float32(-12345.0))


def test_release_then_eval_round_trip():
    """beagle_release frees the workspace and the staging buffers; the next calls allocate again and give the same bits."""
    import torch
    from paper_2607_06731_b200 import api
    from tests.gpu_util import gpu_eval, gpu_eval_chunked
    col = colonies.make_colony(2, 20000)
    a = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    api.beagle_release()
    junk = [torch.empty(1 << 20, device="cuda") for _ in range(8)]                # other users of the allocator in between
    b = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    api.beagle_release(); api.beagle_release()                                   # twice in a row is harmless
    c = gpu_eval_chunked(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax, 1 << 20)
    d = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    for x in (b, c, d):
        assert np.array_equal(_bits(a), _bits(x))
    del junk


def test_unreserved_call_inside_capture_is_refused():
    """include/beagle.h "Blocking": a call that would have to grow its workspace inside a stream capture returns
    BEAGLE_ERR_NOT_RESERVED and enqueues nothing; after beagle_reserve the same call is captured and replays."""
    import torch
    from paper_2607_06731_b200 import api
    from tests.gpu_util import dev, gpu_eval
    col = colonies.make_colony(2, 30000)
    ref = gpu_eval(col.genomes, col.lengths, col.consts, col.X, col.y, col.tax)
    api.beagle_release()
    N, d = col.X.shape
    g, l, c, X, y = dev(col.genomes), dev(col.lengths), dev(col.consts), dev(col.X), dev(col.y)
    out = torch.zeros(col.P, dtype=torch.float32, device="cuda")
    s = torch.cuda.Stream()
    args = (g.data_ptr(), l.data_ptr(), col.P, c.data_ptr(), len(col.consts), X.data_ptr(), y.data_ptr(), N, d, col.tax, out.data_ptr())
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        out.zero_()                                                              # (something to capture: the refused call enqueues nothing)
        status = api.raw_status("beagle_eval", *args, s.cuda_stream)
    assert status == api.ERR_NOT_RESERVED
    assert "beagle_reserve" in api.beagle_status_string(status)
    # reserved for P but with no token bound: still not capturable (the token total would have to be read back)
    api.beagle_reserve(col.P, 0)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        out.zero_()
        status = api.raw_status("beagle_eval", *args, s.cuda_stream)
    assert status == api.ERR_NOT_RESERVED
    api.beagle_reserve(col.P, int(col.T))
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        status = api.raw_status("beagle_eval", *args, s.cuda_stream)
    assert status == api.OK
    graph.replay(); torch.cuda.synchronize()
    assert np.array_equal(_bits(out.cpu().numpy()), _bits(ref))


@pytest.mark.parametrize("N,d", [(512, 5), (1024, 9)])
def test_stack_commands_run_on_the_interpreter(oracle, N, d):
    """programs of the eleven commands plus DUP SWAP DEL SIGN SQUARE CUBE, the paper's printed genomes among
    them, are compiled to micro-ops (none goes to the blockwise kernel) and are bit-identical to the blockwise kernel."""
    import torch
    from paper_2607_06731_b200 import api
    from tests.gpu_util import gpu_eval
    from tests.util import random_gcl_programs
    rng = np.random.default_rng(77)
    X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
    y = (X[:, 0] * X[:, 1] - X[:, 2]).astype(np.float32)
    names = ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP", "SIGN", "SQUARE", "CUBE", "DUP", "SWAP", "DEL"]
    texts = random_gcl_programs(rng, 3000, d, names)
    consts = []
    progs = [asm(t, consts)[0] for t in texts]
    g, l, c = pack(progs, consts)
    a0 = gpu_eval(g, l, c, X, y, 0.001)
    cnt0 = api.beagle_debug_counts(torch.cuda.current_stream().cuda_stream)
    a = gpu_eval(g, l, c, X, y, 0.001)             # the second call compiles them in k_compile's own walk (k_compile<F1>)
    cnt = api.beagle_debug_counts(torch.cuda.current_stream().cuda_stream)
    assert np.array_equal(_bits(a0), _bits(a))
    assert cnt0["n_slow"] == 0 and cnt0["n_malformed"] == 0, cnt0
    assert cnt["n_slow"] == 0 and cnt["n_malformed"] == 0 and cnt["n_general"] == 0, cnt
    b = gpu_eval(g, l, c, X, y, 0.001, fn="beagle_eval_blockwise")
    assert np.array_equal(_bits(a), _bits(b))
    orc = oracle.evaluate_parallel(g, l, c, X, y, 0.001)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)


@pytest.mark.parametrize("N,d", [(513, 9), (700, 12), (1000, 20), (1023, 32), (1024, 17)])
def test_split_passes_ragged_and_wide(oracle, N, d):
    """Calls with more than 512 cases whose variable rows crowd the slot rows are split into one interpreter launch per pass
    (DESIGN.md §7): ragged second passes, variable counts that fit tensor memory only when split (d > 16), deep stacks;
    bit-identical to the blockwise kernel, parity with the oracle, and bitwise equal to the per-case outputs' own sum order
    (the chunked call, which cuts the colony differently, gives the same bits)."""
    from tests.gpu_util import gpu_eval, gpu_eval_chunked
    from tests.util import random_gcl_programs
    rng = np.random.default_rng(1000 + N + d)
    X = rng.uniform(-3, 3, (N, d)).astype(np.float32)
    y = (X[:, 0] * X[:, d - 1] - np.cos(X[:, d // 2])).astype(np.float32)
    names = ["ADD", "SUB", "MUL", "DIV", "SIN", "COS", "LOG", "SQRT", "EXP", "SQUARE", "DUP", "SWAP"]
    texts = random_gcl_programs(rng, 1500, d, names)
    deep = " ".join(f"x{j % d} SIN" for j in range(20)) + " ADD" * 19          # 20 computed values waiting: slots in local memory
    consts = []
    progs = [asm(t, consts)[0] for t in texts + [deep] * 8]
    g, l, c = pack(progs, consts)
    a = gpu_eval(g, l, c, X, y, 0.001)
    b = gpu_eval(g, l, c, X, y, 0.001, fn="beagle_eval_blockwise")
    assert np.array_equal(_bits(a), _bits(b))
    ch = gpu_eval_chunked(g, l, c, X, y, 0.001, 64 << 10)
    assert np.array_equal(_bits(a), _bits(ch))
    orc = oracle.evaluate_parallel(g, l, c, X, y, 0.001)
    rep = parity.compare(a, orc)
    assert len(rep["bad"]) == 0, parity.describe(rep, a, orc)
