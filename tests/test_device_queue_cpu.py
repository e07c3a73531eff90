"""CPU-only: the scheduling loop of the interpreter kernel, run on the host (beagle_debug_queue = csrc/queue_body.inc, the source k_eval
itself is compiled from, with its device operations replaced by a recorder; the library's SASS is unchanged by the arrangement).

What one warp does with the work queue is replayed from the recorded events and held to what the design promises (DESIGN.md section 7,
"Fetch"): every entry the warp takes that has records is copied exactly once and handed to the interpreter exactly once, in order;
a group is a run of neighbours whose record blocks are contiguous, fits its stage and has at most 32 members; stages are used round
robin, never refilled before they were consumed, never more than NS in flight; the barrier phase the warp waits on is the one the
copy completes; entries without records (malformed, slow path) cost nothing. The mistake of round 1 (entries of different visits in
one 64-entry window taken for neighbours) showed only at full size on the GPU: here full-size conditions (32 entries per visit,
other warps' visits in between) are the default.
"""
import numpy as np
import pytest

from paper_2607_06731_b200 import api

STAGE_MAX = 4128            # bytes of the records of one 512-token program: (512 + 3 + 1) * 8


def stride(length):
    return (int(length) + 3 + 1) & ~1


def make_meta(rng, total, max_len, holes=0.0, shape="sorted"):
    """Queue entries as k_compile leaves them: evaluation order = length-sorted, longest first; record blocks laid out in the same
    order; a share `holes` of the entries has nothing to run (z = 0: malformed or handed to the blockwise kernel; their block is
    still reserved, as on the device)."""
    if shape == "sorted":
        lengths = np.sort(rng.integers(1, max_len + 1, total))[::-1]
    elif shape == "equal":
        lengths = np.full(total, max_len)
    else:                                           # heavy tail: a few long programs, many short ones
        lengths = np.sort(np.minimum(max_len, (max_len / rng.uniform(1, max_len, total)).astype(np.int64) + 1))[::-1]
    lengths[0] = max_len
    meta = np.zeros((total, 4), np.int32)
    y = 0
    for i, L in enumerate(lengths.tolist()):
        hole = rng.random() < holes
        meta[i] = (int(rng.integers(0, 1 << 30)), 0 if hole else y, 0 if hole else (stride(L) & ~1), L)
        y += stride(L) // 2                         # 16-byte units: 8 bytes per record
    return meta


def replay(meta, events, sizing, total, grouped, queue_start=0):
    """Checks every promise on the recorded events; returns the indices of the entries this warp took."""
    batch, stage_bytes, NS = sizing
    assert 1 <= batch <= 32 and 1 <= NS <= 8
    taken = []                                      # global indices, in the order the warp took them
    pending = []                                    # groups copied and not yet consumed: (stage, [indices])
    next_item = 0                                   # position in `taken` of the next entry not yet looked at for a copy
    n_copies = n_consumed = 0
    waiting = None                                  # the group a WAIT event announced
    one_by_one = []                                 # (non-grouped) members of the group being handed over
    expect_base = queue_start
    for kind, a, b, c in events.tolist():
        if kind == 0:                               # a visit to the queue
            assert b == batch
            assert a >= expect_base                 # the cursor only moves on (other warps may have moved it further)
            expect_base = a + batch
            taken += list(range(a, min(a + batch, total))) if a < total else []
        elif kind == 1:                             # a bulk copy of one group
            st, y16, nbytes = a, b, c
            assert st == n_copies % NS, "stages are used round robin"
            assert len(pending) < NS, "more copies in flight than stages"
            while next_item < len(taken) and meta[taken[next_item], 2] == 0:
                next_item += 1                      # entries with nothing to run are passed over
            assert next_item < len(taken), "a copy with no entry behind it"
            first = taken[next_item]
            assert meta[first, 1] == y16, "the copy starts at the first waiting entry's records"
            members, got, y = [], 0, y16
            while got < nbytes:
                assert next_item < len(taken), "a group runs past what the warp has taken"
                i = taken[next_item]
                assert meta[i, 2] != 0 and meta[i, 1] == y, "group members are neighbours with contiguous record blocks"
                if members:
                    assert i == members[-1] + 1, "neighbours in the sorted order"
                got += stride(meta[i, 3]) * 8
                y += stride(meta[i, 3]) // 2
                members.append(i)
                next_item += 1
            assert got == nbytes and nbytes <= stage_bytes and len(members) <= 32
            assert nbytes % 16 == 0                 # a bulk copy moves multiples of 16 bytes from a 16-byte aligned source
            if batch < 4:
                assert len(members) == 1            # a small colony keeps one individual per stage
            pending.append((st, members))
            n_copies += 1
        elif kind == 2:                             # the wait before a stage is consumed
            assert waiting is None and not one_by_one and pending, "a wait with nothing in flight"
            st, ph = a, b
            assert st == pending[0][0] == n_consumed % NS, "stages are consumed in the order they were filled"
            assert ph == (n_consumed // NS) % 2, "the phase of the barrier is the number of times the stage was used, mod 2"
            waiting = pending.pop(0)
            n_consumed += 1
        elif kind == 3:                             # grouped: the whole stage to the interpreter
            assert grouped and waiting is not None
            st, members = waiting
            assert a == st * stage_bytes and b == len(members)
            waiting = None
        elif kind == 4:                             # one program at a time
            assert not grouped
            if waiting is not None:
                st, members = waiting
                one_by_one = [(st * stage_bytes + off, i) for off, i in zip(np.cumsum([0] + [stride(meta[i, 3]) * 8 for i in members[:-1]]).tolist(), members)]
                waiting = None
            off, i = one_by_one.pop(0)
            assert a == off and b == meta[i, 0] and c == meta[i, 3]
        else:
            raise AssertionError(kind)
    assert waiting is None and not one_by_one and not pending, "something copied was never consumed"
    while next_item < len(taken) and meta[taken[next_item], 2] == 0:
        next_item += 1
    assert next_item == len(taken), "an entry the warp took was never copied"
    assert n_copies == n_consumed
    return taken


PLANS = [  # (entries, max_len, ring_bytes, grid, threads): rings and block sizes of the real launches (beagle_debug_plan), a grid of one
           # CTA so that a few thousand entries are "a large colony" for the warp (entries per visit = entries / (grid * warps * 8))
    (9000, 128, 5248, 1, 896),                      # config 3's launch: 32 entries per visit, two wide stages of 2560 bytes
    (6000, 128, 5248, 1, 896),                      # 26 entries per visit
    (8000, 512, 4480, 1, 896),                      # config 5's launch: ONE stage, of one maximum-length program
    (8000, 255, 4480, 1, 896),                      # config 4's launch: two stages of 2176 bytes
    (600, 64, 5376, 148, 1024),                     # a small colony (config 1's launch): one entry per visit, no groups, 8 stages
    (3000, 32, 5376, 1, 1024),                      # 11 entries per visit
    (4000, 16, 8 * STAGE_MAX, 1, 128),              # the largest ring a plan can give: stages capped at 2 wide ones
]


@pytest.mark.parametrize("grouped", [True, False])
@pytest.mark.parametrize("plan", PLANS)
def test_one_warp_takes_everything(plan, grouped):
    """With nobody else at the queue the warp's visits cover the whole colony, in order."""
    total, max_len, ring, grid, threads = plan
    rng = np.random.default_rng(total + max_len)
    for shape, holes in (("sorted", 0.0), ("sorted", 0.07), ("tail", 0.02), ("equal", 0.0)):
        meta = make_meta(rng, total, max_len, holes, shape)
        ev, sizing = api.beagle_debug_queue(meta, max_len, ring, grid, threads, grouped)
        # the sizing rules (eval_kernel.inc): entries per visit by the colony's size, wide stages only when there is something to group
        per_warp = len(meta) // (grid * (threads // 32) * 8)
        assert sizing[0] == min(32, max(1, per_warp))
        assert sizing[1] >= stride(max_len) * 8 and sizing[1] * sizing[2] <= ring and sizing[2] == min(8, ring // sizing[1])
        taken = replay(meta, ev, sizing, len(meta), grouped)
        assert taken == list(range(len(meta)))
        if sizing[0] >= 4 and shape != "equal" and max_len <= 128:
            copies = ev[ev[:, 0] == 1]
            runnable = int((meta[:, 2] != 0).sum())
            assert len(copies) < 0.5 * runnable     # grouping happens: far fewer copies than programs


@pytest.mark.parametrize("grouped", [True, False])
def test_with_other_warps_at_the_queue(grouped):
    """Other warps take batches between this warp's visits, so its window holds entries of several visits that are not neighbours:
    no group may span two visits, and what the others took is not touched."""
    rng = np.random.default_rng(99)
    for seed in range(1, 9):
        total, max_len, ring, grid, threads = PLANS[seed % 4]
        meta = make_meta(rng, total, max_len, 0.05 if seed % 2 else 0.0, "sorted" if seed % 3 else "tail")
        start = int(rng.integers(0, len(meta) // 2))
        ev, sizing = api.beagle_debug_queue(meta, max_len, ring, grid, threads, grouped, skip_seed=seed, queue_start=start)
        taken = replay(meta, ev, sizing, len(meta), grouped, queue_start=start)
        assert taken and taken[0] == start and len(set(taken)) == len(taken)
        visits = ev[ev[:, 0] == 0][:, 1]
        assert np.any(np.diff(visits) > sizing[0])  # the others really were there
        # equal lengths make record blocks of different visits look alike except for their address: the contiguity test is what separates them
    meta = make_meta(rng, 12_000, 64, 0.0, "equal")
    ev, sizing = api.beagle_debug_queue(meta, 64, 5248, 1, 896, grouped, skip_seed=5, queue_start=0)
    replay(meta, ev, sizing, len(meta), grouped)


def test_edges():
    rng = np.random.default_rng(3)
    # an empty colony: the kernel returns before the loop
    ev, sizing = api.beagle_debug_queue(np.zeros((0, 4), np.int32), 1, STAGE_MAX, 148, 1024, True)
    assert len(ev) == 0 and sizing == (0, 0, 0)
    # nothing to run at all: visits only
    meta = make_meta(rng, 3000, 40, 1.0)
    ev, sizing = api.beagle_debug_queue(meta, 40, 5248, 2, 64, True)
    assert set(ev[:, 0].tolist()) == {0}
    assert replay(meta, ev, sizing, len(meta), True) == list(range(len(meta)))
    # one program
    meta = make_meta(rng, 1, 512, 0.0)
    for grouped in (True, False):
        ev, sizing = api.beagle_debug_queue(meta, 512, STAGE_MAX, 148, 1024, grouped)
        replay(meta, ev, sizing, 1, grouped)
        assert (ev[:, 0] == 1).sum() == 1
    # the queue already past the end when the warp arrives
    meta = make_meta(rng, 100, 20, 0.0)
    ev, sizing = api.beagle_debug_queue(meta, 20, 5248, 148, 896, True, queue_start=500)
    assert len(ev) == 1 and ev[0, 0] == 0
    # argument errors
    l = api.lib()
    import ctypes
    n = ctypes.c_int32(); s3 = (ctypes.c_int32 * 3)()
    assert l.beagle_debug_queue(None, 5, 10, STAGE_MAX, 1, 32, 1, 0, 0, None, 0, ctypes.byref(n), s3) == api.ERR_INVALID_ARG
    assert l.beagle_debug_queue(None, 0, 10, STAGE_MAX - 8, 1, 32, 1, 0, 0, None, 0, ctypes.byref(n), s3) == api.ERR_INVALID_ARG
    assert l.beagle_debug_queue(None, 0, 10, STAGE_MAX, 1, 48, 1, 0, 0, None, 0, ctypes.byref(n), s3) == api.ERR_INVALID_ARG
    assert l.beagle_debug_queue(None, 0, 10, STAGE_MAX, 1, 32, 1, 0, 0, None, 0, ctypes.byref(n), s3) == api.OK
