"""dex_brick_slots_static: the brick occupancy + compaction step for callers that cannot allocate device memory.

Some users of the library run where cudaMalloc is off the table: inside a memory budget that was fixed and carved up at
start-up, inside a host application that owns the GPU's allocator, or in a loop that cannot afford to wait on the driver's
allocation lock.  For them the library has one entry that allocates nothing: outputs are the caller's buffers and the
per-brick flag scratch is a fixed 4 MiB array compiled into libdex.so (hence a limit of DEX_STATIC_MAX_BRICKS bricks).

The array is shared by every call on a GPU and keeps the previous call's contents, so the test makes TWO calls in a row
-- a larger, denser grid first, then a smaller, sparser one -- and checks each against the allocating path
(dex_build_sparse_grid) exactly: slots are integers, the bar is equality.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes alone in a fresh process (the first call does the one-time address look-up) and after
the other tests (the library's pool and torch's allocator already warm).
"""
import ctypes as C

import numpy as np
import pytest
import torch


def _mask(dims, brick, fill, seed):
    """Random brick-structured activity: a fraction `fill` of the bricks gets a few active voxels."""
    rng = np.random.default_rng(seed)
    ndim = len(dims)
    nb = [d // brick for d in dims]
    act = np.zeros(tuple(reversed(dims)), dtype=np.uint8)      # [z][y][x]
    on = rng.random(tuple(reversed(nb))) < fill
    for idx in np.argwhere(on):
        lo = [int(i) * brick for i in idx]
        for _ in range(int(rng.integers(1, 4))):                # 1-3 voxels anywhere in the brick, corners included
            off = rng.integers(0, brick, size=ndim)
            act[tuple(l + int(o) for l, o in zip(lo, off))] = 1
    return act.ravel()


def _existing_path(P, ndim, dims, brick, active_dev):
    g = P.dex_build_sparse_grid(ndim, dims, brick, 1.0, active_dev)
    slots = g.slots()
    _, n_active = g.info()
    g.destroy()
    return slots, n_active


def _static_path(P, ndim, dims, brick, active_dev):
    n_bricks = int(np.prod([d // brick for d in dims]))
    # the caller's buffers, poisoned so that an entry the call fails to write shows up
    slot = torch.full((n_bricks,), -7, dtype=torch.int32, device="cuda")
    bricks = torch.full((n_bricks,), -7, dtype=torch.int32, device="cuda")
    count = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    P.dex_brick_slots_static(ndim, dims, brick, 1.0, active_dev, slot, bricks, count)
    torch.cuda.synchronize()
    return slot.cpu().numpy(), bricks.cpu().numpy(), int(count.item())


def _compare(P, ndim, dims, brick, active):
    active_dev = None if active is None else torch.from_numpy(active).cuda()
    want_slots, want_n = _existing_path(P, ndim, dims, brick, active_dev)
    slot, bricks, n = _static_path(P, ndim, dims, brick, active_dev)
    assert n == want_n
    assert np.array_equal(slot, want_slots)
    # slot -> brick list: the allocating path keeps it inside the handle; it is the inverse of the slot table
    assert np.array_equal(bricks[:n], np.flatnonzero(want_slots >= 0).astype(np.int32))
    assert np.all(bricks[n:] == -7)          # documented: entries from A on are left alone
    return n


@pytest.mark.gpu
def test_static_scratch_entry_matches_allocating_path_twice_in_a_row():
    import paper_2511_08498_b200 as P
    # call 1: 3D, 64 x 40 x 24 bricks of 8 (61,440 bricks, ragged against the scan's 1024 chunks), mostly full
    n1 = _compare(P, 3, (512, 320, 192), 8, _mask((512, 320, 192), 8, 0.7, seed=11))
    # call 2 reuses the same static array, which still holds call 1's 61,440 flags: a smaller, much emptier 2D grid
    n2 = _compare(P, 2, (1104, 720), 16, _mask((1104, 720), 16, 0.15, seed=12))
    assert 0 < n2 < n1
    # and once more on the first shape with another mask: stale flags of call 2 must not leak either
    _compare(P, 3, (512, 320, 192), 8, _mask((512, 320, 192), 8, 0.3, seed=13))
    # NULL activity map = every brick populated; 1024 x 1024 bricks is exactly the size of the static array
    from paper_2511_08498_b200.binding import DEX_STATIC_MAX_BRICKS
    assert _compare(P, 2, (16 * 1024, 16 * 1024), 16, None) == DEX_STATIC_MAX_BRICKS


@pytest.mark.gpu
def test_static_scratch_entry_second_call_holds_device_memory_steady():
    """Two identical calls back to back with the caller's buffers made beforehand: free device memory does not move."""
    import paper_2511_08498_b200 as P
    dims, brick = (2048, 2048), 16
    active = torch.from_numpy(_mask(dims, brick, 0.5, seed=21)).cuda()
    nb = (dims[0] // brick) * (dims[1] // brick)
    slot = torch.empty(nb, dtype=torch.int32, device="cuda")
    bricks = torch.empty(nb, dtype=torch.int32, device="cuda")
    count = torch.empty(1, dtype=torch.int32, device="cuda")
    P.dex_brick_slots_static(2, dims, brick, 1.0, active, slot, bricks, count)      # first call: one-time set-up
    torch.cuda.synchronize()
    first = slot.clone()
    free0, _ = torch.cuda.mem_get_info()
    P.dex_brick_slots_static(2, dims, brick, 1.0, active, slot, bricks, count)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    assert torch.equal(slot, first)


def test_static_scratch_entry_rejects_grids_beyond_its_array():
    """More bricks than the compiled-in array holds: a clear DEX_ERR_SHAPE before anything touches the GPU (runs anywhere)."""
    from paper_2511_08498_b200 import binding as B
    d = B._GridDesc()
    d.ndim, d.brick, d.voxel_size = 2, 16, 1.0
    d.dims[0], d.dims[1], d.dims[2] = 16 * 2048, 16 * 1024, 1        # 2,097,152 bricks > 1,048,576
    dummy = C.c_void_p(256)                                          # never dereferenced: the size check comes first
    st = B._L.dex_brick_slots_static(C.byref(d), None, dummy, dummy, dummy, None)
    assert st == B.DEX_ERR_SHAPE
    msg = B._L.dex_last_error().decode()
    assert "DEX_STATIC_MAX_BRICKS" in msg and str(B.DEX_STATIC_MAX_BRICKS) in msg
    st = B._L.dex_brick_slots_static(C.byref(d), None, None, dummy, dummy, None)
    assert st == B.DEX_ERR_INVALID_ARG                               # a NULL output is refused as well
