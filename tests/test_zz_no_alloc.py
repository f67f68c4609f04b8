"""sph_comm_hash_noalloc -- the communication hash for callers that cannot allocate device memory.

Some users of this library cannot call cudaMalloc: a solver whose own pool took the whole GPU at
start-up, a plug-in whose host forbids allocations (and the device-wide stall of cudaFree) inside
the time loop.  Every other entry point needs an sph_ctx, whose scratch sph_create allocates; this
one works out of a 16 MiB array built into the library.  The tests below check what such a user
relies on:
  * the result is bit for bit the comm_hash / boundary_count of the ordinary sph_comm_hash
    (integer work: the tolerance of every other comm-hash test here is exact equality);
  * a second call right after the first is still right although both share the built-in array and
    the first one left its owner masks in it (the second input has FEWER flagged buckets, so stale
    masks would show up as extra boundary particles);
  * a grid the array cannot hold is refused with a clear error instead of being clipped.
This file sorts last on purpose (pytest -x stops at the first failure; a problem here must not
hide the parity tests), and it passes alone in a fresh process as well as after all other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2310_03596_b200 import workloads as wl


def _sorted_inputs(sph, w):
    """Stages 1-3 of the ordinary path: sorted hashes / owners and the reference comm hash."""
    import torch
    ctx = sph.Context.for_workload(w)
    posm = torch.from_numpy(w.posm).cuda()
    owner = torch.from_numpy(w.owner).cuda()
    h = ctx.sph_hash(posm)
    sh, perm = ctx.sph_sort(h)
    so = owner[perm.long()].contiguous()
    cs, ce = ctx.sph_cell_ranges(sh)
    ch, _, cnt, _ = ctx.sph_comm_hash(sh, so, perm, cs, ce)
    torch.cuda.synchronize()
    want = (sph.as_u32(ch).copy(), int(sph.as_u32(cnt)[0]))
    ctx.close()
    return sh, so, want


@pytest.mark.gpu
def test_noalloc_matches_comm_hash_on_two_calls_in_a_row():
    import torch
    from paper_2310_03596_b200 import sph

    # same 33^3 lattice and grid twice: 16 interleaved owners (every bucket flagged), then four
    # slabs (only the buckets at the three interfaces) -- stale masks from call 1 would over-flag call 2
    w1 = wl.lattice_block(33, 33, 33, 0.1, 7, owners=("random", 16))
    w2 = wl.config(1, side=33)
    assert tuple(w1.dims) == tuple(w2.dims)
    cases = [(w, *_sorted_inputs(sph, w)) for w in (w1, w2)]
    assert cases[0][3][1] > cases[1][3][1] > 0          # call 2 really has fewer boundary particles

    # the caller owns inputs AND outputs: allocate them up front, then make the two calls back to back
    outs = [(torch.full((w.n,), 0x55555555, dtype=torch.int32, device="cuda"),
             torch.full((1,), -7, dtype=torch.int32, device="cuda")) for w, *_ in cases]
    for (w, sh, so, _), (ch, cnt) in zip(cases, outs):
        sph.sph_comm_hash_noalloc(w.dims, w.n_owners, sh, so, comm_hash=ch, boundary_count=cnt)
    torch.cuda.synchronize()
    for (w, _, _, (want_ch, want_cnt)), (ch, cnt) in zip(cases, outs):
        got = sph.as_u32(ch)
        assert int(sph.as_u32(cnt)[0]) == want_cnt, w.name
        assert np.array_equal(got, want_ch), (w.name, int((got != want_ch).sum()))
        assert int((got != sph.GARBAGE_HASH).sum()) == want_cnt

    # y / z reach of the stencil and a ragged tail: clipped geometry with RCB labels, n % 256 != 0
    w3 = wl.config(3, scale=0.12)
    sh, so, (want_ch, want_cnt) = _sorted_inputs(sph, w3)
    ch, cnt = sph.sph_comm_hash_noalloc(w3.dims, w3.n_owners, sh, so)
    torch.cuda.synchronize()
    assert int(sph.as_u32(cnt)[0]) == want_cnt and np.array_equal(sph.as_u32(ch), want_ch)

    # empty input: count 0, nothing else touched
    e = torch.empty(0, dtype=torch.int32, device="cuda")
    _, cnt = sph.sph_comm_hash_noalloc(w3.dims, w3.n_owners, e, e)
    torch.cuda.synchronize()
    assert int(cnt.item()) == 0


def _params(dims, n_owners=2):
    from paper_2310_03596_b200 import sph
    p = sph._Params()
    for a in range(3):
        p.dims[a] = dims[a]
    p.n_owners = n_owners
    return p


def test_noalloc_refuses_grids_beyond_its_built_in_scratch():
    """The size check comes before any CUDA call, so it is testable (and tested) without a GPU."""
    from paper_2310_03596_b200 import build, sph

    build.build()
    lib = sph.load_library()
    assert sph.NOALLOC_MAX_CELLS == 1 << 22
    too_big = _params((2048, 2048, 2))                      # 2^23 buckets
    assert lib.sph_comm_hash_noalloc(C.byref(too_big), 0, None, None, None, C.c_void_p(8), None) == sph.SPH_ELIMIT
    huge = _params((2 ** 31 - 1, 2 ** 31 - 1, 2 ** 31 - 1))  # the product would wrap 64 bits
    assert lib.sph_comm_hash_noalloc(C.byref(huge), 0, None, None, None, C.c_void_p(8), None) == sph.SPH_ELIMIT
    assert b"SPH_NOALLOC_MAX_CELLS" in lib.sph_strerror(sph.SPH_ELIMIT)      # the message names the limit
    ok_grid = _params((256, 128, 128))                      # exactly 2^22: passes the size check ...
    assert lib.sph_comm_hash_noalloc(C.byref(ok_grid), -1, None, None, None, C.c_void_p(8), None) == sph.SPH_EINVAL
    assert lib.sph_comm_hash_noalloc(C.byref(ok_grid), 5, None, None, None, C.c_void_p(8), None) == sph.SPH_EINVAL
    assert lib.sph_comm_hash_noalloc(None, 0, None, None, None, C.c_void_p(8), None) == sph.SPH_EINVAL
    assert lib.sph_comm_hash_noalloc(C.byref(_params((4, 4, 0))), 0, None, None, None, C.c_void_p(8), None) == sph.SPH_EINVAL
