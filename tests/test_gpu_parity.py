"""GPU parity tests (-m gpu): the CUDA path through the C-ABI binding vs the CPU oracle.

Every case feeds the same seeded inputs (paper_2310_03596_b200.workloads) to both sides.
Sizes span several onesweep tiles (8192 keys) with a ragged tail; the full-size configs are
covered by tests/test_gpu_fullsize.py.
"""
import numpy as np
import pytest
import torch

from paper_2310_03596_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sph():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2310_03596_b200 import sph as s
    s.load_library()
    return s


# ------------------------------------------------------------------ whole step, lock-step parity
@pytest.mark.parametrize("flags", [0, 1], ids=["tiled", "direct"])
def test_cfg0_one_step(sph, oracle, flags):
    w = wl.config(0)
    rep = parity.lockstep(sph, oracle, w, steps=1, flags=flags)
    assert 0 < rep[0]["boundary"] < w.n


@pytest.mark.parametrize("flags", [0, 1], ids=["tiled", "direct"])
def test_t1b_every_float_path(sph, oracle, flags):
    w = wl.t1b()
    rep = parity.lockstep(sph, oracle, w, steps=3, flags=flags)
    assert rep[0]["pairs"] > 0


@pytest.mark.parametrize("k,side,steps", [(1, 33, 3), (2, 37, 3), (4, 29, 2)])
def test_scaled_configs(sph, oracle, k, side, steps):
    w = wl.config(k, side=side)          # odd sides: ragged tiles everywhere
    parity.lockstep(sph, oracle, w, steps=steps)


def test_scaled_config3_clipped_geometry(sph, oracle):
    w = wl.config(3, scale=0.1)          # plate + cylinders: long runs of empty buckets
    assert w.n > 20000, w.n
    parity.lockstep(sph, oracle, w, steps=2)


def test_t1b_bigger_many_steps(sph, oracle):
    w = wl.t1b(side=24, seed=1101)
    parity.lockstep(sph, oracle, w, steps=5)


# ------------------------------------------------------------------ degenerate cases
def test_single_owner_has_no_boundary(sph, oracle):
    w = wl.lattice_block(20, 20, 20, 0.1, 7, velocity=("normal", 0.05), owners=("single",))
    rep = parity.lockstep(sph, oracle, w, steps=1)
    assert rep[0]["boundary"] == 0


def test_random_owners_everything_is_boundary(sph, oracle):
    w = wl.lattice_block(20, 20, 20, 0.1, 8, velocity=("normal", 0.05), owners=("random", 16))
    rep = parity.lockstep(sph, oracle, w, steps=1)
    assert rep[0]["boundary"] == w.n


def test_32_owners(sph, oracle):
    w = wl.lattice_block(24, 20, 16, 0.1, 9, velocity=("normal", 0.05), owners=("random", 32))
    parity.lockstep(sph, oracle, w, steps=1)


def test_empty_and_tiny_inputs(sph, oracle):
    w = wl.t1b(side=6)
    for n in (0, 1, 2, 31, 33):
        sub = wl.Workload("sub", w.posm[:n].copy(), w.velr[:n].copy(), w.sig[:, :n].copy(),
                          w.owner[:n].copy(), w.origin, w.dims, n_owners=2)
        ctx = sph.Context.for_workload(sub, max_n=64)
        st = sph.State.from_numpy(sub.posm, sub.velr, sub.sig, sub.owner)
        out = ctx.alloc_outputs(n)
        ref = oracle.step(sub.posm, sub.velr, sub.sig, sub.owner, sub.origin, sub.dims, sub.h, sub.K,
                          sub.G, 2, sub.dt)
        ctx.sph_step(st, sub.dt, out)
        torch.cuda.synchronize()
        parity.compare_integers(out, ref, n)
        if n:
            parity.compare_rates(out, ref.rates)
            parity.compare_state(st, ref)
        ctx.close()


def test_single_bucket_grid_and_clamping(sph, oracle):
    # every particle far outside a 1x1x1 grid: clamped, zero sort passes
    w = wl.t1b(side=5)
    w.dims = np.array([1, 1, 1], np.int32)
    parity.lockstep(sph, oracle, w, steps=1)
    # a 2x3x2 grid with most particles clamped onto its border buckets
    w = wl.t1b(side=7)
    w.dims = np.array([2, 3, 2], np.int32)
    w.origin = np.array([1.0, 0.5, 2.0], np.float32)
    parity.lockstep(sph, oracle, w, steps=1)


def test_coincident_particles(sph, oracle):
    w = wl.t1b(side=8)
    w.posm[1::7, :3] = w.posm[0::7, :3][: w.posm[1::7].shape[0]]   # exact duplicates (S15)
    rep = parity.lockstep(sph, oracle, w, steps=1)
    assert np.isfinite(rep[0]["acc"])


def test_hash_at_bucket_faces(sph, oracle):
    # positions exactly on, and one ulp either side of, bucket faces (reading S2)
    h = np.float32(1.3)
    edge = np.float32(2.0) * h
    origin = np.array([-2.6, -2.6, -2.6], np.float32)
    dims = np.array([9, 9, 9], np.int32)
    faces = (np.arange(0, 9, dtype=np.float32) * edge + origin[0]).astype(np.float32)
    xs = np.concatenate([faces, np.nextafter(faces, np.float32(1e9)), np.nextafter(faces, np.float32(-1e9)),
                         np.array([-100.0, 100.0, 0.0, -0.0], np.float32)])
    n = xs.shape[0]
    posm = np.zeros((n, 4), np.float32)
    posm[:, 0] = xs
    posm[:, 1] = xs[::-1]
    posm[:, 2] = np.roll(xs, 5)
    ctx = sph.Context(origin, dims, h, max_n=n)
    got = parity.u32(ctx.sph_hash(torch.from_numpy(posm).cuda()))
    np.testing.assert_array_equal(got, oracle.hash(posm, origin, dims, h))
    ctx.close()


# ------------------------------------------------------------------ stage-by-stage C-ABI calls
def test_stage_calls_match_oracle(sph, oracle):
    w = wl.config(1, side=30)
    ctx = sph.Context.for_workload(w)
    st = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
    ref = oracle.step(w.posm, w.velr, w.sig, w.owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt)
    hsh = ctx.sph_hash(st.posm)
    sh, perm = ctx.sph_sort(hsh)
    srt = ctx.sph_reorder(perm, st)
    cs, ce = ctx.sph_cell_ranges(sh)
    ch, bids, cnt, oc = ctx.sph_comm_hash(sh, srt.owner, perm, cs, ce)
    drho, acc, dsig, pc = ctx.sph_interact(srt, sh, cs, ce)
    new = ctx.sph_integrate(w.dt, srt, drho, acc, dsig)
    torch.cuda.synchronize()
    out = sph.StepOutputs(hsh, sh, perm, cs, ce, ch, bids, cnt, oc, drho, acc, dsig, pc)
    parity.compare_integers(out, ref, w.n)
    parity.compare_rates(out, ref.rates)
    p = ref.perm.astype(np.int64)
    np.testing.assert_array_equal(srt.posm.cpu().numpy(), w.posm[p])
    np.testing.assert_array_equal(srt.velr.cpu().numpy(), w.velr[p])
    np.testing.assert_array_equal(srt.sig.cpu().numpy(), w.sig[:, p])
    np.testing.assert_array_equal(srt.owner.cpu().numpy(), w.owner[p])
    # sph_integrate is elementwise (sorted order in, sorted order out)
    assert parity.field_err(new.posm.cpu().numpy(), ref.posm[p]) <= parity.STATE_TOL
    assert parity.field_err(new.velr.cpu().numpy(), ref.velr[p]) <= parity.STATE_TOL
    assert parity.field_err(new.sig.cpu().numpy(), ref.sig[:, p]) <= parity.STATE_TOL
    assert ctx.launch_count() > 0
    ctx.close()


def test_sort_random_keys_many_tiles(sph, oracle):
    # sort alone on adversarial key distributions: uniform random, all equal, descending, two values
    rng = np.random.default_rng(5)
    dims = np.array([156, 156, 156], np.int32)     # 22 live bits, 3 passes
    cells = int(np.prod(dims.astype(np.int64)))
    n = 5 * 8192 + 1234
    ctx = sph.Context(np.zeros(3, np.float32), dims, 1.3, max_n=n)
    for keys in (rng.integers(0, cells, n), np.full(n, cells - 1), np.arange(n)[::-1] % cells,
                 rng.integers(0, 2, n) * (cells - 1), rng.integers(0, 300, n)):
        keys = keys.astype(np.uint32)
        sh, perm = ctx.sph_sort(torch.from_numpy(keys.view(np.int32)).cuda())
        rs, rp = oracle.sort(keys)
        np.testing.assert_array_equal(parity.u32(sh), rs)
        np.testing.assert_array_equal(parity.u32(perm), rp)
    ctx.close()


def test_sort_from_unaligned_key_pointer(sph, oracle):
    # include/sph.h promises 4-byte alignment for hash arrays: sort from views offset by 1, 2, 3 keys
    rng = np.random.default_rng(6)
    dims = np.array([79, 79, 79], np.int32)
    cells = int(np.prod(dims.astype(np.int64)))
    n = 3 * 8192 + 77
    ctx = sph.Context(np.zeros(3, np.float32), dims, 1.3, max_n=n)
    buf = torch.from_numpy(rng.integers(0, cells, n + 3).astype(np.uint32).view(np.int32)).cuda()
    for off in (1, 2, 3):
        view = buf[off:off + n]
        assert view.data_ptr() % 16 == 4 * off
        sh, perm = ctx.sph_sort(view)
        rs, rp = oracle.sort(parity.u32(view))
        np.testing.assert_array_equal(parity.u32(sh), rs)
        np.testing.assert_array_equal(parity.u32(perm), rp)
    ctx.close()


def test_step_host_end_to_end(sph, oracle):
    w = wl.t1b(side=12)
    ctx = sph.Context.for_workload(w)
    host = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner, device="cpu", pin=True)
    bids = np.zeros(w.n, np.uint32)
    m, pairs = ctx.sph_step_host(host, w.dt, steps=1, boundary_ids=bids)
    ref = oracle.step(w.posm, w.velr, w.sig, w.owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt)
    assert m == ref.boundary_ids.shape[0]
    np.testing.assert_array_equal(bids[:m], ref.boundary_ids)
    assert abs(pairs - ref.rates.pair_count) <= 2
    parity.compare_state(host, ref)
    ctx.close()


def test_step_host_two_streams_steps0_repeat_and_multistep(sph, oracle):
    """sph_step_host uploads posm on the ctx's stream and the rest of the state on a second one:
    steps = 0 must hand the state back bit for bit (the download has to wait for BOTH uploads),
    two calls of one step equal one call of two steps bit for bit (the staging is reused), and
    the two-step result matches the oracle run in lock-step."""
    w = wl.t1b(side=14, seed=1112)
    ctx = sph.Context.for_workload(w)
    host = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner, device="cpu", pin=True)
    m0, _ = ctx.sph_step_host(host, w.dt, steps=0)
    assert m0 == 0
    np.testing.assert_array_equal(host.posm.numpy(), w.posm)
    np.testing.assert_array_equal(host.velr.numpy(), w.velr)
    np.testing.assert_array_equal(host.sig.numpy(), w.sig)
    a = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner, device="cpu", pin=True)
    b = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner, device="cpu", pin=True)
    ctx.sph_step_host(a, w.dt, steps=1)
    r1 = oracle.step(w.posm, w.velr, w.sig, w.owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt)
    parity.compare_state(a, r1)
    ma, _ = ctx.sph_step_host(a, w.dt, steps=1)
    mb, _ = ctx.sph_step_host(b, w.dt, steps=2)
    assert ma == mb
    for x, y in ((a.posm, b.posm), (a.velr, b.velr), (a.sig, b.sig)):
        np.testing.assert_array_equal(x.numpy(), y.numpy())
    ctx.close()


def test_error_codes(sph):
    with pytest.raises(sph.SphError):
        sph.Context([0, 0, 0], [0, 1, 1], 1.3, max_n=10)
    with pytest.raises(sph.SphError):
        sph.Context([0, 0, 0], [4, 4, 4], -1.0, max_n=10)
    with pytest.raises(sph.SphError):
        sph.Context([0, 0, 0], [4, 4, 4], 1.3, n_owners=33, max_n=10)
    with pytest.raises(sph.SphError):
        sph.Context([0, 0, 0], [2048, 2048, 2048], 1.3, max_n=10)
    with pytest.raises(sph.SphError):
        sph.Context([0, 0, 0], [(1 << 24) + 1, 1, 1], 1.3, max_n=10)   # coordinate not exact in fp32
    sph.Context([0, 0, 0], [1 << 24, 1, 1], 1.3, max_n=10).close()
    ctx = sph.Context([0, 0, 0], [4, 4, 4], 1.3, max_n=8)
    with pytest.raises(sph.SphError):
        ctx.sph_hash(torch.zeros((9, 4), device="cuda"))       # n > max_n
    # the NEXT entry points reject bad arguments the same way
    posm = torch.zeros((8, 4), device="cuda")
    own = torch.zeros(8, dtype=torch.int32, device="cuda")
    with pytest.raises(sph.SphError):
        ctx.sph_balance(posm, own, hmax=0)
    with pytest.raises(sph.SphError):
        ctx.sph_balance(posm, own, hmax=2000)
    with pytest.raises(sph.SphError):
        ctx.sph_balance_types(posm, own, own, n_types=9)
    with pytest.raises(sph.SphError):
        ctx.sph_balance_types(posm, own, own, n_types=2, alpha=1.5)
    st = sph.State.empty(8)
    with pytest.raises(sph.SphError):
        ctx.sph_pack_boundary(st, own, 9)                      # m > n
    with pytest.raises(sph.SphError):
        ctx.sph_interact_split(st, own, own, own, 3)           # which must be 1 or 2
    ctx.close()


def test_repeated_runs_are_bit_identical(sph):
    """Race detector of last resort (compute-sanitizer is not available on the GPU pool): every
    kernel assigns its work deterministically (tickets only order the look-back), so repeated steps
    from the same state must agree bit for bit -- integers AND floats."""
    w = wl.config(2, side=41)
    ctx = sph.Context.for_workload(w)
    ref = None
    for rep in range(6):
        state = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
        out = ctx.alloc_outputs(w.n)
        ctx.sph_step(state, w.dt, out)
        ctx.sph_step(state, w.dt, out)
        torch.cuda.synchronize()
        got = [t.clone() for t in (out.perm, out.sorted_hash, out.cell_start, out.cell_end, out.comm_hash,
                                   out.boundary_count, out.owner_counts, out.drho, out.acc, out.dsig,
                                   out.pair_count, state.posm, state.velr, state.sig)]
        m = int(parity.u32(out.boundary_count)[0])
        got.append(out.boundary_ids[:m].clone())
        if ref is None:
            ref = got
        else:
            for a, b in zip(ref, got):
                assert torch.equal(a, b)
    ctx.close()


# ------------------------------------------------------------------ NEXT-1: per-owner send buffers
@pytest.mark.parametrize("make", [lambda: wl.config(0), lambda: wl.config(1, side=33),
                                  lambda: wl.config(2, side=37), lambda: wl.config(3, scale=0.1),
                                  lambda: wl.lattice_block(12, 12, 12, 0.1, 5, owners=("single",))],
                         ids=["cfg0", "cfg1", "cfg2", "cfg3", "one-owner"])
def test_pack_boundary_matches_oracle(sph, oracle, make):
    """sph_pack_boundary against oracle.pack_boundary: pure index and copy work,
    so everything is bit-exact.  The boundary list fed to both sides is the GPU step's, which the
    lock-step tests above pin to the oracle's."""
    w = make()
    ctx = sph.Context.for_workload(w)
    state = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
    out = ctx.alloc_outputs(w.n)
    ctx.sph_step(state, w.dt, out)
    torch.cuda.synchronize()
    m = int(parity.u32(out.boundary_count)[0])
    offs, ids, packed = ctx.sph_pack_boundary(state, out.boundary_ids, m)
    torch.cuda.synchronize()
    ref = oracle.pack_boundary(parity.u32(out.boundary_ids)[:m], state.owner.cpu().numpy(), w.n_owners,
                               state.posm.cpu().numpy(), state.velr.cpu().numpy(), state.sig.cpu().numpy())
    np.testing.assert_array_equal(parity.u32(offs), ref.offsets)
    np.testing.assert_array_equal(parity.u32(ids), ref.ids)
    np.testing.assert_array_equal(packed.posm.cpu().numpy(), ref.posm)
    np.testing.assert_array_equal(packed.velr.cpu().numpy(), ref.velr)
    np.testing.assert_array_equal(packed.sig.cpu().numpy(), ref.sig)
    np.testing.assert_array_equal(packed.owner.cpu().numpy(), ref.owner)
    np.testing.assert_array_equal(np.diff(ref.offsets.astype(np.int64)), parity.u32(out.owner_counts))
    ctx.close()


@pytest.mark.parametrize("scale", [0.93, 0.8], ids=["window-borderline", "window-overflow"])
def test_denser_packing_exercises_the_fallback_paths(sph, oracle, scale):
    """The tiled interaction kernel holds at most kCap window records and 640 table entries per
    bucket; denser regions fall back to the direct walk (whole tile, or single bucket).  Half of
    the block is compressed towards x = 0 so that tiled, borderline and fallback tiles coexist."""
    import dataclasses
    w = wl.t1b(side=22, seed=1103)
    posm = w.posm.copy()
    left = posm[:, 0] < 11.0
    posm[left, :3] *= np.float32(scale)               # denser on the left, unchanged lattice on the right
    w2 = dataclasses.replace(w, posm=posm, name=f"dense{scale}")
    rep = parity.lockstep(sph, oracle, w2, steps=2)
    assert rep[-1]["pairs"] > 0


# ------------------------------------------------------------------ NEXT-3: steps e and f as separate passes
@pytest.mark.parametrize("flags", [0, 1], ids=["tiled", "direct"])
@pytest.mark.parametrize("make", [lambda: wl.t1b(side=18, seed=1105), lambda: wl.config(2, side=33)],
                         ids=["t1b-mixed-owners", "cfg2"])
def test_split_passes_match_oracle_and_sum_to_single_pass(sph, oracle, make, flags):
    """sph_interact_split: each pass against oracle.interact_split at 1e-5 (per
    field, normalised by the SINGLE pass's field maximum), pair counts exact-ish (S25), and pass e +
    pass f against sph_interact."""
    w = make()
    owner = w.owner if w.n_owners > 2 else (np.arange(w.n) % 5).astype(np.int32)
    n_owners = max(w.n_owners, 5)
    ctx = sph.Context(w.origin, w.dims, w.h, w.K, w.G, n_owners=n_owners, max_n=w.n, flags=flags)
    state = sph.State.from_numpy(w.posm, w.velr, w.sig, owner)
    h = ctx.sph_hash(state.posm)
    sh, perm = ctx.sph_sort(h)
    st = ctx.sph_reorder(perm, state)
    cs, ce = ctx.sph_cell_ranges(sh)
    full = ctx.sph_interact(st, sh, cs, ce)
    torch.cuda.synchronize()
    p = parity.u32(perm)
    sp, sv, ss, so = w.posm[p], w.velr[p], np.ascontiguousarray(w.sig[:, p]), owner[p]
    args = (sp, sv, ss, parity.u32(sh), w.dims, parity.u32(cs), parity.u32(ce), w.h, w.K, w.G)
    ref_full = oracle.interact(*args)
    scale = {"drho": np.max(np.abs(ref_full.drho)), "acc": np.max(np.abs(ref_full.acc)),
             "dsig": np.max(np.abs(ref_full.dsig))}
    total = [0.0, 0.0, 0.0]
    pairs = 0
    for which in (1, 2):
        drho, acc, dsig, pc = ctx.sph_interact_split(st, sh, cs, ce, which)
        torch.cuda.synchronize()
        ref = oracle.interact_split(*args, so, which)
        g = {"drho": drho.cpu().numpy(), "acc": acc.cpu().numpy()[:, :3], "dsig": dsig.cpu().numpy().T}
        r = {"drho": ref.drho, "acc": ref.acc, "dsig": ref.dsig}
        for k_ in g:
            dif = np.max(np.abs(g[k_] - r[k_]))
            err = dif / scale[k_] if scale[k_] > 0 else (0.0 if dif < 1e-30 else np.inf)   # S21
            assert err <= parity.RATE_TOL, (which, k_, err)
        assert abs(int(pc.cpu()[0]) - ref.pair_count) <= max(1e-6 * ref.pair_count, 2)
        pairs += int(pc.cpu()[0])
        total = [total[0] + g["drho"], total[1] + g["acc"], total[2] + g["dsig"]]
    gf = [full[0].cpu().numpy(), full[1].cpu().numpy()[:, :3], full[2].cpu().numpy().T]
    for t_, f_, k_ in zip(total, gf, ("drho", "acc", "dsig")):
        dif = np.max(np.abs(t_ - f_))
        assert (dif / scale[k_] if scale[k_] > 0 else (0.0 if dif < 1e-30 else np.inf)) <= parity.RATE_TOL, k_
    assert abs(pairs - int(full[3].cpu()[0])) <= 4
    ctx.close()


# ------------------------------------------------------------------ NEXT-2: balancing sweep
@pytest.mark.parametrize("make,g", [(lambda: wl.lattice_block(24, 24, 24, 0.1, 21, owners=("random", 5)), 5),
                                    (lambda: wl.lattice_block(30, 26, 22, 0.1, 23, owners=("slabs_mixed", 3, 0.1)), 3),
                                    (lambda: wl.config(1, side=32), 4),
                                    (lambda: wl.config(4, side=20), 16),
                                    (lambda: wl.lattice_block(9, 9, 9, 0.1, 24, owners=("single",)), 1)],
                         ids=["random5", "mixed3", "slabs-fixed-point", "random16", "one-owner"])
def test_balance_sweep_matches_oracle_bit_exact(sph, oracle, make, g):
    """sph_balance against oracle.balance: labels, balancing hashes and the swap count
    are integers decided by pinned arithmetic (fixed-point Cg sums, fp64 projection without
    contraction) -- bit-exact, over three consecutive sweeps."""
    w = make()
    ctx = sph.Context.for_workload(w)
    posm = torch.from_numpy(w.posm).cuda()
    own_gpu = torch.from_numpy(w.owner.copy()).cuda()
    own_ref = w.owner.copy()
    for sweep in range(3):
        bh, sw = ctx.sph_balance(posm, own_gpu)
        torch.cuda.synchronize()
        own_ref, k, bh_ref = oracle.balance(w.posm, own_ref, g)
        assert int(sw.cpu()[0]) == k, sweep
        np.testing.assert_array_equal(bh.cpu().numpy(), bh_ref, err_msg=f"bal_hash sweep {sweep}")
        np.testing.assert_array_equal(own_gpu.cpu().numpy(), own_ref, err_msg=f"owner sweep {sweep}")
        np.testing.assert_array_equal(np.bincount(own_ref, minlength=g), np.bincount(w.owner, minlength=g))
    ctx.close()


@pytest.mark.parametrize("hmax", [1, 5, 37])
def test_balance_tie_heavy_small_hmax(sph, oracle, hmax):
    """Few hash values (hmax = 1, 5, 37 on 46 k particles): thousands of particles share the
    threshold hash of every pair, so the id-ordered choice among the ties (reading B6; a three-level
    radix select on the id in the kernel, a sort in the oracle) decides almost every swap."""
    w = wl.lattice_block(40, 36, 32, 0.1, 29, owners=("random", 4))
    ctx = sph.Context.for_workload(w)
    posm = torch.from_numpy(w.posm).cuda()
    own_gpu = torch.from_numpy(w.owner.copy()).cuda()
    own_ref = w.owner.copy()
    for sweep in range(2):
        bh, sw = ctx.sph_balance(posm, own_gpu, hmax=hmax)
        torch.cuda.synchronize()
        own_ref, k, bh_ref = oracle.balance(w.posm, own_ref, 4, hmax=hmax)
        assert int(sw.cpu()[0]) == k and (sweep > 0 or k > 0), sweep
        np.testing.assert_array_equal(bh.cpu().numpy(), bh_ref, err_msg=f"bal_hash sweep {sweep}")
        np.testing.assert_array_equal(own_gpu.cpu().numpy(), own_ref, err_msg=f"owner sweep {sweep}")
    ctx.close()


@pytest.mark.parametrize("g,nt,alpha", [(3, 2, 0.1), (5, 3, 0.1), (4, 2, 1.0), (4, 1, 0.0)])
def test_balance_types_matches_oracle_bit_exact(sph, oracle, g, nt, alpha):
    """sph_balance_types (Cg' = alpha Cg_all + (1 - alpha) Cg_type) against
    oracle.balance_types, bit-exact over two sweeps; every (owner, type) count is kept."""
    w = wl.lattice_block(26, 22, 20, 0.1, 31 + g, owners=("random", g))
    rng = np.random.default_rng(100 + g)
    ptype = rng.integers(0, nt, w.n).astype(np.int32)
    ctx = sph.Context.for_workload(w)
    posm = torch.from_numpy(w.posm).cuda()
    pt = torch.from_numpy(ptype).cuda()
    own_gpu = torch.from_numpy(w.owner.copy()).cuda()
    own_ref = w.owner.copy()
    for sweep in range(2):
        bh, sw = ctx.sph_balance_types(posm, own_gpu, pt, nt, alpha)
        torch.cuda.synchronize()
        own_ref, k, bh_ref = oracle.balance_types(w.posm, own_ref, ptype, g, nt, alpha=alpha)
        assert int(sw.cpu()[0]) == k and k > 0
        np.testing.assert_array_equal(bh.cpu().numpy(), bh_ref)
        np.testing.assert_array_equal(own_gpu.cpu().numpy(), own_ref)
    for t in range(nt):
        np.testing.assert_array_equal(np.bincount(own_ref[ptype == t], minlength=g),
                                      np.bincount(w.owner[ptype == t], minlength=g))
    ctx.close()


@pytest.mark.parametrize("flags", [0, 1], ids=["tiled", "direct"])
@pytest.mark.parametrize("make,dense", [(lambda: wl.t1b(side=18, seed=1105), False), (lambda: wl.config(2, side=33), False),
                                        (lambda: wl.config(4, side=29), True)], ids=["t1b", "cfg2", "cfg4-dense"])
def test_interact_ef_one_search_two_rate_sets(sph, oracle, make, dense, flags):
    """sph_interact_ef: steps e and f from ONE neighbour search.  Each rate set
    against orc_interact_split, pair counts exact against the split calls, e + f = single pass.
    The dense case (lattice squeezed to 0.85) drives tiles into the direct-walk fallbacks."""
    w = make()
    if w.sig.max() == 0:
        rng = np.random.default_rng(78)
        w.sig[:] = (rng.standard_normal((6, w.n)) * 1e-3).astype(np.float32)
        w.velr[:, 3] = (1.0 + (rng.random(w.n) * 2 - 1) * 0.01).astype(np.float32)
    if dense:
        w.posm[:, :3] *= np.float32(0.85)
    ctx = sph.Context.for_workload(w, flags=flags)
    st = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
    sh, perm = ctx.sph_sort(ctx.sph_hash(st.posm))
    sst = ctx.sph_reorder(perm, st)
    cs, ce = ctx.sph_cell_ranges(sh)
    e, f, pc = ctx.sph_interact_ef(sst, sh, cs, ce)
    single = ctx.sph_interact(sst, sh, cs, ce)
    se = ctx.sph_interact_split(sst, sh, cs, ce, 1)
    sf = ctx.sph_interact_split(sst, sh, cs, ce, 2)
    torch.cuda.synchronize()
    p = parity.u32(perm).astype(np.int64)
    args = (w.posm[p], w.velr[p], np.ascontiguousarray(w.sig[:, p]), parity.u32(sh), w.dims, parity.u32(cs),
            parity.u32(ce), w.h, w.K, w.G)
    full = oracle.interact(*args)
    scale = {k: max(np.abs(getattr(full, k)).max(), 1e-300) for k in ("drho", "acc", "dsig")}
    pcs = pc.cpu().numpy()
    assert pcs[0] == int(se[3].cpu()[0]) and pcs[1] == int(sf[3].cpu()[0])
    assert pcs[0] + pcs[1] == int(single[3].cpu()[0])
    tot = {}
    for which, got in ((1, e), (2, f)):
        ref = oracle.interact_split(*args, w.owner[p], which)
        g = {"drho": got[0].cpu().numpy(), "acc": got[1].cpu().numpy()[:, :3], "dsig": got[2].cpu().numpy().T}
        for name in ("drho", "acc", "dsig"):
            err = np.abs(g[name] - getattr(ref, name)).max() / scale[name]
            assert err <= parity.RATE_TOL, (which, name, err)
            tot[name] = tot.get(name, 0) + g[name]
        assert abs(int(pcs[which - 1]) - ref.pair_count) <= max(1e-6 * ref.pair_count, 2)
    sg = {"drho": single[0].cpu().numpy(), "acc": single[1].cpu().numpy()[:, :3], "dsig": single[2].cpu().numpy().T}
    for name in ("drho", "acc", "dsig"):
        assert np.abs(tot[name] - sg[name]).max() <= parity.RATE_TOL * scale[name], name
    ctx.close()


# ------------------------------------------------------------------ NEXT-4: per-particle smoothing lengths
@pytest.mark.parametrize("flags", [0, 1], ids=["tiled", "direct"])
@pytest.mark.parametrize("kind", [("species", 2, 0.75), ("random", 0.5), ("uniform",)],
                         ids=["two-species", "random", "uniform"])
def test_varh_step_matches_oracle(sph, oracle, kind, flags):
    """sph_step_varh (readings H1-H3) lock-step against the oracle: integers
    bit-exact (they do not depend on h), rates 1e-5, state 1e-6, pair counts 1e-6."""
    w = wl.t1b(side=18, seed=1108)
    hp = wl.particle_h(w, kind)
    rep = parity.lockstep(sph, oracle, w, steps=2, flags=flags, hp=hp)
    assert rep[0]["pairs"] > 0
    if kind[0] != "uniform":
        full = parity.lockstep(sph, oracle, w, steps=1, flags=flags)
        assert rep[0]["pairs"] < full[0]["pairs"]         # shorter lengths lose neighbours


def test_varh_scaled_config_many_tiles_and_split_passes(sph, oracle):
    """Several tiles with ragged edges, 16 mixed owners, three species; the stage call with
    which = 0 / 1 / 2 against orc_interact_varh, and pass e + pass f = the single pass."""
    w = wl.config(2, side=33)
    rng = np.random.default_rng(77)                        # a state in which every rate is non-trivial
    w.sig[:] = (rng.standard_normal((6, w.n)) * 1e-3).astype(np.float32)
    w.velr[:, :3] += (rng.standard_normal((w.n, 3)) * 0.01).astype(np.float32)
    w.velr[:, 3] = (1.0 + (rng.random(w.n) * 2 - 1) * 0.01).astype(np.float32)
    hp = wl.particle_h(w, ("species", 3, 0.6))
    ctx = sph.Context.for_workload(w)
    st = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
    hh = ctx.sph_hash(st.posm)
    sh, perm = ctx.sph_sort(hh)
    sst = ctx.sph_reorder(perm, st)
    cs, ce = ctx.sph_cell_ranges(sh)
    p = parity.u32(perm).astype(np.int64)
    sh_h = torch.from_numpy(hp[p]).cuda()
    sp, sv, ss, so = w.posm[p], w.velr[p], np.ascontiguousarray(w.sig[:, p]), w.owner[p]
    res = {}
    for which in (0, 1, 2):
        drho, acc, dsig, pc = ctx.sph_interact_varh(sst, sh_h, sh, cs, ce, which)
        torch.cuda.synchronize()
        ref = oracle.interact_varh(sp, sv, ss, hp[p], parity.u32(sh), w.dims, parity.u32(cs), parity.u32(ce),
                                   w.h, w.K, w.G, owner=so, which=which)
        if which == 0:
            scale = {"drho": np.abs(ref.drho).max(), "acc": np.abs(ref.acc).max(), "dsig": np.abs(ref.dsig).max()}
        got = {"drho": drho.cpu().numpy(), "acc": acc.cpu().numpy()[:, :3], "dsig": dsig.cpu().numpy().T}
        for name in ("drho", "acc", "dsig"):
            err = np.abs(got[name] - getattr(ref, name)).max() / scale[name]
            assert err <= parity.RATE_TOL, (which, name, err)
        assert abs(int(pc.cpu()[0]) - ref.pair_count) <= max(1e-6 * ref.pair_count, 2)
        res[which] = (got, int(pc.cpu()[0]))
    assert res[1][1] + res[2][1] == res[0][1]
    for name in ("drho", "acc", "dsig"):
        assert np.abs(res[1][0][name] + res[2][0][name] - res[0][0][name]).max() <= parity.RATE_TOL * scale[name]
    # both passes from ONE search with per-particle lengths (sph_interact_ef, sorted_h != NULL),
    # tiled and direct kernel: each rate set against orc_interact_varh(which = 1 / 2), counts exact
    # against the split calls above
    for flags in (0, 1):
        c2 = ctx if flags == 0 else sph.Context.for_workload(w, flags=1)
        e, f, pcs = c2.sph_interact_ef(sst, sh, cs, ce, sorted_h=sh_h)
        torch.cuda.synchronize()
        pcs = pcs.cpu().numpy()
        assert int(pcs[0]) == res[1][1] and int(pcs[1]) == res[2][1], (flags, pcs, res[1][1], res[2][1])
        for which, got_t in ((1, e), (2, f)):
            ref = oracle.interact_varh(sp, sv, ss, hp[p], parity.u32(sh), w.dims, parity.u32(cs), parity.u32(ce),
                                       w.h, w.K, w.G, owner=so, which=which)
            got = {"drho": got_t[0].cpu().numpy(), "acc": got_t[1].cpu().numpy()[:, :3],
                   "dsig": got_t[2].cpu().numpy().T}
            for name in ("drho", "acc", "dsig"):
                err = np.abs(got[name] - getattr(ref, name)).max() / scale[name]
                assert err <= parity.RATE_TOL, ("ef", flags, which, name, err)
        if c2 is not ctx:
            c2.close()
    ctx.close()


def test_long_run_then_lockstep(sph, oracle):
    """300 steps of the benchmark's configuration on a scaled configs[1] (state re-hashed and
    re-sorted every step), then one lock-step comparison with the oracle from the GPU's state:
    accumulated drift must not break any stage (particles have moved across bucket faces by then)."""
    w = wl.config(1, side=33)
    ctx = sph.Context.for_workload(w)
    state = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
    for _ in range(300):
        ctx.sph_step(state, 10 * w.dt)                 # larger dt: particles really travel
    torch.cuda.synchronize()
    posm, velr = state.posm.cpu().numpy(), state.velr.cpu().numpy()
    sig, owner = state.sig.cpu().numpy(), state.owner.cpu().numpy()
    assert np.isfinite(posm).all() and np.isfinite(velr).all() and np.isfinite(sig).all()
    moved = np.abs(posm[:, :3] - w.posm[:, :3]).max()
    assert moved > 1e-3, moved
    ref = oracle.step(posm, velr, sig, owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt)
    out = ctx.alloc_outputs(w.n)
    ctx.sph_step(state, w.dt, out)
    torch.cuda.synchronize()
    parity.compare_integers(out, ref, w.n)
    parity.compare_rates(out, ref.rates)
    parity.compare_state(state, ref)
    ctx.close()


def test_balancing_cadence_inside_a_run(sph, oracle):
    """PAPER.md:32 "activate the balancing algorithm every 20 integration loops": 20 sph_steps, one
    sph_balance sweep on the positions the run has reached (bit-exact labels against the oracle),
    then the step AFTER the labels changed in lock-step against the oracle -- the new labels must
    reach the communication hash, the boundary list and the owner counts; twice in a row."""
    w = wl.config(2, side=37)
    g = w.n_owners
    ctx = sph.Context.for_workload(w)
    state = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
    out = ctx.alloc_outputs(w.n)
    count0 = np.bincount(w.owner, minlength=g)
    boundary = []
    for cycle in range(2):
        for _ in range(20):
            ctx.sph_step(state, w.dt)
        torch.cuda.synchronize()
        posm = state.posm.cpu().numpy()
        own_before = state.owner.cpu().numpy()
        own_ref, k, bh_ref = oracle.balance(posm, own_before, g)
        bh, sw = ctx.sph_balance(state.posm, state.owner)
        torch.cuda.synchronize()
        assert int(sw.cpu()[0]) == k and k > 0, (cycle, k)
        np.testing.assert_array_equal(bh.cpu().numpy(), bh_ref)
        np.testing.assert_array_equal(state.owner.cpu().numpy(), own_ref)
        np.testing.assert_array_equal(np.bincount(own_ref, minlength=g), count0)
        # the step after the sweep, from the GPU's state with the NEW labels
        velr, sig = state.velr.cpu().numpy(), state.sig.cpu().numpy()
        ref = oracle.step(posm, velr, sig, own_ref, w.origin, w.dims, w.h, w.K, w.G, g, w.dt)
        stale = oracle.step(posm, velr, sig, own_before, w.origin, w.dims, w.h, w.K, w.G, g, w.dt, floats=False)
        assert not np.array_equal(ref.comm_hash, stale.comm_hash) or \
            not np.array_equal(ref.owner_counts, stale.owner_counts)   # the sweep changed stage 3's product
        ctx.sph_step(state, w.dt, out)
        torch.cuda.synchronize()
        parity.compare_integers(out, ref, w.n)
        parity.compare_rates(out, ref.rates)
        parity.compare_state(state, ref)
        np.testing.assert_array_equal(state.owner.cpu().numpy(), own_ref)
        boundary.append(int(ref.boundary_ids.shape[0]))
    ctx.close()


def test_balance_three_owner_golden_example_on_the_gpu(sph):
    """The hand-worked three-owner sweep of tests/golden/balancing_three_owner_example.txt (pair
    order (0,1), (0,2), (1,2), Cgs recomputed after every pair -- reading B1) through
    sph_balance and sph_balance_types (one type, alpha = 0): compared with the file, not the oracle."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "balancing_three_owner_example.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    posm = np.zeros((len(rows), 4), np.float32)
    posm[:, 0] = [float(r[1]) for r in rows]; posm[:, 3] = 1
    own0 = np.array([int(r[2]) for r in rows], np.int32)
    ctx = sph.Context(origin=(-1.0, -1.0, -1.0), dims=(8, 2, 2), h=1.0, n_owners=3, max_n=len(rows))
    p = torch.from_numpy(posm).cuda()
    for typed in (False, True):
        own = torch.from_numpy(own0.copy()).cuda()
        if typed:
            bh, sw = ctx.sph_balance_types(p, own, torch.zeros(len(rows), dtype=torch.int32, device="cuda"), 1, 0.0)
        else:
            bh, sw = ctx.sph_balance(p, own)
        torch.cuda.synchronize()
        assert int(sw.cpu()[0]) == 3
        np.testing.assert_array_equal(bh.cpu().numpy(), [int(r[3]) for r in rows])
        np.testing.assert_array_equal(own.cpu().numpy(), [int(r[4]) for r in rows])
    ctx.close()


# ------------------------------------------------------------------ NEXT-1, second half: per-destination lists
@pytest.mark.parametrize("make", [lambda: wl.config(0), lambda: wl.config(1, side=33), lambda: wl.config(2, side=37),
                                  lambda: wl.config(3, scale=0.1), lambda: wl.config(4, side=29),
                                  lambda: wl.lattice_block(20, 20, 20, 0.1, 25, owners=("random", 32)),
                                  lambda: wl.lattice_block(9, 9, 9, 0.1, 24, owners=("single",)),
                                  lambda: wl.lattice_block(40, 6, 6, 0.1, 80, owners=("slabs", 3))],
                         ids=["cfg0", "cfg1", "cfg2", "cfg3-rcb", "cfg4", "32-owners", "one-owner", "wide-slabs"])
def test_pack_destinations_matches_oracle(sph, oracle, make):
    """sph_pack_destinations (PAPER.md:23 step d, reading D1) against orc_pack_destinations, bit-exact:
    offsets and every list; also the count-only call, a too-small buffer (nothing written beyond
    its capacity, total still reported) and a second call on the same ctx (scratch re-use)."""
    w = make()
    g = w.n_owners
    ctx = sph.Context.for_workload(w)
    st = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner)
    sh, perm = ctx.sph_sort(ctx.sph_hash(st.posm))
    so = st.owner[perm.long()].contiguous()
    cs, ce = ctx.sph_cell_ranges(sh)
    torch.cuda.synchronize()
    p = parity.u32(perm)
    ref_off, ref_ids = oracle.pack_destinations(parity.u32(sh), w.owner[p.astype(np.int64)], p, w.dims,
                                                parity.u32(cs), parity.u32(ce), g)
    for rep in range(2):
        offs, ids = ctx.sph_pack_destinations(sh, so, perm)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(parity.u32(offs), ref_off, err_msg=f"dest_offsets (call {rep})")
        np.testing.assert_array_equal(parity.u32(ids), ref_ids, err_msg=f"dest_ids (call {rep})")
    # union of the lists = the boundary set stage 3 produces
    _, bids, cnt, _ = ctx.sph_comm_hash(sh, so, perm, cs, ce)
    torch.cuda.synchronize()
    m = int(parity.u32(cnt)[0])
    np.testing.assert_array_equal(np.unique(ref_ids), np.sort(parity.u32(bids)[:m]))
    assert ref_ids.size <= m * max(g - 1, 0)
    # a buffer that is too small: the head is written, the guard word behind it is not, the total is
    total = int(ref_off[-1])
    if total > 1:
        cap = total // 2
        buf = torch.full((cap + 1,), -1, dtype=torch.int32, device="cuda")
        offs2, _ = ctx.sph_pack_destinations(sh, so, perm, dest_ids=buf[:cap])
        torch.cuda.synchronize()
        assert int(parity.u32(offs2)[-1]) == total
        got = parity.u32(buf)
        assert got[cap] == 0xFFFFFFFF
        # slots below cap belong to the lists that start below cap
        np.testing.assert_array_equal(got[:cap], ref_ids[:cap])
    ctx.close()
