"""CPU oracle for the SPH hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front end to oracle/sph_oracle.c (plain single-threaded C, fp64).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package; it imports nothing from paper_2310_03596_b200.

Every function cites the passage it follows in sph_oracle.c; `step` chains them in the order of
PAPER.md:19-26 (steps a, c, e/f, g; steps b and d are the multi-GPU exchange, out of scope).
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

GARBAGE = 0xFFFFFFFF

_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(_build.build())
    i64, f32, f64, vp = C.c_int64, C.c_float, C.c_double, C.c_void_p
    lib.orc_hash.argtypes = [i64, vp, vp, vp, f32, vp]
    lib.orc_hash.restype = None
    lib.orc_sort.argtypes = [i64, vp, vp, vp]
    lib.orc_sort.restype = C.c_int
    lib.orc_cell_ranges.argtypes = [i64, vp, i64, vp, vp]
    lib.orc_cell_ranges.restype = None
    lib.orc_comm_hash.argtypes = [i64, vp, vp, vp, vp, vp, vp]
    lib.orc_comm_hash.restype = None
    lib.orc_boundary.argtypes = [i64, vp, vp, vp, C.c_int32, vp, vp]
    lib.orc_boundary.restype = i64
    lib.orc_pack_boundary.argtypes = [i64, i64, vp, vp, C.c_int32] + [vp] * 9
    lib.orc_pack_boundary.restype = None
    lib.orc_pack_destinations.argtypes = [i64, vp, vp, vp, vp, vp, vp, C.c_int32, vp, vp, i64]
    lib.orc_pack_destinations.restype = i64
    lib.orc_balance.argtypes = [i64, vp, vp, C.c_int32, C.c_int32, vp]
    lib.orc_balance.restype = i64
    lib.orc_balance_types.argtypes = [i64, vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, f64, vp]
    lib.orc_balance_types.restype = i64
    lib.orc_kernel_W.argtypes = [f64, f64]
    lib.orc_kernel_W.restype = f64
    lib.orc_kernel_F.argtypes = [f64, f64]
    lib.orc_kernel_F.restype = f64
    lib.orc_interact.argtypes = [i64, vp, vp, vp, vp, vp, vp, vp, f32, f32, f32, i64, vp,
                                 vp, vp, vp, vp, vp]
    lib.orc_interact.restype = None
    lib.orc_interact_split.argtypes = [i64, vp, vp, vp, vp, vp, vp, vp, f32, f32, f32, vp, C.c_int,
                                       i64, vp, vp, vp, vp, vp, vp]
    lib.orc_interact_split.restype = None
    lib.orc_interact_varh.argtypes = [i64, vp, vp, vp, vp, vp, vp, vp, vp, f32, f32, f32, vp, C.c_int,
                                      i64, vp, vp, vp, vp, vp, vp]
    lib.orc_interact_varh.restype = None
    lib.orc_integrate.argtypes = [i64, f64, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.orc_integrate.restype = None
    _lib = lib
    return lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def kernel_W(r: float, h: float) -> float:
    return _load().orc_kernel_W(float(r), float(h))


def kernel_F(r: float, h: float) -> float:
    return _load().orc_kernel_F(float(r), float(h))


def hash(posm, origin, dims, h) -> np.ndarray:  # noqa: A001 - the paper's word
    posm = _c(posm, np.float32)
    origin = _c(origin, np.float32)
    dims = _c(dims, np.int32)
    n = posm.shape[0]
    out = np.empty(n, np.uint32)
    _load().orc_hash(n, _p(posm), _p(origin), _p(dims), np.float32(h), _p(out))
    return out


def sort(hash_):
    hash_ = _c(hash_, np.uint32)
    n = hash_.shape[0]
    sh = np.empty(n, np.uint32)
    perm = np.empty(n, np.uint32)
    rc = _load().orc_sort(n, _p(hash_), _p(sh), _p(perm))
    if rc != 0:
        raise MemoryError("orc_sort")
    return sh, perm


def cell_ranges(sorted_hash, n_cells: int):
    sorted_hash = _c(sorted_hash, np.uint32)
    start = np.empty(n_cells, np.uint32)
    end = np.empty(n_cells, np.uint32)
    _load().orc_cell_ranges(sorted_hash.shape[0], _p(sorted_hash), int(n_cells), _p(start), _p(end))
    return start, end


def comm_hash(sorted_hash, sorted_owner, dims, cell_start, cell_end) -> np.ndarray:
    sorted_hash = _c(sorted_hash, np.uint32)
    sorted_owner = _c(sorted_owner, np.int32)
    dims = _c(dims, np.int32)
    cell_start = _c(cell_start, np.uint32)
    cell_end = _c(cell_end, np.uint32)
    out = np.empty(sorted_hash.shape[0], np.uint32)
    _load().orc_comm_hash(sorted_hash.shape[0], _p(sorted_hash), _p(sorted_owner), _p(dims),
                          _p(cell_start), _p(cell_end), _p(out))
    return out


def boundary(comm_hash_, perm, sorted_owner, n_owners: int):
    comm_hash_ = _c(comm_hash_, np.uint32)
    perm = _c(perm, np.uint32)
    sorted_owner = _c(sorted_owner, np.int32)
    n = comm_hash_.shape[0]
    ids = np.empty(max(n, 1), np.uint32)
    counts = np.zeros(n_owners, np.uint32)
    m = _load().orc_boundary(n, _p(comm_hash_), _p(perm), _p(sorted_owner), int(n_owners),
                             _p(ids), _p(counts))
    if m < 0:
        raise MemoryError("orc_boundary")
    return ids[:m].copy(), counts


def balance(posm, owner, n_owners: int, hmax: int = 1000):
    """One sweep of the paper's communication-load balancing over all owner pairs (sph_oracle.c
    O10).  Returns (new owner labels, number of swapped pairs, balancing hash of the
    last pair that touched each particle)."""
    posm = _c(posm, np.float32)
    own = np.array(owner, dtype=np.int32, copy=True)
    bh = np.zeros(posm.shape[0], np.int32)
    k = _load().orc_balance(posm.shape[0], _p(posm), _p(own), int(n_owners), int(hmax), _p(bh))
    if k < 0:
        raise MemoryError("orc_balance")
    return own, int(k), bh


def balance_types(posm, owner, ptype, n_owners: int, n_types: int, hmax: int = 1000, alpha: float = 0.1):
    """Balancing sweep per particle type with the biased Cg' of PAPER.md:56 (sph_oracle.c O11)."""
    posm = _c(posm, np.float32)
    ptype = _c(ptype, np.int32)
    own = np.array(owner, dtype=np.int32, copy=True)
    bh = np.zeros(posm.shape[0], np.int32)
    k = _load().orc_balance_types(posm.shape[0], _p(posm), _p(own), _p(ptype), int(n_owners), int(n_types),
                                  int(hmax), float(alpha), _p(bh))
    if k < 0:
        raise MemoryError("orc_balance_types")
    return own, int(k), bh


@dataclass
class PackedBoundary:
    offsets: np.ndarray      # [n_owners + 1] u32, segment g = [offsets[g], offsets[g + 1])
    ids: np.ndarray          # [M] u32, per segment in (hash, id) order
    posm: np.ndarray         # [M,4] f32
    velr: np.ndarray         # [M,4] f32
    sig: np.ndarray          # [6,M] f32
    owner: np.ndarray        # [M] i32


def pack_boundary(boundary_ids, owner, n_owners: int, posm, velr, sig) -> PackedBoundary:
    """Per-owner send buffers (sph_oracle.c O5b).  State arrays in id order; sig is [6, n]."""
    boundary_ids = _c(boundary_ids, np.uint32)
    owner = _c(owner, np.int32)
    posm = _c(posm, np.float32)
    velr = _c(velr, np.float32)
    sig = _c(sig, np.float32)
    n, m = posm.shape[0], boundary_ids.shape[0]
    off = np.zeros(n_owners + 1, np.uint32)
    ids = np.empty(max(m, 1), np.uint32)
    pp = np.empty((max(m, 1), 4), np.float32)
    pv = np.empty((max(m, 1), 4), np.float32)
    ps = np.empty((6, max(m, 1)), np.float32)
    po = np.empty(max(m, 1), np.int32)
    if m == 0:
        return PackedBoundary(off, ids[:0], pp[:0], pv[:0], ps[:, :0], po[:0])
    _load().orc_pack_boundary(n, m, _p(boundary_ids), _p(owner), int(n_owners), _p(posm), _p(velr),
                              _p(sig), _p(off), _p(ids), _p(pp), _p(pv), _p(ps), _p(po))
    return PackedBoundary(off, ids, pp, pv, ps, po)


def pack_destinations(sorted_hash, sorted_owner, perm, dims, cell_start, cell_end, n_owners: int):
    """Per-destination send lists (sph_oracle.c O5c, reading D1): returns
    (dest_offsets [n_owners + 1] u32, dest_ids [total] u32); list g = dest_ids[offsets[g]:offsets[g + 1]]
    = ids, in (hash, id) order, of the particles not owned by g that have a particle of g in their
    27-bucket stencil.  All inputs in sorted order."""
    sorted_hash = _c(sorted_hash, np.uint32)
    sorted_owner = _c(sorted_owner, np.int32)
    perm = _c(perm, np.uint32)
    dims = _c(dims, np.int32)
    cell_start = _c(cell_start, np.uint32)
    cell_end = _c(cell_end, np.uint32)
    n = sorted_hash.shape[0]
    off = np.zeros(n_owners + 1, np.uint32)
    lib = _load()
    total = lib.orc_pack_destinations(n, _p(sorted_hash), _p(sorted_owner), _p(perm), _p(dims), _p(cell_start),
                                      _p(cell_end), int(n_owners), _p(off), None, 0)
    ids = np.empty(max(total, 1), np.uint32)
    t2 = lib.orc_pack_destinations(n, _p(sorted_hash), _p(sorted_owner), _p(perm), _p(dims), _p(cell_start),
                                   _p(cell_end), int(n_owners), _p(off), _p(ids), total)
    assert t2 == total
    return off, ids[:total]


@dataclass
class Rates:
    drho: np.ndarray        # [m]      f64
    L: np.ndarray           # [m,3,3]  f64  L[a][b] = d v_a / d x_b
    acc: np.ndarray         # [m,3]    f64
    dsig: np.ndarray        # [m,6]    f64  xx,yy,zz,xy,xz,yz
    pair_count: int


def interact(posm, velr, sig, sorted_hash, dims, cell_start, cell_end, h, K, G, idx=None) -> Rates:
    """All arrays in sorted order.  sig is [6, n]."""
    posm = _c(posm, np.float32)
    velr = _c(velr, np.float32)
    sig = _c(sig, np.float32)
    n = posm.shape[0]
    assert posm.shape == (n, 4) and velr.shape == (n, 4) and sig.shape == (6, n)
    sorted_hash = _c(sorted_hash, np.uint32)
    dims = _c(dims, np.int32)
    cell_start = _c(cell_start, np.uint32)
    cell_end = _c(cell_end, np.uint32)
    if idx is not None:
        idx = _c(idx, np.int64)
        m = idx.shape[0]
    else:
        m = n
    drho = np.zeros(m, np.float64)
    L = np.zeros((m, 3, 3), np.float64)
    acc = np.zeros((m, 3), np.float64)
    dsig = np.zeros((m, 6), np.float64)
    pc = C.c_int64(0)
    _load().orc_interact(n, _p(posm), _p(velr), _p(sig), _p(sorted_hash), _p(dims), _p(cell_start),
                         _p(cell_end), np.float32(h), np.float32(K), np.float32(G),
                         m if idx is not None else 0, _p(idx) if idx is not None else None,
                         _p(drho), _p(L), _p(acc), _p(dsig), C.byref(pc))
    return Rates(drho, L, acc, dsig, int(pc.value))


def interact_split(posm, velr, sig, sorted_hash, dims, cell_start, cell_end, h, K, G, owner, which,
                   idx=None) -> Rates:
    """Step e alone (which = 1: same-owner neighbours) or step f alone (which = 2: other owners);
    sph_oracle.c orc_interact_split.  All arrays in sorted order; idx = sorted
    positions to compute (None = all)."""
    posm = _c(posm, np.float32)
    velr = _c(velr, np.float32)
    sig = _c(sig, np.float32)
    owner = _c(owner, np.int32)
    n = posm.shape[0]
    sorted_hash = _c(sorted_hash, np.uint32)
    dims = _c(dims, np.int32)
    cell_start = _c(cell_start, np.uint32)
    cell_end = _c(cell_end, np.uint32)
    if idx is not None:
        idx = _c(idx, np.int64)
        m = idx.shape[0]
    else:
        m = n
    drho = np.zeros(m, np.float64)
    L = np.zeros((m, 3, 3), np.float64)
    acc = np.zeros((m, 3), np.float64)
    dsig = np.zeros((m, 6), np.float64)
    pc = C.c_int64(0)
    _load().orc_interact_split(n, _p(posm), _p(velr), _p(sig), _p(sorted_hash), _p(dims), _p(cell_start),
                               _p(cell_end), np.float32(h), np.float32(K), np.float32(G), _p(owner),
                               int(which), m if idx is not None else 0,
                               _p(idx) if idx is not None else None,
                               _p(drho), _p(L), _p(acc), _p(dsig), C.byref(pc))
    return Rates(drho, L, acc, dsig, int(pc.value))


def interact_varh(posm, velr, sig, hp, sorted_hash, dims, cell_start, cell_end, hmax, K, G, owner=None, which=0,
                  idx=None) -> Rates:
    """O7 with a smoothing length per particle (sph_oracle.c orc_interact_varh; PAPER.md:13, 54;
    readings H1-H3): pair length h_ij = (h_i + h_j) / 2, bucket grid on hmax.  All arrays in sorted
    order; owner / which select a split pass, idx a sample of sorted positions."""
    posm = _c(posm, np.float32)
    velr = _c(velr, np.float32)
    sig = _c(sig, np.float32)
    hp = _c(hp, np.float32)
    n = posm.shape[0]
    assert hp.shape == (n,)
    if owner is not None:
        owner = _c(owner, np.int32)
    sorted_hash = _c(sorted_hash, np.uint32)
    dims = _c(dims, np.int32)
    cell_start = _c(cell_start, np.uint32)
    cell_end = _c(cell_end, np.uint32)
    if idx is not None:
        idx = _c(idx, np.int64)
        m = idx.shape[0]
    else:
        m = n
    drho = np.zeros(m, np.float64)
    L = np.zeros((m, 3, 3), np.float64)
    acc = np.zeros((m, 3), np.float64)
    dsig = np.zeros((m, 6), np.float64)
    pc = C.c_int64(0)
    _load().orc_interact_varh(n, _p(posm), _p(velr), _p(sig), _p(hp), _p(sorted_hash), _p(dims),
                              _p(cell_start), _p(cell_end), np.float32(hmax), np.float32(K), np.float32(G),
                              _p(owner) if owner is not None else None, int(which),
                              m if idx is not None else 0, _p(idx) if idx is not None else None,
                              _p(drho), _p(L), _p(acc), _p(dsig), C.byref(pc))
    return Rates(drho, L, acc, dsig, int(pc.value))


def integrate(dt, posm, velr, sig, drho, acc, dsig):
    posm = _c(posm, np.float32)
    velr = _c(velr, np.float32)
    sig = _c(sig, np.float32)
    drho = _c(drho, np.float64)
    acc = _c(acc, np.float64)
    dsig = _c(dsig, np.float64)
    n = posm.shape[0]
    po = np.empty((n, 4), np.float64)
    vo = np.empty((n, 4), np.float64)
    so = np.empty((6, n), np.float64)
    _load().orc_integrate(n, float(dt), _p(posm), _p(velr), _p(sig), _p(drho), _p(acc), _p(dsig),
                          _p(po), _p(vo), _p(so))
    return po, vo, so


@dataclass
class StepResult:
    hash: np.ndarray
    sorted_hash: np.ndarray
    perm: np.ndarray
    cell_start: np.ndarray
    cell_end: np.ndarray
    comm_hash: np.ndarray
    boundary_ids: np.ndarray
    owner_counts: np.ndarray
    rates: Rates | None      # indexed by sorted position k (or by idx sample)
    posm: np.ndarray | None  # id order, f64
    velr: np.ndarray | None
    sig: np.ndarray | None


def step(posm, velr, sig, owner, origin, dims, h, K, G, n_owners, dt, floats=True, hp=None) -> StepResult:
    """One iteration from an id-ordered fp32 state.  sig is [6, n].

    floats=False stops after the integer stages (steps a and c and the boundary set).
    hp = per-particle smoothing lengths in id order (None = uniform h); h is then h_max (H1).
    """
    posm = _c(posm, np.float32)
    velr = _c(velr, np.float32)
    sig = _c(sig, np.float32)
    owner = _c(owner, np.int32)
    dims = _c(dims, np.int32)
    n_cells = int(dims[0]) * int(dims[1]) * int(dims[2])
    hsh = hash(posm, origin, dims, h)                                # step a
    sh, perm = sort(hsh)
    cs, ce = cell_ranges(sh, n_cells)
    so_owner = owner[perm]
    ch = comm_hash(sh, so_owner, dims, cs, ce)                       # step c
    bids, ocnt = boundary(ch, perm, so_owner, n_owners)
    if not floats:
        return StepResult(hsh, sh, perm, cs, ce, ch, bids, ocnt, None, None, None, None)
    sp, sv, ss = posm[perm], velr[perm], np.ascontiguousarray(sig[:, perm])
    if hp is None:
        rates = interact(sp, sv, ss, sh, dims, cs, ce, h, K, G)     # steps e, f
    else:
        rates = interact_varh(sp, sv, ss, _c(hp, np.float32)[perm], sh, dims, cs, ce, h, K, G)
    po_s, vo_s, so_s = integrate(dt, sp, sv, ss, rates.drho, rates.acc, rates.dsig)  # step g
    n = posm.shape[0]
    po = np.empty((n, 4)); vo = np.empty((n, 4)); so = np.empty((6, n))
    po[perm] = po_s
    vo[perm] = vo_s
    so[:, perm] = so_s
    return StepResult(hsh, sh, perm, cs, ce, ch, bids, ocnt, rates, po, vo, so)
