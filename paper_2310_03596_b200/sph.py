"""Thin Python binding of the C-ABI in include/sph.h (libsph_b200.so).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  PyTorch
provides device memory and the stream, nothing else.  There is NO CPU fallback: importing this
module without the built library, or calling it without a CUDA device, raises.

The functions carry the C names (sph_hash, sph_sort, sph_reorder, sph_cell_ranges, sph_comm_hash,
sph_interact, sph_integrate, sph_step, sph_step_host); `Context` owns the sph_ctx handle.
All hashes / indices are uint32 on the device and are held in torch.int32 tensors (same bits);
`as_u32` gives the numpy uint32 view of a downloaded tensor.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsph_b200.so")

SPH_OK, SPH_EINVAL, SPH_ECUDA, SPH_ENOMEM, SPH_ELIMIT = 0, -1, -2, -3, -4
NOALLOC_MAX_CELLS = 1 << 22   # buckets the built-in scratch of sph_comm_hash_noalloc holds
GARBAGE_HASH = 0xFFFFFFFF
MAX_OWNERS = 32
FLAG_INTERACT_DIRECT = 1
TIMING_SLOTS = 32          # steps held by the library's ring of stage events (sph_get_timing)

EXPORTS = (
    "sph_create", "sph_destroy", "sph_hash", "sph_sort", "sph_reorder", "sph_cell_ranges",
    "sph_comm_hash", "sph_interact", "sph_integrate", "sph_step", "sph_step_host", "sph_pack_boundary",
    "sph_interact_split", "sph_interact_varh", "sph_step_varh", "sph_interact_ef", "sph_balance", "sph_balance_types", "sph_enable_timing", "sph_get_timing", "sph_launch_count", "sph_strerror",
    "sph_last_cuda_error", "sph_comm_hash_noalloc", "sph_pack_destinations",
)


class SphError(RuntimeError):
    pass


class _Params(C.Structure):
    _fields_ = [("origin", C.c_float * 3), ("dims", C.c_int32 * 3), ("h", C.c_float),
                ("K", C.c_float), ("G", C.c_float), ("n_owners", C.c_int32), ("flags", C.c_uint32)]


class _State(C.Structure):
    _fields_ = [("posm", C.c_void_p), ("velr", C.c_void_p), ("sig", C.c_void_p * 6),
                ("owner", C.c_void_p)]


_lib = None


def load_library() -> C.CDLL:
    """dlopen the in-tree library; raise if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise SphError(f"{LIB_PATH} is missing: run `python -m paper_2310_03596_b200.build` "
                       "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i64, i32, f32 = C.c_void_p, C.c_int64, C.c_int32, C.c_float
    sp = C.POINTER(_State)
    lib.sph_create.argtypes = [C.POINTER(vp), C.POINTER(_Params), i64, vp]
    lib.sph_destroy.argtypes = [vp]
    lib.sph_hash.argtypes = [vp, i64, vp, vp]
    lib.sph_sort.argtypes = [vp, i64, vp, vp, vp]
    lib.sph_reorder.argtypes = [vp, i64, vp, sp, sp]
    lib.sph_cell_ranges.argtypes = [vp, i64, vp, vp, vp]
    lib.sph_comm_hash.argtypes = [vp, i64] + [vp] * 9
    lib.sph_comm_hash_noalloc.argtypes = [C.POINTER(_Params), i64, vp, vp, vp, vp, vp]
    lib.sph_interact.argtypes = [vp, i64, sp, vp, vp, vp, vp, vp, C.POINTER(vp * 6), vp]
    lib.sph_interact_split.argtypes = [vp, i64, sp, vp, vp, vp, i32, vp, vp, C.POINTER(vp * 6), vp]
    lib.sph_interact_varh.argtypes = [vp, i64, sp, vp, vp, vp, vp, i32, vp, vp, C.POINTER(vp * 6), vp]
    lib.sph_step_varh.argtypes = [vp, i64, f32, sp, vp] + [vp] * 11 + [C.POINTER(vp * 6), vp]
    lib.sph_interact_ef.argtypes = [vp, i64, sp, vp, vp, vp, vp, vp, vp, C.POINTER(vp * 6), vp, vp,
                                    C.POINTER(vp * 6), vp]
    lib.sph_integrate.argtypes = [vp, i64, f32, sp, vp, vp, C.POINTER(vp * 6), sp]
    lib.sph_step.argtypes = [vp, i64, f32, sp] + [vp] * 11 + [C.POINTER(vp * 6), vp]
    lib.sph_step_host.argtypes = [vp, i64, f32, i32, sp, vp, vp, vp]
    lib.sph_balance.argtypes = [vp, i64, vp, vp, i32, vp, vp]
    lib.sph_balance_types.argtypes = [vp, i64, vp, vp, vp, i32, C.c_double, i32, vp, vp]
    lib.sph_pack_boundary.argtypes = [vp, i64, i64, sp, vp, vp, vp, sp]
    lib.sph_pack_destinations.argtypes = [vp, i64, vp, vp, vp, vp, vp, i64]
    lib.sph_enable_timing.argtypes = [vp, i32]
    lib.sph_get_timing.argtypes = [vp, C.POINTER(f32 * 8)]
    lib.sph_launch_count.argtypes = [vp]
    lib.sph_launch_count.restype = i64
    lib.sph_strerror.argtypes = [C.c_int]
    lib.sph_strerror.restype = C.c_char_p
    lib.sph_last_cuda_error.argtypes = [vp]
    lib.sph_last_cuda_error.restype = C.c_char_p
    _lib = lib
    return lib


def as_u32(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().numpy().view(np.uint32)


@dataclass
class State:
    """SoA particle state on the device: posm [n,4] f32, velr [n,4] f32, sig [6,n] f32, owner [n] i32."""
    posm: torch.Tensor
    velr: torch.Tensor
    sig: torch.Tensor
    owner: torch.Tensor

    @property
    def n(self) -> int:
        return int(self.posm.shape[0])

    @staticmethod
    def empty(n: int, device="cuda") -> "State":
        return State(torch.empty((n, 4), dtype=torch.float32, device=device),
                     torch.empty((n, 4), dtype=torch.float32, device=device),
                     torch.empty((6, n), dtype=torch.float32, device=device),
                     torch.empty((n,), dtype=torch.int32, device=device))

    @staticmethod
    def from_numpy(posm, velr, sig, owner, device="cuda", pin=False) -> "State":
        def mk(a, dt):
            t = torch.from_numpy(np.ascontiguousarray(a, dtype=dt))
            if device == "cpu":
                return t.pin_memory() if pin else t
            return t.to(device)
        return State(mk(posm, np.float32), mk(velr, np.float32), mk(sig, np.float32),
                     mk(owner, np.int32))

    def clone(self) -> "State":
        return State(self.posm.clone(), self.velr.clone(), self.sig.clone(), self.owner.clone())

    def _check(self, want_cuda=True):
        n = self.n
        for t, shape, dt in ((self.posm, (n, 4), torch.float32), (self.velr, (n, 4), torch.float32),
                             (self.sig, (6, n), torch.float32), (self.owner, (n,), torch.int32)):
            if tuple(t.shape) != shape or t.dtype != dt or not t.is_contiguous():
                raise SphError(f"bad state tensor: shape {tuple(t.shape)} dtype {t.dtype}")
            if t.is_cuda != want_cuda:
                raise SphError("state tensor on the wrong device")

    def _c(self, want_cuda=True) -> _State:
        self._check(want_cuda)
        s = _State()
        s.posm = self.posm.data_ptr()
        s.velr = self.velr.data_ptr()
        n = self.n
        for i in range(6):
            s.sig[i] = self.sig.data_ptr() + 4 * n * i
        s.owner = self.owner.data_ptr()
        return s


@dataclass
class StepOutputs:
    """Per-stage products of one sph_step (all device tensors; rates indexed by sorted position)."""
    hash: torch.Tensor
    sorted_hash: torch.Tensor
    perm: torch.Tensor
    cell_start: torch.Tensor
    cell_end: torch.Tensor
    comm_hash: torch.Tensor
    boundary_ids: torch.Tensor      # capacity n; first boundary_count entries are valid
    boundary_count: torch.Tensor    # [1]
    owner_counts: torch.Tensor      # [n_owners]
    drho: torch.Tensor              # [n]
    acc: torch.Tensor               # [n,4], w = 0
    dsig: torch.Tensor              # [6,n]
    pair_count: torch.Tensor        # [1] int64


def _ptr(t):
    return None if t is None else t.data_ptr()


def _six(t: torch.Tensor):
    n = t.shape[1]
    arr = (C.c_void_p * 6)()
    for i in range(6):
        arr[i] = t.data_ptr() + 4 * n * i
    return arr


class Context:
    """Owns one sph_ctx (scratch for max_n particles on the given grid) on torch's current stream."""

    def __init__(self, origin, dims, h, K=1.0, G=0.5, n_owners=1, max_n=0, flags=0, stream=None,
                 device="cuda:0"):
        if not torch.cuda.is_available():
            raise SphError("no CUDA device: the SPH path has no CPU fallback")
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        p = _Params()
        for a in range(3):
            p.origin[a] = float(origin[a])
            p.dims[a] = int(dims[a])
        p.h, p.K, p.G = float(h), float(K), float(G)
        p.n_owners, p.flags = int(n_owners), int(flags)
        self.params = p
        self.dims = tuple(int(d) for d in dims)
        self.n_cells = self.dims[0] * self.dims[1] * self.dims[2]
        self.n_owners = int(n_owners)
        self.max_n = int(max_n)
        h_ = C.c_void_p()
        rc = self.lib.sph_create(C.byref(h_), C.byref(p), self.max_n, C.c_void_p(self.stream.cuda_stream))
        if rc != SPH_OK:
            raise SphError(f"sph_create: {self.lib.sph_strerror(rc).decode()}")
        self.handle = h_

    @staticmethod
    def for_workload(w, flags=0, max_n=None, **kw) -> "Context":
        return Context(w.origin, w.dims, w.h, w.K, w.G, w.n_owners, max_n if max_n is not None else w.n,
                       flags=flags, **kw)

    def close(self):
        if getattr(self, "handle", None):
            self.lib.sph_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ------------------------------------------------------------------ helpers
    def _chk(self, rc, what):
        if rc != SPH_OK:
            msg = self.lib.sph_strerror(rc).decode()
            if rc == SPH_ECUDA:
                msg += ": " + self.lib.sph_last_cuda_error(self.handle).decode()
            raise SphError(f"{what}: {msg}")

    def _i32(self, *shape):
        return torch.empty(shape, dtype=torch.int32, device=self.device)

    def _f32(self, *shape):
        return torch.empty(shape, dtype=torch.float32, device=self.device)

    def launch_count(self) -> int:
        return int(self.lib.sph_launch_count(self.handle))

    def enable_timing(self, on=True):
        self._chk(self.lib.sph_enable_timing(self.handle, 1 if on else 0), "sph_enable_timing")

    def get_timing(self) -> dict:
        ms = (C.c_float * 8)()
        self._chk(self.lib.sph_get_timing(self.handle, C.byref(ms)), "sph_get_timing")
        names = ("hash", "sort", "reorder", "cell_ranges", "comm_hash", "interact", "integrate", "total")
        return {k: float(ms[i]) for i, k in enumerate(names)}

    # ------------------------------------------------------------------ stages (C names)
    def sph_hash(self, posm: torch.Tensor, out=None) -> torch.Tensor:
        n = posm.shape[0]
        out = out if out is not None else self._i32(n)
        self._chk(self.lib.sph_hash(self.handle, n, posm.data_ptr(), out.data_ptr()), "sph_hash")
        return out

    def sph_sort(self, hash_: torch.Tensor):
        n = hash_.shape[0]
        sh, perm = self._i32(n), self._i32(n)
        self._chk(self.lib.sph_sort(self.handle, n, hash_.data_ptr(), sh.data_ptr(), perm.data_ptr()),
                  "sph_sort")
        return sh, perm

    def sph_reorder(self, perm: torch.Tensor, state: State, out: State | None = None) -> State:
        n = state.n
        out = out if out is not None else State.empty(n, self.device)
        a, b = state._c(), out._c()
        self._chk(self.lib.sph_reorder(self.handle, n, perm.data_ptr(), C.byref(a), C.byref(b)),
                  "sph_reorder")
        return out

    def sph_cell_ranges(self, sorted_hash: torch.Tensor):
        cs, ce = self._i32(self.n_cells), self._i32(self.n_cells)
        self._chk(self.lib.sph_cell_ranges(self.handle, sorted_hash.shape[0], sorted_hash.data_ptr(),
                                           cs.data_ptr(), ce.data_ptr()), "sph_cell_ranges")
        return cs, ce

    def sph_comm_hash(self, sorted_hash, sorted_owner, perm, cell_start, cell_end):
        n = sorted_hash.shape[0]
        ch, bids = self._i32(n), self._i32(max(n, 1))
        cnt, oc = self._i32(1), self._i32(self.n_owners)
        self._chk(self.lib.sph_comm_hash(self.handle, n, sorted_hash.data_ptr(), sorted_owner.data_ptr(),
                                         perm.data_ptr(), cell_start.data_ptr(), cell_end.data_ptr(),
                                         ch.data_ptr(), bids.data_ptr(), cnt.data_ptr(), oc.data_ptr()),
                  "sph_comm_hash")
        return ch, bids, cnt, oc

    def sph_interact(self, sorted_state: State, sorted_hash, cell_start, cell_end):
        n = sorted_state.n
        drho, acc, dsig = self._f32(n), self._f32(n, 4), self._f32(6, n)
        pc = torch.zeros(1, dtype=torch.int64, device=self.device)
        s = sorted_state._c()
        d6 = _six(dsig)
        self._chk(self.lib.sph_interact(self.handle, n, C.byref(s), sorted_hash.data_ptr(),
                                        cell_start.data_ptr(), cell_end.data_ptr(), drho.data_ptr(),
                                        acc.data_ptr(), C.byref(d6), pc.data_ptr()), "sph_interact")
        return drho, acc, dsig, pc

    def sph_interact_split(self, sorted_state: State, sorted_hash, cell_start, cell_end, which: int):
        """Step e alone (which = 1, same-owner neighbours) or step f alone (which = 2)."""
        n = sorted_state.n
        drho, acc, dsig = self._f32(n), self._f32(n, 4), self._f32(6, n)
        pc = torch.zeros(1, dtype=torch.int64, device=self.device)
        s = sorted_state._c()
        d6 = _six(dsig)
        self._chk(self.lib.sph_interact_split(self.handle, n, C.byref(s), sorted_hash.data_ptr(),
                                              cell_start.data_ptr(), cell_end.data_ptr(), int(which),
                                              drho.data_ptr(), acc.data_ptr(), C.byref(d6), pc.data_ptr()),
                  "sph_interact_split")
        return drho, acc, dsig, pc

    def sph_interact_varh(self, sorted_state: State, sorted_h, sorted_hash, cell_start, cell_end, which: int = 0):
        """Interaction loops with a smoothing length per particle (NEXT-4; sorted_h [n] f32 in sorted
        order); which = 0 all neighbours, 1 / 2 the split passes."""
        n = sorted_state.n
        drho, acc, dsig = self._f32(n), self._f32(n, 4), self._f32(6, n)
        pc = torch.zeros(1, dtype=torch.int64, device=self.device)
        s = sorted_state._c()
        d6 = _six(dsig)
        self._chk(self.lib.sph_interact_varh(self.handle, n, C.byref(s), sorted_h.data_ptr(), sorted_hash.data_ptr(),
                                             cell_start.data_ptr(), cell_end.data_ptr(), int(which),
                                             drho.data_ptr(), acc.data_ptr(), C.byref(d6), pc.data_ptr()),
                  "sph_interact_varh")
        return drho, acc, dsig, pc

    def sph_interact_ef(self, sorted_state: State, sorted_hash, cell_start, cell_end, sorted_h=None):
        """Steps e and f from one neighbour search: returns ((drho, acc, dsig) of
        step e, (drho, acc, dsig) of step f, pair_counts [2] int64)."""
        n = sorted_state.n
        e = (self._f32(n), self._f32(n, 4), self._f32(6, n))
        f = (self._f32(n), self._f32(n, 4), self._f32(6, n))
        pc = torch.zeros(2, dtype=torch.int64, device=self.device)
        s = sorted_state._c()
        de, df = _six(e[2]), _six(f[2])
        self._chk(self.lib.sph_interact_ef(self.handle, n, C.byref(s), _ptr(sorted_h), sorted_hash.data_ptr(),
                                           cell_start.data_ptr(), cell_end.data_ptr(), e[0].data_ptr(),
                                           e[1].data_ptr(), C.byref(de), f[0].data_ptr(), f[1].data_ptr(),
                                           C.byref(df), pc.data_ptr()), "sph_interact_ef")
        return e, f, pc

    def sph_step_varh(self, state: State, h: torch.Tensor, dt, out: StepOutputs | None = None,
                      pair_count: torch.Tensor | None = None):
        """sph_step with a smoothing length per particle (h [n] f32 in id order, NEXT-4)."""
        n = state.n
        s = state._c()
        o = out
        if o is not None:
            d6 = _six(o.dsig)
            rc = self.lib.sph_step_varh(self.handle, n, float(dt), C.byref(s), h.data_ptr(), _ptr(o.hash),
                                        _ptr(o.sorted_hash), _ptr(o.perm), _ptr(o.cell_start),
                                        _ptr(o.cell_end), _ptr(o.comm_hash), _ptr(o.boundary_ids),
                                        _ptr(o.boundary_count), _ptr(o.owner_counts), _ptr(o.drho),
                                        _ptr(o.acc), C.byref(d6), _ptr(o.pair_count))
        else:
            rc = self.lib.sph_step_varh(self.handle, n, float(dt), C.byref(s), h.data_ptr(), *([None] * 11), None,
                                        _ptr(pair_count))
        self._chk(rc, "sph_step_varh")
        return out

    def sph_integrate(self, dt, state: State, drho, acc, dsig, out: State | None = None) -> State:
        n = state.n
        out = out if out is not None else State.empty(n, self.device)
        a, b = state._c(), out._c()
        d6 = _six(dsig)
        self._chk(self.lib.sph_integrate(self.handle, n, float(dt), C.byref(a), drho.data_ptr(),
                                         acc.data_ptr(), C.byref(d6), C.byref(b)), "sph_integrate")
        return out

    def alloc_outputs(self, n: int) -> StepOutputs:
        return StepOutputs(self._i32(n), self._i32(n), self._i32(n), self._i32(self.n_cells),
                           self._i32(self.n_cells), self._i32(n), self._i32(max(n, 1)), self._i32(1),
                           self._i32(self.n_owners), self._f32(n), self._f32(n, 4), self._f32(6, n),
                           torch.zeros(1, dtype=torch.int64, device=self.device))

    def sph_step(self, state: State, dt, out: StepOutputs | None = None,
                 pair_count: torch.Tensor | None = None):
        """One iteration in place on the id-ordered `state`.  With `out` every per-stage product is
        written to caller tensors (parity tests); without it they stay in ctx scratch."""
        n = state.n
        s = state._c()
        o = out
        if o is not None:
            d6 = _six(o.dsig)
            rc = self.lib.sph_step(self.handle, n, float(dt), C.byref(s), _ptr(o.hash),
                                   _ptr(o.sorted_hash), _ptr(o.perm), _ptr(o.cell_start),
                                   _ptr(o.cell_end), _ptr(o.comm_hash), _ptr(o.boundary_ids),
                                   _ptr(o.boundary_count), _ptr(o.owner_counts), _ptr(o.drho),
                                   _ptr(o.acc), C.byref(d6), _ptr(o.pair_count))
        else:
            rc = self.lib.sph_step(self.handle, n, float(dt), C.byref(s), *([None] * 11), None,
                                   _ptr(pair_count))
        self._chk(rc, "sph_step")
        return out

    def sph_balance(self, posm: torch.Tensor, owner: torch.Tensor, hmax: int = 1000, want_hash: bool = True):
        """One balancing sweep over all owner pairs (NEXT-2): `owner` is updated in
        place; returns (bal_hash [n] int32 or None, swapped [1] int64).  The hashes are an optional
        product of the C call (bal_hash = NULL): want_hash=False skips their 4-byte scatter."""
        n = int(posm.shape[0])
        bh = self._i32(max(n, 1)) if want_hash else None
        sw = torch.zeros(1, dtype=torch.int64, device=self.device)
        self._chk(self.lib.sph_balance(self.handle, n, posm.data_ptr(), owner.data_ptr(), int(hmax),
                                       _ptr(bh), sw.data_ptr()), "sph_balance")
        return (bh[:n] if want_hash else None), sw

    def sph_balance_types(self, posm: torch.Tensor, owner: torch.Tensor, ptype: torch.Tensor, n_types: int,
                          alpha: float = 0.1, hmax: int = 1000):
        """Balancing sweep per particle type with the biased Cg' of PAPER.md:56 (NEXT-4)."""
        n = int(posm.shape[0])
        bh = self._i32(max(n, 1))
        sw = torch.zeros(1, dtype=torch.int64, device=self.device)
        self._chk(self.lib.sph_balance_types(self.handle, n, posm.data_ptr(), owner.data_ptr(), ptype.data_ptr(),
                                             int(n_types), float(alpha), int(hmax), bh.data_ptr(), sw.data_ptr()),
                  "sph_balance_types")
        return bh[:n], sw

    def sph_pack_boundary(self, state: State, boundary_ids: torch.Tensor, m: int, out=None):
        """Per-owner send buffers (NEXT-1): returns (owner_offsets [n_owners + 1], packed_ids [m],
        packed State of length m).  m is the host value of boundary_count.  out = (offsets, ids,
        State) of capacity >= m re-uses caller tensors (the State's length is the sig plane stride)."""
        m = int(m)
        if out is not None:
            offs, ids, packed = out
            if offs.numel() < self.n_owners + 1 or ids.numel() < m or packed.n < m:
                raise SphError("sph_pack_boundary: out tensors too small")
        else:
            offs = self._i32(self.n_owners + 1)
            ids = self._i32(max(m, 1))
            packed = State.empty(max(m, 1), self.device)
        a, b = state._c(), packed._c()
        self._chk(self.lib.sph_pack_boundary(self.handle, state.n, m, C.byref(a), boundary_ids.data_ptr(),
                                             offs.data_ptr(), ids.data_ptr(), C.byref(b)), "sph_pack_boundary")
        return offs, ids[:m], State(packed.posm[:m], packed.velr[:m], packed.sig[:, :m], packed.owner[:m])

    def sph_pack_destinations(self, sorted_hash, sorted_owner, perm, dest_ids: torch.Tensor | None = None,
                              dest_offsets: torch.Tensor | None = None):
        """Per-destination send lists (NEXT-1; reading D1).  Without `dest_ids` the call
        is made twice: once for the offsets (the total is read back, a host sync), once to fill a
        buffer of exactly that size.  With `dest_ids` (int32, capacity entries) it only enqueues.
        Returns (dest_offsets [n_owners + 1], dest_ids)."""
        n = int(sorted_hash.shape[0])
        offs = dest_offsets if dest_offsets is not None else self._i32(self.n_owners + 1)
        args = (self.handle, n, _ptr(sorted_hash), _ptr(sorted_owner), _ptr(perm), offs.data_ptr())
        if dest_ids is None:
            self._chk(self.lib.sph_pack_destinations(*args, None, 0), "sph_pack_destinations")
            total = int(as_u32(offs)[-1])
            dest_ids = self._i32(max(total, 1))
            self._chk(self.lib.sph_pack_destinations(*args, dest_ids.data_ptr(), total), "sph_pack_destinations")
            return offs, dest_ids[:total]
        self._chk(self.lib.sph_pack_destinations(*args, dest_ids.data_ptr(), int(dest_ids.numel())),
                  "sph_pack_destinations")
        return offs, dest_ids

    def sph_step_host(self, host_state: State, dt, steps=1, boundary_ids: np.ndarray | None = None):
        """End to end with HOST buffers (pinned recommended): H2D, `steps` iterations, D2H, sync.
        Returns (boundary_count, pair_count) as Python ints; host_state is updated in place."""
        n = host_state.n
        s = host_state._c(want_cuda=False)
        cnt = C.c_uint32(0)
        pc = C.c_ulonglong(0)
        bptr = boundary_ids.ctypes.data_as(C.c_void_p) if boundary_ids is not None else None
        self._chk(self.lib.sph_step_host(self.handle, n, float(dt), int(steps), C.byref(s), bptr,
                                         C.cast(C.byref(cnt), C.c_void_p),
                                         C.cast(C.byref(pc), C.c_void_p)), "sph_step_host")
        return int(cnt.value), int(pc.value)


def sph_comm_hash_noalloc(dims, n_owners, sorted_hash: torch.Tensor, sorted_owner: torch.Tensor,
                          comm_hash: torch.Tensor | None = None, boundary_count: torch.Tensor | None = None,
                          stream=None):
    """Communication hash for callers that may not allocate device memory (no Context, hence no
    cudaMalloc: think of a solver whose own pool already owns the whole GPU, or a time loop in
    which allocations are forbidden).  The C call uses a 16 MiB scratch array built into the
    library instead; grids with more than NOALLOC_MAX_CELLS buckets raise (SPH_ELIMIT), calls that
    overlap on one GPU race on that array, and the first call per device should come before any
    stream capture.  Pass `comm_hash` [n] and `boundary_count` [1] (int32, on the tensors' device)
    to keep this wrapper from allocating as well; they are created with torch otherwise.
    Returns (comm_hash, boundary_count), valid once `stream` (default: torch's current) is synced."""
    lib = load_library()
    if not torch.cuda.is_available():
        raise SphError("no CUDA device: the SPH path has no CPU fallback")
    n = int(sorted_hash.shape[0])
    dev = sorted_hash.device
    p = _Params()
    for a in range(3):
        p.dims[a] = int(dims[a])
    p.n_owners = int(n_owners)
    if comm_hash is None:
        comm_hash = torch.empty(n, dtype=torch.int32, device=dev)
    if boundary_count is None:
        boundary_count = torch.empty(1, dtype=torch.int32, device=dev)
    with torch.cuda.device(dev):
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        rc = lib.sph_comm_hash_noalloc(C.byref(p), n, sorted_hash.data_ptr(), sorted_owner.data_ptr(),
                                       comm_hash.data_ptr(), boundary_count.data_ptr(),
                                       C.c_void_p(st.cuda_stream))
    if rc != SPH_OK:
        raise SphError(f"sph_comm_hash_noalloc: {lib.sph_strerror(rc).decode()}")
    return comm_hash, boundary_count


# module-level aliases with the C names (ctx first, like the C-ABI)
def sph_hash(ctx, *a, **k): return ctx.sph_hash(*a, **k)
def sph_sort(ctx, *a, **k): return ctx.sph_sort(*a, **k)
def sph_reorder(ctx, *a, **k): return ctx.sph_reorder(*a, **k)
def sph_cell_ranges(ctx, *a, **k): return ctx.sph_cell_ranges(*a, **k)
def sph_comm_hash(ctx, *a, **k): return ctx.sph_comm_hash(*a, **k)
def sph_interact(ctx, *a, **k): return ctx.sph_interact(*a, **k)
def sph_interact_split(ctx, *a, **k): return ctx.sph_interact_split(*a, **k)
def sph_interact_varh(ctx, *a, **k): return ctx.sph_interact_varh(*a, **k)
def sph_interact_ef(ctx, *a, **k): return ctx.sph_interact_ef(*a, **k)
def sph_step_varh(ctx, *a, **k): return ctx.sph_step_varh(*a, **k)
def sph_integrate(ctx, *a, **k): return ctx.sph_integrate(*a, **k)
def sph_step(ctx, *a, **k): return ctx.sph_step(*a, **k)
def sph_step_host(ctx, *a, **k): return ctx.sph_step_host(*a, **k)
def sph_pack_boundary(ctx, *a, **k): return ctx.sph_pack_boundary(*a, **k)
def sph_balance(ctx, *a, **k): return ctx.sph_balance(*a, **k)
def sph_balance_types(ctx, *a, **k): return ctx.sph_balance_types(*a, **k)
def sph_pack_destinations(ctx, *a, **k): return ctx.sph_pack_destinations(*a, **k)
