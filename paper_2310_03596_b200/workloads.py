"""Seeded synthetic workloads (inputs only -- none of the method's arithmetic lives here).

This module feeds BOTH the CUDA path and the CPU oracle; it imports neither.  It restates the
five `BASELINE.json -> configs` as concrete arrays.  The paper measures
on proprietary IMPETUS models that are not available; these lattices stand in
for them (DESIGN.md section 4 gives the recipe).

Recipe common to all configs: lattice point (i, j, k) * dx with dx = 1 and i, j, k from 0;
particle id = lattice enumeration order, x fastest (this is what the (hash, id) tie-break uses);
jitter independent uniform +-J*dx per component; positions rounded to fp32; h = 1.3;
bucket edge 2h; m = 1; rho = 1; sigma = 0; K = 1; G = 0.5; dt = 1e-3.
Grid (reading S3): origin = (-2h, -2h, -2h) in fp32, dims_a = floor((max lattice coord_a + 0.1 +
4h) / 2h) + 1, so no particle is ever clamped.

Random streams: numpy Generator(PCG64(seed)), drawn in the fixed order jitter -> velocity ->
owners (-> density, stress for T1b); config 3's cylinder centres come from PCG64(seed + 10000).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

H = np.float32(1.3)
DX = 1.0


@dataclass
class Workload:
    name: str
    posm: np.ndarray      # [n,4] f32  x,y,z,m        (id order)
    velr: np.ndarray      # [n,4] f32  vx,vy,vz,rho
    sig: np.ndarray       # [6,n] f32  xx,yy,zz,xy,xz,yz
    owner: np.ndarray     # [n]   i32
    origin: np.ndarray    # [3]   f32
    dims: np.ndarray      # [3]   i32
    h: np.float32 = H
    K: np.float32 = np.float32(1.0)
    G: np.float32 = np.float32(0.5)
    n_owners: int = 1
    dt: float = 1e-3
    steps: int = 1
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.posm.shape[0])

    @property
    def n_cells(self) -> int:
        return int(self.dims[0]) * int(self.dims[1]) * int(self.dims[2])


def grid_for(max_coord, h=H):
    """Reading S3: origin and dims from the largest lattice coordinate per axis."""
    h = float(np.float32(h))
    origin = np.full(3, np.float32(-2.0) * np.float32(h), np.float32)
    dims = np.array([int(np.floor((float(m) + 0.1 + 4.0 * h) / (2.0 * h))) + 1 for m in max_coord],
                    np.int32)
    return origin, dims


def _lattice_coords(nx, ny, nz):
    """Integer lattice coordinates in id order (x fastest), as three int32 arrays."""
    n = nx * ny * nz
    ids = np.arange(n, dtype=np.int64)
    ix = (ids % nx).astype(np.int32)
    iy = ((ids // nx) % ny).astype(np.int32)
    iz = (ids // (nx * ny)).astype(np.int32)
    return ix, iy, iz


def _jittered(rng, ix, iy, iz, jitter):
    n = ix.shape[0]
    posm = np.empty((n, 4), np.float32)
    u = rng.random((n, 3), dtype=np.float32)
    u *= np.float32(2.0 * jitter)
    u -= np.float32(jitter)
    posm[:, 0] = ix.astype(np.float32) + u[:, 0]
    posm[:, 1] = iy.astype(np.float32) + u[:, 1]
    posm[:, 2] = iz.astype(np.float32) + u[:, 2]
    posm[:, 3] = 1.0
    return posm


def _blank_state(n):
    velr = np.zeros((n, 4), np.float32)
    velr[:, 3] = 1.0
    sig = np.zeros((6, n), np.float32)
    return velr, sig


def _equal_count_slabs(x, n_slabs):
    """owner = floor(n_slabs * rank / n), rank in (x, id) order (stable argsort on x)."""
    n = x.shape[0]
    order = np.argsort(x, kind="stable")
    owner = np.empty(n, np.int32)
    owner[order] = (np.arange(n, dtype=np.int64) * n_slabs // n).astype(np.int32)
    return owner


def _rcb(posm, levels):
    """Recursive coordinate bisection on particle count: split along the longest bounding-box
    axis (ties -> lowest axis) at rank floor(n/2) in (coord, id) order."""
    n = posm.shape[0]
    owner = np.zeros(n, np.int32)
    groups = [np.arange(n, dtype=np.int64)]
    for _ in range(levels):
        nxt = []
        for g in groups:
            if g.size == 0:
                nxt += [g, g]
                continue
            p = posm[g, :3]
            ext = p.max(axis=0) - p.min(axis=0)
            ax = int(np.argmax(ext))            # first maximum -> lowest axis on ties
            order = np.argsort(p[:, ax], kind="stable")
            half = g.size // 2
            nxt += [np.sort(g[order[:half]]), np.sort(g[order[half:]])]
        groups = nxt
    for o, g in enumerate(groups):
        owner[g] = o
    return owner


def lattice_block(nx, ny, nz, jitter, seed, name="block", velocity=None, owners=("single",),
                  dt=1e-3, steps=1):
    """Generic jittered block used by the configs and by scaled-down test cases.

    velocity: None | ("sin_y", amp, period) | ("grad_z", slope) | ("normal", std)
    owners:   ("single",) | ("plane_x", x0) | ("slabs", g) | ("slabs_mixed", g, prob) |
              ("random", g) | ("rcb", levels)
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    ix, iy, iz = _lattice_coords(nx, ny, nz)
    posm = _jittered(rng, ix, iy, iz, jitter)
    n = posm.shape[0]
    velr, sig = _blank_state(n)
    if velocity is not None:
        kind = velocity[0]
        if kind == "sin_y":
            _, amp, period = velocity
            velr[:, 0] = (amp * np.sin(2.0 * np.pi * posm[:, 1].astype(np.float64) / period)
                          ).astype(np.float32)
        elif kind == "grad_z":
            velr[:, 2] = (velocity[1] * posm[:, 2].astype(np.float64)).astype(np.float32)
        elif kind == "normal":
            velr[:, :3] = rng.standard_normal((n, 3), dtype=np.float32) * np.float32(velocity[1])
        else:
            raise ValueError(kind)
    kind = owners[0]
    if kind == "single":
        owner, g = np.zeros(n, np.int32), 1
    elif kind == "plane_x":
        owner, g = np.where(posm[:, 0] < np.float32(owners[1]), 0, 1).astype(np.int32), 2
    elif kind == "slabs":
        g = owners[1]
        owner = _equal_count_slabs(posm[:, 0], g)
    elif kind == "slabs_mixed":
        g, prob = owners[1], owners[2]
        owner = _equal_count_slabs(posm[:, 0], g)
        move = rng.random(n) < prob
        shift = rng.integers(0, g - 1, size=n, dtype=np.int32)
        owner = np.where(move, (owner + 1 + shift) % g, owner).astype(np.int32)
    elif kind == "random":
        g = owners[1]
        owner = rng.integers(0, g, size=n, dtype=np.int32)
    elif kind == "rcb":
        g = 1 << owners[1]
        owner = _rcb(posm, owners[1])
    else:
        raise ValueError(kind)
    origin, dims = grid_for((nx - 1, ny - 1, nz - 1))
    return Workload(name, posm, velr, sig, owner, origin, dims, n_owners=g, dt=dt, steps=steps,
                    meta={"lattice": (nx, ny, nz), "jitter": jitter, "seed": seed})


def t1b(side=16, seed=1100):
    """Supplementary tiny case: config-0 geometry with every float path
    non-trivial: v ~ N(0, 0.05), rho = 1 + U(+-0.01), sigma = symmetric N(0, 1e-3)."""
    w = lattice_block(side, side, side, 0.05, seed, name="T1b", velocity=("normal", 0.05),
                      owners=("plane_x", side / 2.0))
    rng = np.random.Generator(np.random.PCG64(seed + 1))
    n = w.n
    w.velr[:, 3] = (1.0 + (rng.random(n) * 2.0 - 1.0) * 0.01).astype(np.float32)
    w.sig[:] = (rng.standard_normal((6, n)) * 1e-3).astype(np.float32)
    return w


def particle_h(w: Workload, kind=("species", 2, 0.75), seed=2000) -> np.ndarray:
    """Per-particle smoothing lengths in id order for the non-uniform-h cases (SURVEY.md 8(f)
    NEXT-4; "h the maximum smoothing length of the particles", PAPER.md:54 particle
    types "with different smoothing lengths").  The grid of `w` stays built on w.h = h_max.
    kind: ("species", k, fmin)  particle type = seeded uniform in 0..k-1, h = h_max (1 - (1 - fmin) type / (k - 1))
          ("checker", f)        h_max on even lattice sites (id parity along x, y, z), f h_max on odd ones
          ("uniform",)          every particle h_max
          ("random", fmin)      h_max U(fmin, 1)"""
    n, hmax = w.n, np.float32(w.h)
    rng = np.random.Generator(np.random.PCG64(seed))
    if kind[0] == "uniform":
        return np.full(n, hmax, np.float32)
    if kind[0] == "species":
        k, fmin = int(kind[1]), float(kind[2])
        typ = rng.integers(0, k, n)
        return (hmax * (1.0 - (1.0 - fmin) * typ / max(k - 1, 1))).astype(np.float32)
    if kind[0] == "checker":
        site = np.rint(w.posm[:, :3]).astype(np.int64)
        odd = (site.sum(1) & 1).astype(bool)
        return np.where(odd, np.float32(kind[1]) * hmax, hmax).astype(np.float32)
    if kind[0] == "random":
        return (hmax * rng.uniform(float(kind[1]), 1.0, n)).astype(np.float32)
    raise ValueError(kind)


def _config3(seed, scale=1.0):
    """Plate [0,400)x[0,400)x[0,100) U 8 cylinders (axis z, radius 40, z in [100,250)), centres
    uniform in [40,360]^2 rejecting overlaps.  `scale` shrinks every length (tests)."""
    L = int(round(400 * scale)); T = int(round(100 * scale)); R = 40.0 * scale
    Hc = int(round(150 * scale))
    grng = np.random.Generator(np.random.PCG64(seed + 10000))
    centres = []
    while len(centres) < 8:
        c = grng.uniform(R, L - R, size=2)
        if all(np.hypot(*(c - d)) >= 2 * R for d in centres):
            centres.append(c)
    nzl = T + Hc
    # lattice sites in id order (x fastest), clipped
    ixs, iys, izs = [], [], []
    xs = np.arange(L, dtype=np.int32)
    X, Y = np.meshgrid(xs, xs, indexing="xy")          # X varies fastest along axis 1
    cyl = np.zeros((L, L), bool)
    for c in centres:
        cyl |= (X - c[0]) ** 2 + (Y - c[1]) ** 2 < R * R
    for z in range(nzl):
        m = np.ones((L, L), bool) if z < T else cyl
        yy, xx = np.nonzero(m)                           # row-major: y slow, x fast
        ixs.append(xx.astype(np.int32)); iys.append(yy.astype(np.int32))
        izs.append(np.full(xx.shape[0], z, np.int32))
    ix, iy, iz = np.concatenate(ixs), np.concatenate(iys), np.concatenate(izs)
    rng = np.random.Generator(np.random.PCG64(seed))
    posm = _jittered(rng, ix, iy, iz, 0.1)
    n = posm.shape[0]
    velr, sig = _blank_state(n)
    velr[:, :3] = rng.standard_normal((n, 3), dtype=np.float32) * np.float32(0.01)
    owner = _rcb(posm, 4)
    origin, dims = grid_for((L - 1, L - 1, nzl - 1))
    return Workload("cfg3", posm, velr, sig, owner, origin, dims, n_owners=16, steps=10,
                    meta={"centres": [tuple(map(float, c)) for c in centres], "seed": seed,
                          "scale": scale})


def config(k: int, side: int | None = None, scale: float | None = None) -> Workload:
    """BASELINE.json configs[k].  `side` (configs 0,1,2,4) / `scale` (config 3) give the same
    recipe on a smaller lattice for tests."""
    if k == 0:
        s = side or 16
        w = lattice_block(s, s, s, 0.05, 1000, "cfg0", None, ("plane_x", s / 2.0), steps=1)
    elif k == 1:
        s = side or 100
        w = lattice_block(s, s, s, 0.1, 1001, "cfg1", ("sin_y", 0.01, float(s)), ("slabs", 4),
                          steps=10)
    elif k == 2:
        s = side or 200
        w = lattice_block(s, s, s, 0.1, 1002, "cfg2", ("grad_z", -0.001), ("slabs_mixed", 16, 0.1),
                          steps=10)
    elif k == 3:
        w = _config3(1003, scale or 1.0)
    elif k == 4:
        s = side or 400
        w = lattice_block(s, s, s, 0.1, 1004, "cfg4", ("normal", 0.05), ("random", 16), steps=20)
    else:
        raise ValueError(k)
    w.meta["config"] = k
    return w
