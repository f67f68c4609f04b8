"""Pins for the CPU oracle (oracle/sph_oracle.c) -- everything here runs without a GPU.

The oracle is pinned to things other than itself: brute-force O(N^2) enumeration written with
dense numpy (no buckets), library routines (numpy.lexsort / searchsorted, scipy quad / expm),
closed forms and invariants (I0-I10), and the lattice constants in
tests/golden/lattice_closed_forms.txt.
"""
import os

import numpy as np
import pytest
from scipy.integrate import quad
from scipy.linalg import expm

import oracle as orc
from paper_2310_03596_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
H = float(np.float32(1.3))


# ----------------------------------------------------------------------------- helpers
def bucket_coords_f32(posm, origin, dims, h):
    """numpy-float32 emulation of the pinned fp32 sequence (reading S2)."""
    edge = np.float32(2.0) * np.float32(h)
    inv = np.float32(1.0) / edge
    t = posm[:, :3].astype(np.float32) - origin.astype(np.float32)[None, :]
    u = (t * inv).astype(np.float32)
    f = np.floor(u)
    f = np.clip(f, 0, (dims - 1)[None, :].astype(np.float32))
    return f.astype(np.int64)


def sym6_to_mat(s6):
    xx, yy, zz, xy, xz, yz = s6
    return np.array([[xx, xy, xz], [xy, yy, yz], [xz, yz, zz]])


def brute_force_rates(posm, velr, sig, h, K, G):
    """Dense O(N^2) evaluation; neighbours by distance only (I0)."""
    x = posm[:, :3].astype(np.float64); m = posm[:, 3].astype(np.float64)
    v = velr[:, :3].astype(np.float64); rho = velr[:, 3].astype(np.float64)
    n = x.shape[0]
    S = np.zeros((n, 3, 3))
    for k, (a, b) in enumerate([(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]):
        S[:, a, b] = sig[k]; S[:, b, a] = sig[k]
    xij = x[:, None, :] - x[None, :, :]
    r = np.sqrt((xij ** 2).sum(-1))
    nb = (r < 2 * h) & ~np.eye(n, dtype=bool)
    alpha = 21.0 / (16.0 * np.pi * h ** 3)
    # dW/dr from the closed form of W, differentiated by hand independently of orc_kernel_F:
    # W = alpha (1-q/2)^4 (1+2q)  =>  dW/dq = -5 alpha q (1-q/2)^3
    q = r / h
    dWdr = np.where(nb, -5.0 * alpha * q * (1 - q / 2) ** 3 / h, 0.0)
    with np.errstate(invalid="ignore", divide="ignore"):
        e = np.where(r[..., None] > 0, xij / r[..., None], 0.0)
    gW = dWdr[..., None] * e                      # grad_i W_ij
    vij = v[:, None, :] - v[None, :, :]
    drho = (m[None, :] * (vij * gW).sum(-1)).sum(1)
    L = np.einsum("j,ija,ijb->iab", m / rho, -vij, gW) if False else \
        np.einsum("ij,ija,ijb->iab", np.broadcast_to((m / rho)[None, :], (n, n)), -vij, gW)
    Sr = S / (rho ** 2)[:, None, None]
    acc = np.einsum("j,ijab,ijb->ia", m, Sr[:, None] + Sr[None, :], gW)
    D = 0.5 * (L + L.transpose(0, 2, 1)); Om = 0.5 * (L - L.transpose(0, 2, 1))
    trD = np.trace(D, axis1=1, axis2=2)
    I = np.eye(3)
    sd = K * trD[:, None, None] * I + 2 * G * (D - trD[:, None, None] / 3 * I) + Om @ S - S @ Om
    dsig = np.stack([sd[:, 0, 0], sd[:, 1, 1], sd[:, 2, 2], sd[:, 0, 1], sd[:, 0, 2], sd[:, 1, 2]], 1)
    return drho, L, acc, dsig, int(nb.sum())


def sorted_view(w):
    r = orc.step(w.posm, w.velr, w.sig, w.owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners,
                 w.dt, floats=False)
    p = r.perm
    return r, w.posm[p], w.velr[p], np.ascontiguousarray(w.sig[:, p]), w.owner[p]


def rates_of(w):
    r, sp, sv, ss, so = sorted_view(w)
    return r, orc.interact(sp, sv, ss, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G), \
        (sp, sv, ss, so)


def custom_block(spacing, side, h, vel_fn=None, sig_fn=None, rho=1.0):
    """Un-jittered lattice with arbitrary spacing (continuum-limit pins)."""
    g = np.arange(side) * spacing
    X, Y, Z = np.meshgrid(g, g, g, indexing="ij")
    x = np.stack([X.ravel(), Y.ravel(), Z.ravel()], 1)
    n = x.shape[0]
    posm = np.empty((n, 4), np.float32); posm[:, :3] = x; posm[:, 3] = rho * spacing ** 3
    velr = np.zeros((n, 4), np.float32); velr[:, 3] = rho
    if vel_fn is not None:
        velr[:, :3] = vel_fn(x)
    sig = np.zeros((6, n), np.float32)
    if sig_fn is not None:
        sig[:] = sig_fn(x)
    origin, dims = W.grid_for((g[-1],) * 3, h)
    return W.Workload("custom", posm, velr, sig, np.zeros(n, np.int32), origin, dims,
                      h=np.float32(h))


def interior_index(w, sp):
    c = sp[:, :3].astype(np.float64)
    centre = 0.5 * (c.max(0) + c.min(0))
    return int(np.argmin(((c - centre) ** 2).sum(1)))


# ----------------------------------------------------------------------------- O1 hash
def test_hash_fp32_sequence_faces_and_clamp():
    origin, dims = W.grid_for((15, 15, 15))
    edge = np.float32(2.0) * np.float32(H)
    pts = []
    for k in range(0, 8):
        face = np.float32(origin[0] + np.float32(k) * edge)
        for d in (-2, -1, 0, 1, 2):
            x = face
            for _ in range(abs(d)):
                x = np.nextafter(x, np.float32(np.inf if d > 0 else -np.inf), dtype=np.float32)
            pts.append([x, 0.0, 0.0, 1.0])
    pts += [[-1e6, 3.0, 3.0, 1.0], [1e6, 1e7, -1e9, 1.0], [3e38, -3e38, 0.0, 1.0]]
    posm = np.array(pts, np.float32)
    got = orc.hash(posm, origin, dims, H)
    c = bucket_coords_f32(posm, origin, dims, H)
    exp = c[:, 0] + dims[0] * (c[:, 1] + dims[1] * c[:, 2])
    assert np.array_equal(got, exp.astype(np.uint32))
    # clamping (S3): far outside -> border buckets
    assert got[-3] == 0 + dims[0] * (c[-3, 1] + dims[1] * c[-3, 2]) and c[-3, 0] == 0
    assert tuple(c[-2]) == (dims[0] - 1, dims[1] - 1, 0)
    assert tuple(c[-1]) == (dims[0] - 1, 0, 1)       # z = 0 - (-2.6) = 2.6 -> bucket 0 or 1
    # monotone in x
    xs = np.sort(np.random.default_rng(0).uniform(-5, 25, 2000).astype(np.float32))
    pm = np.zeros((2000, 4), np.float32); pm[:, 0] = xs
    hx = orc.hash(pm, origin, dims, H).astype(np.int64)
    # y = z = 0 -> bucket (cx, 1, 1) since 0 - (-2.6) = 2.6 = one edge (up to rounding)
    assert np.all(np.diff(hx) >= 0)


def test_hash_bijection_bucket_centres():
    """S1: linear, x fastest -- every bucket gets its own hash, decodable."""
    dims = np.array([5, 4, 3], np.int32)
    origin = np.array([-1.0, 2.0, 0.5], np.float32)
    edge = 2 * H
    cz, cy, cx = np.meshgrid(np.arange(3), np.arange(4), np.arange(5), indexing="ij")
    posm = np.zeros((60, 4), np.float32)
    posm[:, 0] = origin[0] + (cx.ravel() + 0.5) * edge
    posm[:, 1] = origin[1] + (cy.ravel() + 0.5) * edge
    posm[:, 2] = origin[2] + (cz.ravel() + 0.5) * edge
    got = orc.hash(posm, origin, dims, H)
    assert np.array_equal(got, np.arange(60, dtype=np.uint32))   # enumeration order = x fastest


# ----------------------------------------------------------------------------- O2 sort
@pytest.mark.parametrize("n,nkeys", [(0, 4), (1, 4), (1000, 7), (50000, 100000), (4096, 1)])
def test_sort_vs_lexsort(n, nkeys):
    rng = np.random.default_rng(n + nkeys)
    h = rng.integers(0, nkeys, n).astype(np.uint32)
    sh, perm = orc.sort(h)
    exp = np.lexsort((np.arange(n), h))
    assert np.array_equal(perm, exp.astype(np.uint32))
    assert np.array_equal(sh, h[exp])


# ----------------------------------------------------------------------------- O3 cell tables
def test_cell_ranges_vs_searchsorted_and_identities():
    rng = np.random.default_rng(3)
    C = 300
    h = np.sort(rng.choice(np.arange(5, 290), 2000)).astype(np.uint32)    # empty head/tail/gaps
    cs, ce = orc.cell_ranges(h, C)
    assert np.array_equal(cs, np.searchsorted(h, np.arange(C), "left"))
    assert np.array_equal(ce, np.searchsorted(h, np.arange(C), "right"))
    assert cs[0] == 0 and ce[-1] == 2000 and np.array_equal(ce[:-1], cs[1:])
    assert int((ce.astype(np.int64) - cs).sum()) == 2000
    cs0, ce0 = orc.cell_ranges(np.zeros(0, np.uint32), 7)
    assert not cs0.any() and not ce0.any()


# ----------------------------------------------------------------------------- O4/O5 comm hash
def brute_comm_flags(posm, owner, origin, dims, h):
    c = bucket_coords_f32(posm, origin, dims, h)
    near = (np.abs(c[:, None, :] - c[None, :, :]) <= 1).all(-1)
    other = owner[:, None] != owner[None, :]
    return (near & other).any(1)


@pytest.mark.parametrize("owners", [("plane_x", 5.0), ("random", 16), ("single",), ("slabs", 3),
                                    ("slabs_mixed", 4, 0.02), ("rcb", 3), ("plane_y", 4.0),
                                    ("plane_z", 5.0)])
def test_comm_hash_and_boundary_bruteforce(owners):
    # rcb / plane_y / plane_z split the labels across y and z: a foreign particle is then found
    # only through the -y / +y / -z / +z reach of the stencil ("the surrounding
    # buckets": all 26), which x-splits and full mixing never exercise
    if owners[0] in ("plane_y", "plane_z"):
        w = W.lattice_block(11, 9, 10, 0.1, 77)
        axis = 1 if owners[0] == "plane_y" else 2
        w.owner = np.where(w.posm[:, axis] < np.float32(owners[1]), 0, 1).astype(np.int32)
        w.n_owners = 2
    else:
        w = W.lattice_block(11, 9, 10, 0.1, 77, owners=owners)
    r, sp, sv, ss, so = sorted_view(w)
    flags = brute_comm_flags(w.posm, w.owner, w.origin, w.dims, w.h)       # id order
    exp_comm = np.where(flags[r.perm], r.sorted_hash, np.uint32(orc.GARBAGE))
    assert np.array_equal(r.comm_hash, exp_comm)
    # I6: head of the sort on comm hash == stable compaction of the (hash,id)-sorted array
    assert np.array_equal(r.boundary_ids, r.perm[flags[r.perm]])
    assert np.array_equal(r.owner_counts, np.bincount(w.owner[r.boundary_ids], minlength=w.n_owners))
    # I5: the flag is a per-bucket property
    for c in np.unique(r.sorted_hash):
        f = r.comm_hash[r.sorted_hash == c] != orc.GARBAGE
        assert f.all() or not f.any()
    # I4 completeness: every pair r<2h with different owners has both ends in the set
    x = w.posm[:, :3].astype(np.float64)
    d2 = ((x[:, None] - x[None]) ** 2).sum(-1)
    pair = (d2 < (2 * H) ** 2) & (w.owner[:, None] != w.owner[None, :])
    inset = np.zeros(w.n, bool); inset[r.boundary_ids] = True
    ii, jj = np.nonzero(pair)
    assert inset[ii].all() and inset[jj].all()
    if owners[0] == "single":
        assert r.boundary_ids.size == 0                   # I10 / S12
    if owners[0] == "random":
        assert r.boundary_ids.size == w.n                 # PAPER.md:30 full mixing


def test_one_foreign_particle_flags_exactly_its_27_buckets():
    """one particle of another GPU in an interior bucket makes boundary particles of
    exactly the particles in that bucket and its 26 surrounding ones -- every direction counts."""
    w = W.lattice_block(14, 13, 12, 0.1, 78)
    c = bucket_coords_f32(w.posm, w.origin, w.dims, w.h)
    inner = np.nonzero((c == np.array([2, 2, 2])).all(1))[0]       # bucket (2,2,2): not at the grid's edge
    assert inner.size > 0 and (np.array(w.dims) >= 5).all()
    w.owner = np.zeros(w.n, np.int32)
    w.owner[inner[0]] = 1
    w.n_owners = 2
    r, *_ = sorted_view(w)
    flagged = np.zeros(w.n, bool)
    flagged[r.perm[r.comm_hash != orc.GARBAGE]] = True
    near = (np.abs(c - c[inner[0]]) <= 1).all(1)
    # the foreign particle's own bucket holds owner-0 particles too, so it is flagged as well
    assert (w.owner[inner] == 0).any()
    assert np.array_equal(flagged, near)
    # all 27 buckets are occupied and flagged, none beyond
    fb = np.unique(c[flagged], axis=0)
    assert fb.shape[0] == 27 and (fb.min(0) == 1).all() and (fb.max(0) == 3).all()
    assert np.array_equal(np.sort(r.boundary_ids), np.nonzero(near)[0].astype(np.uint32))
    assert np.array_equal(flagged, brute_comm_flags(w.posm, w.owner, w.origin, w.dims, w.h))


def test_boundary_slabs_lie_on_surfaces():
    """with slabs the MGPU boundary particles lie 'onto two surfaces'."""
    w = W.lattice_block(40, 8, 8, 0.1, 5, owners=("slabs", 3))
    r, *_ = sorted_view(w)
    xb = w.posm[r.boundary_ids, 0]
    interfaces = np.array([40 / 3 - 0.5, 80 / 3 - 0.5])
    dist = np.abs(xb[:, None] - interfaces[None, :]).min(1)
    assert dist.max() <= 2 * 2 * H + 0.2                   # within two bucket layers
    assert 0 < r.boundary_ids.size < w.n // 2


# ----------------------------------------------------------------------------- O6 kernel
def test_kernel_normalisation_and_gradient():
    for h in (0.7, H, 2.0):
        val, err = quad(lambda r: 4 * np.pi * r * r * orc.kernel_W(r, h), 0, 2 * h, epsabs=1e-13)
        assert abs(val - 1.0) < 1e-10                                       # I1
        assert orc.kernel_W(2 * h, h) == 0.0 and orc.kernel_F(2 * h, h) == 0.0
        assert orc.kernel_W(2.5 * h, h) == 0.0
        for r in np.linspace(0.05 * h, 1.95 * h, 23):
            e = 1e-6 * h
            dW = (orc.kernel_W(r + e, h) - orc.kernel_W(r - e, h)) / (2 * e)
            assert abs(orc.kernel_F(r, h) * r - dW) < 1e-8 * abs(orc.kernel_W(0, h)) / h
        assert orc.kernel_F(0.3 * h, h) < 0                                  # W decreasing
    # alpha(h=1.3) from SURVEY.md I1
    assert abs(orc.kernel_W(0.0, 1.3) - 0.19016009359) < 1e-10


# ----------------------------------------------------------------------------- O7/O8 vs brute force
@pytest.mark.parametrize("make", [lambda: W.t1b(10, 1100), lambda: W.t1b(12, 1101),
                                  lambda: W.config(1, side=12)])
def test_interact_vs_bruteforce(make):
    w = make()
    r, rt, (sp, sv, ss, so) = rates_of(w)
    drho, L, acc, dsig, pairs = brute_force_rates(sp, sv, ss, float(w.h), float(w.K), float(w.G))
    assert rt.pair_count == pairs
    for got, exp in ((rt.drho, drho), (rt.L, L), (rt.acc, acc), (rt.dsig, dsig)):
        scale = max(np.abs(exp).max(), 1e-300)
        assert np.abs(got - exp).max() <= 1e-11 * scale


def test_interact_subset_matches_full():
    w = W.t1b(10, 1102)
    r, rt, (sp, sv, ss, so) = rates_of(w)
    idx = np.array([0, 5, 17, 400, 999], np.int64)
    sub = orc.interact(sp, sv, ss, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G,
                       idx=idx)
    assert np.array_equal(sub.drho, rt.drho[idx]) and np.array_equal(sub.acc, rt.acc[idx])
    assert np.array_equal(sub.dsig, rt.dsig[idx]) and np.array_equal(sub.L, rt.L[idx])


def test_momentum_conservation():
    """I2: symmetric pair forces => sum_i m_i a_i = 0 to rounding."""
    w = W.t1b(12, 1103)
    w.posm[:, 3] = (1.0 + 0.2 * np.random.default_rng(1).random(w.n)).astype(np.float32)
    r, rt, (sp, *_ ) = rates_of(w)
    f = sp[:, 3:4].astype(np.float64) * rt.acc
    assert np.abs(f.sum(0)).max() <= 1e-12 * np.abs(f).sum()
    assert np.abs(f).sum() > 0


def test_uniform_translation_gives_exact_zero():
    """I3: uniform v => Drho == 0 and L == 0 exactly, any geometry (incl. free surfaces)."""
    w = W.t1b(10, 1104)
    w.velr[:, :3] = np.array([0.3, -1.7, 2.2], np.float32)
    r, rt, _ = rates_of(w)
    assert not rt.drho.any() and not rt.L.any()
    assert np.abs(rt.acc).max() > 0          # stress still acts


def test_rest_lattice_all_zero():
    w = W.config(0, side=8)
    r, rt, _ = rates_of(w)
    assert not rt.drho.any() and not rt.acc.any() and not rt.dsig.any()
    assert rt.pair_count > 0


def test_uniform_density_continuity_identity():
    """I7: uniform rho and m  =>  Drho_i = -rho tr(L_i)."""
    w = W.config(4, side=10)
    r, rt, _ = rates_of(w)
    tr = np.trace(rt.L, axis1=1, axis2=2)
    assert np.abs(rt.drho + 1.0 * tr).max() <= 1e-13 * np.abs(rt.drho).max()


def test_lattice_closed_forms_golden():
    """I8 / tests/golden/lattice_closed_forms.txt (unit lattice, h = 1.3, interior particle)."""
    gold = {}
    for line in open(os.path.join(GOLDEN, "lattice_closed_forms.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()[:2]
            gold[k] = float(v)
    A = np.array([[0.0, 0.0, 0.0], [0.0, 0.0, 0.0], [0.0, 0.0, -0.001]])
    w = custom_block(1.0, 9, H, vel_fn=lambda x: x @ A.T)
    r, rt, (sp, *_ ) = rates_of(w)
    i = interior_index(w, sp)
    sub = orc.interact(sp, w.velr[r.perm], np.ascontiguousarray(w.sig[:, r.perm]), r.sorted_hash,
                       w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G, idx=np.array([i]))
    assert sub.pair_count == int(gold["neighbours"])
    # geometry-only count: lattice points with 0 < |p| < 2.6
    g = np.arange(-3, 4)
    P = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    assert int(((P ** 2).sum(1) < 2.6 ** 2).sum()) - 1 == int(gold["neighbours"])
    sumW = sum(orc.kernel_W(float(np.sqrt(p @ p)), 1.3) for p in P)
    assert abs(sumW - gold["sum_W_incl_self"]) < 2e-9
    assert abs(rt.L[i, 2, 2] / A[2, 2] - gold["moment_M"]) < 2e-6      # fp32 positions/velocities
    assert abs(rt.drho[i] / 0.001 - gold["moment_M"]) < 2e-6


# ----------------------------------------------------------------------------- continuum limits
def test_continuum_velocity_gradient_sign_and_index():
    """Dense lattice (h/dx = 2.6): L -> grad v with L[a][b] = dv_a/dx_b, Drho -> -rho div v."""
    A = np.array([[0.010, 0.020, -0.005], [0.000, -0.030, 0.015], [0.025, -0.010, 0.004]])
    rho = 1.7
    w = custom_block(0.5, 23, H, vel_fn=lambda x: x @ A.T, rho=rho)
    r, sp, sv, ss, so = sorted_view(w)
    i = interior_index(w, sp)
    sub = orc.interact(sp, sv, ss, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G,
                       idx=np.array([i]))
    assert np.abs(sub.L[0] - A).max() < 2e-3 * np.abs(A).max()
    assert abs(sub.drho[0] + rho * np.trace(A)) < 2e-3 * rho * np.abs(A).max()


def test_continuum_stress_divergence_sign_and_index():
    """a_a -> (1/rho) d sigma_ab / d x_b for a linear stress field (tension positive)."""
    rng = np.random.default_rng(11)
    B = rng.normal(size=(6, 3)) * 1e-3                  # d sig6 / d x
    s0 = rng.normal(size=6) * 1e-2
    rho = 0.8

    def sig_fn(x):
        return (s0[:, None] + B @ x.T)

    w = custom_block(0.5, 23, H, sig_fn=sig_fn, rho=rho)
    r, sp, sv, ss, so = sorted_view(w)
    i = interior_index(w, sp)
    sub = orc.interact(sp, sv, ss, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G,
                       idx=np.array([i]))
    # div: a_x = d sxx/dx + d sxy/dy + d sxz/dz ; components xx,yy,zz,xy,xz,yz = 0..5
    div = np.array([B[0, 0] + B[3, 1] + B[4, 2], B[3, 0] + B[1, 1] + B[5, 2],
                    B[4, 0] + B[5, 1] + B[2, 2]]) / rho
    assert np.abs(sub.acc[0] - div).max() < 3e-3 * np.abs(div).max()


# ----------------------------------------------------------------------------- O8 textbook cases
def lattice_L_factor():
    A = np.diag([1e-3, 0.0, 0.0])
    w = custom_block(1.0, 9, H, vel_fn=lambda x: x @ A.T)
    r, rt, (sp, *_ ) = rates_of(w)
    return rt.L[interior_index(w, sp), 0, 0] / 1e-3


def stress_rate_for(A, s6, K=1.0, G=0.5):
    w = custom_block(1.0, 9, H, vel_fn=lambda x: x @ A.T,
                     sig_fn=lambda x: np.repeat(np.asarray(s6)[:, None], x.shape[0], 1))
    w.K, w.G = np.float32(K), np.float32(G)
    r, rt, (sp, *_ ) = rates_of(w)
    i = interior_index(w, sp)
    return rt.dsig[i], rt.L[i]


def test_stress_rate_textbook_cases():
    ms = lattice_L_factor()
    eps, gam = 2e-3, 3e-3
    # pure dilation: sigma_dot = K * 3 eps * I  (bulk modulus definition)
    d, L = stress_rate_for(np.eye(3) * eps, np.zeros(6), K=2.0, G=0.7)
    assert np.allclose(d, [3 * 2.0 * eps * ms] * 3 + [0, 0, 0], rtol=2e-6, atol=1e-12)
    # simple shear v_x = gam*y: sigma_xy_dot = G*gam, no normal stress rate without pre-stress
    A = np.zeros((3, 3)); A[0, 1] = gam
    d, L = stress_rate_for(A, np.zeros(6), K=2.0, G=0.7)
    assert np.allclose(d, [0, 0, 0, 0.7 * gam * ms, 0, 0], rtol=2e-6, atol=1e-12)
    # uniaxial strain: sigma_xx_dot = (K + 4G/3) eps ; sigma_yy_dot = (K - 2G/3) eps
    d, L = stress_rate_for(np.diag([eps, 0, 0]), np.zeros(6), K=2.0, G=0.7)
    assert np.allclose(d, [(2.0 + 4 * 0.7 / 3) * eps * ms, (2.0 - 2 * 0.7 / 3) * eps * ms,
                           (2.0 - 2 * 0.7 / 3) * eps * ms, 0, 0, 0], rtol=2e-6, atol=1e-12)


def test_jaumann_rate_is_finite_rotation_derivative():
    """S17: rigid spin of a pre-stressed body: sigma(t) = R sigma R^T, R = expm(Om t)."""
    ms = lattice_L_factor()
    Om = np.array([[0, -2e-3, 1e-3], [2e-3, 0, 3e-3], [-1e-3, -3e-3, 0]])
    s6 = np.array([0.02, -0.01, 0.005, 0.004, -0.003, 0.006])
    d, L = stress_rate_for(Om, s6)
    S = sym6_to_mat(s6)
    t = 1e-3
    Rp, Rm = expm(ms * Om * t), expm(-ms * Om * t)
    fd = (Rp @ S @ Rp.T - Rm @ S @ Rm.T) / (2 * t)
    got = sym6_to_mat(d)
    assert np.abs(got - fd).max() < 2e-5 * np.abs(fd).max()     # inputs are rounded to fp32
    assert abs(np.trace(got)) < 1e-5 * np.abs(got).max()          # tr(sigma) invariant
    assert abs((S * got).sum()) < 1e-5 * np.abs(S).max() * np.abs(got).max()  # sigma:sigma invariant


# ----------------------------------------------------------------------------- misc readings
def test_coincident_particles_no_nan():
    """S15: distinct coincident particles are a pair with grad W = 0."""
    w = W.t1b(6, 1105)
    w.posm[1, :3] = w.posm[0, :3]
    r, rt, _ = rates_of(w)
    for a in (rt.drho, rt.L, rt.acc, rt.dsig):
        assert np.isfinite(a).all()


def test_integrate_symplectic_euler_by_hand():
    n = 3
    posm = np.array([[1, 2, 3, 1.5]] * n, np.float32)
    velr = np.array([[0.1, -0.2, 0.3, 2.0]] * n, np.float32)
    sig = np.arange(18, dtype=np.float32).reshape(6, n) * 0.01
    drho = np.array([0.5, -0.5, 0.0]); acc = np.array([[1.0, 2.0, -3.0]] * n)
    dsig = np.arange(18, dtype=np.float64).reshape(n, 6)
    dt = 0.25
    po, vo, so = orc.integrate(dt, posm, velr, sig, drho, acc, dsig)
    vexp = velr[0, :3].astype(np.float64) + dt * acc[0]
    assert np.allclose(vo[0, :3], vexp, rtol=0, atol=1e-15)
    assert np.allclose(po[0, :3], posm[0, :3].astype(np.float64) + dt * vexp, rtol=0, atol=1e-15)  # uses v+
    assert po[0, 3] == 1.5 and np.allclose(vo[:, 3], 2.0 + dt * drho)
    assert np.allclose(so, sig.astype(np.float64) + dt * dsig.T)
    po0, vo0, so0 = orc.integrate(0.0, posm, velr, sig, drho, acc, dsig)
    assert np.array_equal(po0, posm.astype(np.float64)) and np.array_equal(vo0, velr.astype(np.float64))


def test_step_composite_consistency():
    w = W.t1b(8, 1106)
    r = orc.step(w.posm, w.velr, w.sig, w.owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt)
    assert np.array_equal(np.sort(r.perm), np.arange(w.n))
    assert np.all(np.diff(r.sorted_hash.astype(np.int64)) >= 0)
    same = np.diff(r.sorted_hash.astype(np.int64)) == 0
    assert np.all(np.diff(r.perm.astype(np.int64))[same] > 0)       # ids increase inside a bucket
    # state comes back in id order, mass and owner untouched
    assert np.array_equal(r.posm[:, 3], w.posm[:, 3].astype(np.float64))
    acc_id = np.empty((w.n, 3)); acc_id[r.perm] = r.rates.acc
    assert np.allclose(r.velr[:, :3], w.velr[:, :3].astype(np.float64) + w.dt * acc_id, atol=1e-15)


def test_expected_boundary_fractions():
    """cfg0 ~46.8 %; random labels 100 %; cfg1-like slabs a minority."""
    w = W.config(0)
    r, *_ = sorted_view(w)
    assert abs(r.boundary_ids.size / w.n - 0.468) < 0.02
    w = W.config(4, side=24)
    r, *_ = sorted_view(w)
    assert r.boundary_ids.size == w.n
    w = W.config(2, side=32)
    r, *_ = sorted_view(w)
    assert r.boundary_ids.size == w.n


# ----------------------------------------------------------------------------- NEXT-1: send buffers
@pytest.mark.parametrize("make", [lambda: W.config(0), lambda: W.config(2, side=20),
                                  lambda: W.config(3, scale=0.05)])
def test_pack_boundary_vs_stable_argsort_and_invariants(make):
    """Per-owner send buffers (O5b) against the library statement of the same
    thing -- a STABLE argsort of the boundary list on the owner label -- and the invariants that
    define it: segments partition the boundary set, each is a subsequence of the (hash, id)
    ordered list, sizes equal owner_counts, records are the state at the packed ids."""
    w = make()
    r = orc.step(w.posm, w.velr, w.sig, w.owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt,
                 floats=False)
    pb = orc.pack_boundary(r.boundary_ids, w.owner, w.n_owners, w.posm, w.velr, w.sig)
    ids = r.boundary_ids
    order = np.argsort(w.owner[ids], kind="stable")
    np.testing.assert_array_equal(pb.ids, ids[order])
    np.testing.assert_array_equal(np.diff(pb.offsets.astype(np.int64)), r.owner_counts)
    assert pb.offsets[0] == 0 and pb.offsets[-1] == ids.size
    assert sorted(pb.ids.tolist()) == sorted(ids.tolist())
    pos_in_list = np.empty(w.n, np.int64); pos_in_list[ids] = np.arange(ids.size)
    for g in range(w.n_owners):
        seg = pb.ids[pb.offsets[g]:pb.offsets[g + 1]]
        assert (w.owner[seg] == g).all()
        assert (np.diff(pos_in_list[seg]) > 0).all()        # list order kept inside a segment
    np.testing.assert_array_equal(pb.posm, w.posm[pb.ids])
    np.testing.assert_array_equal(pb.velr, w.velr[pb.ids])
    np.testing.assert_array_equal(pb.sig, w.sig[:, pb.ids])
    np.testing.assert_array_equal(pb.owner, w.owner[pb.ids])


@pytest.mark.parametrize("owners", [("plane_x", 5.0), ("slabs", 3), ("slabs_mixed", 4, 0.02), ("rcb", 3),
                                    ("random", 5), ("single",)])
def test_pack_destinations_dense_checker_and_invariants(owners):
    """O5c (PAPER.md:23 step d, reading D1): the list of destination g against a dense
    bucket-coordinate checker written in numpy, plus what must hold whatever the layout: every list
    in (hash, id) order, no particle sent to its own owner, union of the lists = the MGPU boundary
    set (a particle is a boundary particle iff SOME other owner is in its stencil), never more
    entries than the paper's broadcast-to-all (M (G - 1)), exactly that many under full mixing."""
    w = W.lattice_block(11, 9, 10, 0.1, 79, owners=owners)
    g_n = w.n_owners
    r, sp, sv, ss, so = sorted_view(w)
    off, ids = orc.pack_destinations(r.sorted_hash, so, r.perm, w.dims, r.cell_start, r.cell_end, g_n)
    assert off[0] == 0 and off[-1] == ids.size and (np.diff(off.astype(np.int64)) >= 0).all()
    c = bucket_coords_f32(w.posm, w.origin, w.dims, w.h)                     # id order
    near = (np.abs(c[:, None, :] - c[None, :, :]) <= 1).all(-1)
    rank = np.empty(w.n, np.int64); rank[r.perm] = np.arange(w.n)            # position in (hash, id) order
    for g in range(g_n):
        lst = ids[off[g]:off[g + 1]]
        want = (w.owner != g) & (near & (w.owner[None, :] == g)).any(1)
        np.testing.assert_array_equal(lst, r.perm[want[r.perm]], err_msg=f"destination {g}")
        assert (w.owner[lst] != g).all()
        assert (np.diff(rank[lst]) > 0).all()
    np.testing.assert_array_equal(np.unique(ids), np.sort(r.boundary_ids))
    m = r.boundary_ids.size
    assert ids.size <= m * (g_n - 1)
    if owners[0] == "random":
        assert ids.size == w.n * (g_n - 1)          # PAPER.md:30 full mixing: nothing is saved
    if owners[0] == "single":
        assert ids.size == 0
    if g_n == 2:
        # two owners: what goes to g is exactly the other owner's send segment of O5b
        pk = orc.pack_boundary(r.boundary_ids, w.owner, 2, w.posm, w.velr, w.sig)
        np.testing.assert_array_equal(ids[off[1]:off[2]], pk.ids[pk.offsets[0]:pk.offsets[1]])
        np.testing.assert_array_equal(ids[off[0]:off[1]], pk.ids[pk.offsets[1]:pk.offsets[2]])


def test_pack_destinations_wide_slabs_halve_the_broadcast():
    """Three slabs, each wider than a stencil (PAPER.md:30 'two surfaces'): every boundary particle
    has exactly ONE foreign neighbour owner, so the per-destination lists hold M entries where the
    paper's broadcast to all other GPUs ships 2 M; the outer slabs exchange nothing."""
    w = W.lattice_block(40, 6, 6, 0.1, 80, owners=("slabs", 3))
    r, sp, sv, ss, so = sorted_view(w)
    off, ids = orc.pack_destinations(r.sorted_hash, so, r.perm, w.dims, r.cell_start, r.cell_end, 3)
    m = r.boundary_ids.size
    assert 0 < m < w.n and ids.size == m and np.unique(ids).size == m
    assert (w.owner[ids[off[0]:off[1]]] == 1).all() and (w.owner[ids[off[2]:off[3]]] == 1).all()
    assert set(w.owner[ids[off[1]:off[2]]]) == {0, 2}


def test_pack_destinations_one_foreign_particle():
    """One particle of owner 1 in an interior bucket: destination 1 receives exactly the owner-0
    particles of the 27 buckets around it, destination 0 receives that one particle."""
    w = W.lattice_block(14, 13, 12, 0.1, 78)
    c = bucket_coords_f32(w.posm, w.origin, w.dims, w.h)
    f = np.nonzero((c == np.array([2, 2, 2])).all(1))[0][0]
    w.owner = np.zeros(w.n, np.int32); w.owner[f] = 1; w.n_owners = 2
    r, sp, sv, ss, so = sorted_view(w)
    off, ids = orc.pack_destinations(r.sorted_hash, so, r.perm, w.dims, r.cell_start, r.cell_end, 2)
    np.testing.assert_array_equal(ids[off[0]:off[1]], [f])
    near = (np.abs(c - c[f]) <= 1).all(1)
    near[f] = False
    np.testing.assert_array_equal(np.sort(ids[off[1]:off[2]]), np.nonzero(near)[0])
    assert len(np.unique(c[ids[off[1]:off[2]]], axis=0)) == 27


def test_pack_boundary_single_owner_is_empty():
    w = W.lattice_block(8, 8, 8, 0.1, 3, owners=("single",))
    r = orc.step(w.posm, w.velr, w.sig, w.owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt,
                 floats=False)
    pb = orc.pack_boundary(r.boundary_ids, w.owner, w.n_owners, w.posm, w.velr, w.sig)
    assert pb.ids.size == 0 and (pb.offsets == 0).all()


# ----------------------------------------------------------------------------- NEXT-3: split passes
def test_split_passes_sum_to_the_single_pass_and_match_bruteforce():
    """Steps e and f as separate passes: pass e + pass f = the single pass (the
    sums are linear in the pair contributions), pair counts add up, and pass f alone equals a
    dense O(N^2) evaluation restricted to pairs with different owners."""
    w = W.t1b(side=10, seed=1104)
    owner = (np.arange(w.n) % 3).astype(np.int32)         # thoroughly mixed labels
    r = orc.step(w.posm, w.velr, w.sig, owner, w.origin, w.dims, w.h, w.K, w.G, 3, w.dt, floats=False)
    p = r.perm
    sp, sv, ss, so = w.posm[p], w.velr[p], np.ascontiguousarray(w.sig[:, p]), owner[p]
    args = (sp, sv, ss, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G)
    full = orc.interact(*args)
    e = orc.interact_split(*args, so, 1)
    f = orc.interact_split(*args, so, 2)
    assert e.pair_count + f.pair_count == full.pair_count and e.pair_count > 0 and f.pair_count > 0
    for name in ("drho", "acc", "dsig", "L"):
        a, b, c = getattr(e, name), getattr(f, name), getattr(full, name)
        assert np.max(np.abs(a + b - c)) <= 1e-13 * max(np.max(np.abs(c)), 1e-300), name
    # dense O(N^2) evaluation by distance only, restricted to same-owner pairs (pass e) and to
    # other-owner pairs (pass f): EVERY output of both loops (drho and L of loop 1, acc of loop 2,
    # dsig from the dense L), so that a swapped owner filter in either loop fails here
    x = sp[:, :3].astype(np.float64); m = sp[:, 3].astype(np.float64)
    v = sv[:, :3].astype(np.float64); rho = sv[:, 3].astype(np.float64)
    sg = ss.astype(np.float64)
    S = np.empty((w.n, 3, 3))
    S[:, 0, 0], S[:, 1, 1], S[:, 2, 2] = sg[0], sg[1], sg[2]
    S[:, 0, 1] = S[:, 1, 0] = sg[3]; S[:, 0, 2] = S[:, 2, 0] = sg[4]; S[:, 1, 2] = S[:, 2, 1] = sg[5]
    Sr = S / (rho ** 2)[:, None, None]
    h = float(w.h)
    xij = x[:, None, :] - x[None, :, :]
    rr = np.sqrt((xij ** 2).sum(-1))
    inside = (rr < 2 * h) & ~np.eye(w.n, dtype=bool)
    alpha = 21.0 / (16.0 * np.pi * h ** 3)
    vij = v[:, None, :] - v[None, :, :]
    for res, sel in ((e, so[:, None] == so[None, :]), (f, so[:, None] != so[None, :])):
        nb = inside & sel
        Fm = np.where(nb, -(5.0 * alpha / h ** 2) * (1 - rr / (2 * h)) ** 3, 0.0)
        gW = Fm[..., None] * xij                                     # [i, j, b]
        drho = (m[None, :] * (vij * gW).sum(-1)).sum(1)
        Ld = np.einsum("j,ija,ijb->iab", m / rho, -vij, gW)          # L[a][b] = sum V_j (v_j - v_i)_a gW_b
        accd = np.einsum("j,ijab,ijb->ia", m, Sr[:, None] + Sr[None, :], gW)
        D = 0.5 * (Ld + Ld.transpose(0, 2, 1)); Om = 0.5 * (Ld - Ld.transpose(0, 2, 1))
        trD = np.trace(D, axis1=1, axis2=2)
        sd = (w.K * trD)[:, None, None] * np.eye(3) + 2 * w.G * (D - (trD / 3)[:, None, None] * np.eye(3)) \
            + Om @ S - S @ Om
        dsd = np.stack([sd[:, 0, 0], sd[:, 1, 1], sd[:, 2, 2], sd[:, 0, 1], sd[:, 0, 2], sd[:, 1, 2]], 1)
        for name, ref in (("drho", drho), ("L", Ld), ("acc", accd), ("dsig", dsd)):
            got = getattr(res, name)
            assert np.max(np.abs(got - ref)) <= 1e-11 * np.max(np.abs(ref)), name
        assert res.pair_count == int(nb.sum())
    # the sampled form (idx) returns the same rows
    pick = np.array([0, 7, w.n // 2, w.n - 1])
    fs = orc.interact_split(*args, so, 2, idx=pick)
    np.testing.assert_array_equal(fs.acc, f.acc[pick])
    np.testing.assert_array_equal(fs.dsig, f.dsig[pick])


# ----------------------------------------------------------------------------- NEXT-4: per-particle h
def _sorted_with_h(w, hp):
    r, sp, sv, ss, so = sorted_view(w)
    return r, sp, sv, ss, so, hp[r.perm]


def test_varh_uniform_reduces_to_the_plain_loops_bit_for_bit():
    """H3: with every h_i = h the pair length (h + h) / 2 is h exactly: same bits as orc_interact."""
    w = W.t1b(10, 1106)
    r, sp, sv, ss, so, sh = _sorted_with_h(w, W.particle_h(w, ("uniform",)))
    a = orc.interact(sp, sv, ss, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G)
    b = orc.interact_varh(sp, sv, ss, sh, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G)
    assert a.pair_count == b.pair_count
    for name in ("drho", "L", "acc", "dsig"):
        assert np.array_equal(getattr(a, name), getattr(b, name)), name


@pytest.mark.parametrize("kind", [("species", 2, 0.75), ("species", 3, 0.6), ("random", 0.5)])
def test_varh_against_dense_evaluation_by_distance(kind):
    """H2: pair length h_ij = (h_i + h_j) / 2, neighbours r < 2 h_ij found by distance alone in an
    O(N^2) numpy evaluation (no buckets): every output of both loops, the pair count, and exact
    momentum conservation (the pair force stays antisymmetric)."""
    w = W.t1b(10, 1107)
    w.posm[:, 3] = (1.0 + 0.2 * np.random.default_rng(2).random(w.n)).astype(np.float32)
    hp = W.particle_h(w, kind)
    assert hp.max() <= w.h and hp.min() < w.h
    r, sp, sv, ss, so, sh = _sorted_with_h(w, hp)
    got = orc.interact_varh(sp, sv, ss, sh, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G)
    x = sp[:, :3].astype(np.float64); m = sp[:, 3].astype(np.float64)
    v = sv[:, :3].astype(np.float64); rho = sv[:, 3].astype(np.float64)
    sg = ss.astype(np.float64)
    S = np.empty((w.n, 3, 3))
    S[:, 0, 0], S[:, 1, 1], S[:, 2, 2] = sg[0], sg[1], sg[2]
    S[:, 0, 1] = S[:, 1, 0] = sg[3]; S[:, 0, 2] = S[:, 2, 0] = sg[4]; S[:, 1, 2] = S[:, 2, 1] = sg[5]
    Sr = S / (rho ** 2)[:, None, None]
    hij = 0.5 * (sh.astype(np.float64)[:, None] + sh.astype(np.float64)[None, :])
    xij = x[:, None, :] - x[None, :, :]
    rr = np.sqrt((xij ** 2).sum(-1))
    nb = (rr < 2 * hij) & ~np.eye(w.n, dtype=bool)
    alpha = 21.0 / (16.0 * np.pi * hij ** 3)
    Fm = np.where(nb, -(5.0 * alpha / hij ** 2) * (1 - rr / (2 * hij)) ** 3, 0.0)
    gW = Fm[..., None] * xij
    vij = v[:, None, :] - v[None, :, :]
    drho = (m[None, :] * (vij * gW).sum(-1)).sum(1)
    Ld = np.einsum("j,ija,ijb->iab", m / rho, -vij, gW)
    accd = np.einsum("j,ijab,ijb->ia", m, Sr[:, None] + Sr[None, :], gW)
    for name, ref in (("drho", drho), ("L", Ld), ("acc", accd)):
        assert np.max(np.abs(getattr(got, name) - ref)) <= 1e-11 * np.max(np.abs(ref)), name
    assert got.pair_count == int(nb.sum())
    f = m[:, None] * got.acc
    assert np.abs(f.sum(0)).max() <= 1e-12 * np.abs(f).sum() and np.abs(f).sum() > 0
    # fewer neighbours than with the maximum length everywhere
    full = orc.interact(sp, sv, ss, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G)
    assert got.pair_count < full.pair_count


def test_varh_two_species_lattice_neighbour_counts():
    """Un-jittered unit lattice, h = 1.3 on even sites and 1.0 on odd ones (checkerboard): the
    neighbours of an interior particle follow from integer arithmetic alone.  Even-even pairs see
    r^2 < 6.76 (h_ij = 1.3), odd-odd pairs r^2 < 4 (h_ij = 1.0), mixed pairs r^2 < 5.29
    (h_ij = 1.15); a lattice vector connects equal parities iff its coordinate sum is even."""
    side = 12
    w = W.lattice_block(side, side, side, 0.0, 5, owners=("single",))
    hp = W.particle_h(w, ("checker", 1.0 / 1.3))
    r, sp, sv, ss, so, sh = _sorted_with_h(w, hp)
    got = orc.interact_varh(sp, sv, ss, sh, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K, w.G,
                            idx=np.arange(w.n))
    d = np.arange(-3, 4)
    DX, DY, DZ = np.meshgrid(d, d, d, indexing="ij")
    r2 = (DX ** 2 + DY ** 2 + DZ ** 2).ravel()
    same = ((DX + DY + DZ) % 2 == 0).ravel()
    nz = r2 > 0
    n_even = int((nz & same & (r2 < 6.76)).sum() + (nz & ~same & (r2 < 5.29)).sum())
    n_odd = int((nz & same & (r2 < 4.0)).sum() + (nz & ~same & (r2 < 5.29)).sum())
    # per-particle neighbour counts through the single-particle form of the oracle
    site = np.rint(sp[:, :3]).astype(int)
    interior = np.all((site >= 3) & (site < side - 3), axis=1)
    for parity, expect in ((0, n_even), (1, n_odd)):
        pick = np.nonzero(interior & ((site.sum(1) & 1) == parity))[0][:5]
        for i in pick:
            one = orc.interact_varh(sp, sv, ss, sh, r.sorted_hash, w.dims, r.cell_start, r.cell_end, w.h, w.K,
                                    w.G, idx=np.array([i]))
            assert one.pair_count == expect, (parity, one.pair_count, expect)
    assert n_even != n_odd


# ----------------------------------------------------------------------------- NEXT-2: balancing
def test_balance_hand_worked_example_golden():
    """PAPER.md:36 on four particles, worked by hand (tests/golden/balancing_worked_example.txt)."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "balancing_worked_example.txt"))
            if l.strip() and not l.startswith("#")]
    x = np.array([float(r[1]) for r in rows], np.float32)
    posm = np.zeros((len(rows), 4), np.float32); posm[:, 0] = x; posm[:, 3] = 1
    own0 = np.array([int(r[2]) for r in rows], np.int32)
    own, k, bh = orc.balance(posm, own0, 2)
    assert k == 1
    np.testing.assert_array_equal(bh, [int(r[3]) for r in rows])
    np.testing.assert_array_equal(own, [int(r[4]) for r in rows])


def test_balance_three_owner_pair_order_golden():
    """Reading B1 ("repeated for each GPU pair"): pairs (0,1), (0,2), (1,2) in this
    order, each with the labels and centres of gravity the previous pair left.  Worked by hand in
    tests/golden/balancing_three_owner_example.txt; every other pair order and Cgs frozen at the
    start of the sweep give other hashes / labels / swap counts.  The typed sweep with one type and
    alpha = 0 is the same computation (Cg' = Cg_type) and must give the same rows."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "balancing_three_owner_example.txt"))
            if l.strip() and not l.startswith("#")]
    posm = np.zeros((len(rows), 4), np.float32)
    posm[:, 0] = [float(r[1]) for r in rows]; posm[:, 3] = 1
    own0 = np.array([int(r[2]) for r in rows], np.int32)
    want_hash, want_own = [int(r[3]) for r in rows], [int(r[4]) for r in rows]
    own, k, bh = orc.balance(posm, own0, 3)
    assert k == 3
    np.testing.assert_array_equal(bh, want_hash)
    np.testing.assert_array_equal(own, want_own)
    own_t, k_t, bh_t = orc.balance_types(posm, own0, np.zeros(len(rows), np.int32), 3, 1, alpha=0.0)
    assert k_t == 3
    np.testing.assert_array_equal(bh_t, want_hash)
    np.testing.assert_array_equal(own_t, want_own)


def test_balance_keeps_counts_slabs_are_a_fixed_point_single_owner_noop():
    """'The computational workload will stay balanced for all the swapping operations'
    (PAPER.md:30): every swap exchanges one particle each way; a slab decomposition has no
    particle past the middle of any Cg pair, so nothing moves."""
    w = W.lattice_block(24, 24, 24, 0.1, 21, owners=("random", 5))
    own, k, _ = orc.balance(w.posm, w.owner, 5)
    assert k > 0
    np.testing.assert_array_equal(np.bincount(own, minlength=5), np.bincount(w.owner, minlength=5))
    w1 = W.config(1, side=32)
    own1, k1, _ = orc.balance(w1.posm, w1.owner, w1.n_owners)
    assert k1 == 0 and np.array_equal(own1, w1.owner)
    w2 = W.lattice_block(10, 10, 10, 0.1, 22, owners=("single",))
    own2, k2, _ = orc.balance(w2.posm, w2.owner, 1)
    assert k2 == 0 and (own2 == 0).all()


def test_balance_hash_against_independent_projection():
    """One pair, dense numpy: projection on the Cg-Cg line, 0 on the own side of the middle,
    hmax beyond the other Cg, proportional in between; swap count = min of the
    positive counts; the swapped particles are the ones with the largest hashes."""
    rng = np.random.default_rng(5)
    n = 400
    posm = np.ones((n, 4), np.float32); posm[:, :3] = rng.random((n, 3), dtype=np.float32) * 10
    own0 = (rng.random(n) < 0.5).astype(np.int32)
    own, k, bh = orc.balance(posm, own0, 2)
    x = posm[:, :3].astype(np.float64)
    cg = [x[own0 == g].mean(0) for g in (0, 1)]
    h = np.zeros(n, np.int64)
    for g in (0, 1):
        d = cg[1 - g] - cg[g]
        s = ((x - cg[g]) @ d) / (d @ d)
        hv = np.where(s >= 1, 1000, np.where(s > 0.5, np.clip(np.ceil(1000 * (2 * s - 1)), 1, 1000), 0))
        h[own0 == g] = hv[own0 == g]
    assert np.mean(bh == h) > 0.995              # fixed-point Cg vs fp64 mean: a few ceil() flips at most
    na, nb = int(((bh > 0) & (own0 == 0)).sum()), int(((bh > 0) & (own0 == 1)).sum())
    assert k == min(na, nb)
    moved = own != own0
    assert moved.sum() == 2 * k and (bh[moved] > 0).all()
    for g in (0, 1):                              # the movers of a side have the largest hashes of that side
        side = own0 == g
        if (side & moved).any() and (side & ~moved & (bh > 0)).any():
            assert bh[side & moved].min() >= bh[side & ~moved].max()


def test_balance_hash_exact_rational_arithmetic_and_tie_order():
    """Readings B2-B4 and B6 pinned by exact arithmetic.  Positions on the 2^-6 dyadic grid are exact
    in the 2^-16 fixed point of B2, so the centres of gravity are exact rationals; the projection s
    and hmax (2 s - 1) are evaluated with fractions.Fraction (no rounding at all) and the oracle's
    fp64 hash must equal the exact ceil() for EVERY particle whose exact value is not within 1e-9
    of an integer.  The coarse grid also produces many equal hashes: the n movers of a side must be
    the first n of that side in the order (hash descending, id ascending) -- reading B6 -- which is
    recomputed here with a plain sort."""
    from fractions import Fraction as Fr
    import math
    for hmax, seed in ((1000, 17), (6, 18)):        # hmax = 6: six hash values only -> ties everywhere
        rng = np.random.default_rng(seed)
        n = 240
        xi = rng.integers(0, 8 * 64, size=(n, 3))              # multiples of 2^-6 in [0, 8)
        posm = np.ones((n, 4), np.float32)
        posm[:, :3] = (xi / 64.0).astype(np.float32)
        own0 = (rng.random(n) < 0.45).astype(np.int32)
        own, k, bh = orc.balance(posm, own0, 2, hmax=hmax)
        X = [[Fr(int(v), 64) for v in row] for row in xi]
        cg = []
        for g in (0, 1):
            ids = [i for i in range(n) if own0[i] == g]
            cg.append([sum(X[i][a] for i in ids) / len(ids) for a in range(3)])
        exact = np.zeros(n, np.int64)
        near_integer = np.zeros(n, bool)
        for i in range(n):
            g = int(own0[i])
            d = [cg[1 - g][a] - cg[g][a] for a in range(3)]
            s = sum((X[i][a] - cg[g][a]) * d[a] for a in range(3)) / sum(da * da for da in d)
            if s >= 1:
                exact[i] = hmax
            elif s > Fr(1, 2):
                v = hmax * (2 * s - 1)
                exact[i] = min(max(math.ceil(v), 1), hmax)
                near_integer[i] = abs(v - round(v)) < Fr(1, 10 ** 9)
        ok = ~near_integer
        assert ok.sum() >= n - 2
        np.testing.assert_array_equal(bh[ok], exact[ok])
        # B6: the movers of each side are the first n_move in (hash descending, id ascending)
        pos = [np.nonzero((own0 == g) & (bh > 0))[0] for g in (0, 1)]
        n_move = min(len(pos[0]), len(pos[1]))
        assert k == n_move and n_move > 0
        for g in (0, 1):
            order = sorted(pos[g].tolist(), key=lambda i: (-int(bh[i]), i))
            assert set(np.nonzero((own != own0) & (own0 == g))[0].tolist()) == set(order[:n_move])
        if hmax == 6:
            # the side that keeps some of its positive hashes cuts INSIDE a group of equal hashes,
            # so the id order decides who moves
            g = 0 if len(pos[0]) > len(pos[1]) else 1
            order = sorted(pos[g].tolist(), key=lambda i: (-int(bh[i]), i))
            assert n_move < len(order) and bh[order[n_move - 1]] == bh[order[n_move]]


def test_balance_restores_a_compact_decomposition():
    """The Fig. 1 -> Fig. 2 effect (PAPER.md:38 'the information exchange subset is always close
    to a surface'): random labels make every particle a boundary particle; a few sweeps bring the
    boundary fraction down towards that of a slab decomposition."""
    w = W.lattice_block(40, 40, 40, 0.1, 78, owners=("random", 3))
    own = w.owner
    for _ in range(3):
        own, _, _ = orc.balance(w.posm, own, 3)
    r = orc.step(w.posm, w.velr, w.sig, own, w.origin, w.dims, w.h, w.K, w.G, 3, w.dt, floats=False)
    assert r.boundary_ids.size < 0.55 * w.n
    r0 = orc.step(w.posm, w.velr, w.sig, w.owner, w.origin, w.dims, w.h, w.K, w.G, 3, w.dt, floats=False)
    assert r0.boundary_ids.size == w.n


# ----------------------------------------------------------------------------- NEXT-4: multi-type balancing
def test_balance_types_formula_counts_and_limits():
    """PAPER.md:56 Cg' = alpha Cg_all + (1 - alpha) Cg_type, alpha = 0.1:
      * every (owner, type) count is kept (only same-type particles swap);
      * alpha = 0 with ONE type is exactly the single-type algorithm of section III.A;
      * alpha = 1 uses the all-type Cg for every type (same lines for both types);
      * a hand-checkable pair: the biased centres are the alpha-blend of numpy means."""
    rng = np.random.default_rng(9)
    n = 600
    posm = np.ones((n, 4), np.float32); posm[:, :3] = rng.random((n, 3), dtype=np.float32) * 12
    owner = rng.integers(0, 3, n).astype(np.int32)
    ptype = (rng.random(n) < 0.3).astype(np.int32)
    own, k, bh = orc.balance_types(posm, owner, ptype, 3, 2)
    assert k > 0
    for t in (0, 1):
        np.testing.assert_array_equal(np.bincount(own[ptype == t], minlength=3),
                                      np.bincount(owner[ptype == t], minlength=3))
    # one type, alpha = 0  ==  section III.A
    own_a, k_a, bh_a = orc.balance(posm, owner, 3)
    own_b, k_b, bh_b = orc.balance_types(posm, owner, np.zeros(n, np.int32), 3, 1, alpha=0.0)
    assert k_a == k_b and np.array_equal(own_a, own_b) and np.array_equal(bh_a, bh_b)
    # two owners only (so that exactly one pair runs per type): the type-0 hashes of owner 0 follow
    # from numpy means blended with alpha = 0.1, written out independently of the oracle
    keep = owner < 2
    pm, ow, pt = posm[keep], owner[keep], ptype[keep]
    _, _, bh2 = orc.balance_types(pm, ow, pt, 2, 2)
    xs = pm[:, :3].astype(np.float64)
    cg2 = [0.1 * xs[ow == g].mean(0) + 0.9 * xs[(ow == g) & (pt == 0)].mean(0) for g in (0, 1)]
    d2 = cg2[1] - cg2[0]
    sel2 = (ow == 0) & (pt == 0)
    s2 = ((xs[sel2] - cg2[0]) @ d2) / (d2 @ d2)
    e2 = np.where(s2 >= 1, 1000, np.where(s2 > 0.5, np.clip(np.ceil(1000 * (2 * s2 - 1)), 1, 1000), 0))
    assert np.mean(bh2[sel2] == e2) > 0.99          # fixed-point Cg vs fp64 mean: a ceil() flip at most
    # alpha = 1: both types are balanced along the same (all-type) Cg line of a pair
    _, _, bh3 = orc.balance_types(pm, ow, pt, 2, 2, alpha=1.0)
    cg3 = [xs[ow == g].mean(0) for g in (0, 1)]
    d3 = cg3[1] - cg3[0]
    sel3 = (ow == 0) & (pt == 0)                     # type 0 runs first: labels still the input's
    s3 = ((xs[sel3] - cg3[0]) @ d3) / (d3 @ d3)
    e3 = np.where(s3 >= 1, 1000, np.where(s3 > 0.5, np.clip(np.ceil(1000 * (2 * s3 - 1)), 1, 1000), 0))
    assert np.mean(bh3[sel3] == e3) > 0.99
