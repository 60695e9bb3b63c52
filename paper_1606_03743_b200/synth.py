"""Seeded synthetic inputs for the five BASELINE.json configs (DESIGN.md §4 gives the recipe).

This module serves BOTH the CPU oracle and the CUDA path and therefore holds none of the
method's arithmetic: no cubature tables, no point mapping, no potential/field sums, no
distance-ratio logic.  It only builds meshes (vertices of flat triangles / rectangles),
charge densities and field points from fixed seeds.  numpy only; it imports neither
`oracle` nor the CUDA binding.

Element layout (the one `include/bemcub.h` states, following PAPER.md L101-111):
  etype[n]        uint8   0 = triangle, 1 = rectangle
  verts[n][3][3]  float64 triangle: A, B, C;  rectangle: P0, P1 = P0 + a*u_x, P3 = P0 + b*u_y
                          (the fourth corner P0 + a*u_x + b*u_y is implied)
  sigma[n]        float64 constant charge density per element, C/m^2
Field points: pts[m][3] float64.

These inputs stand in for the paper's KATRIN main-spectrometer meshes,
which are not available.
"""
from __future__ import annotations

import numpy as np

TRI = 0
RECT = 1

SEED_CFG1_PTS = 160603743
SEED_CFG2_SIGMA = 160603744
SEED_CFG2_PTS = 160603745
SEED_CFG4_SIGMA = 160603746
SEED_CFG4_TRACKS = 160603747
SEED_CFG5_PTS = 160603748


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def isotropic_directions(rng: np.random.Generator, m: int) -> np.ndarray:
    """m unit vectors uniform on the sphere (z uniform in [-1,1], azimuth uniform)."""
    z = rng.uniform(-1.0, 1.0, m)
    ph = rng.uniform(0.0, 2.0 * np.pi, m)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(ph), s * np.sin(ph), z], axis=1)


# --------------------------------------------------------------------------- meshes

def icosphere(level: int, radius: float = 1.0):
    """Icosahedron subdivided `level` times, edge midpoints re-projected to the sphere.

    Returns (vertices[nv][3], faces[nf][3] int64); nf = 20 * 4**level (level 3: 1280,
    level 5: 20480).  Faces are counter-clockwise seen from outside.
    """
    g = (1.0 + np.sqrt(5.0)) / 2.0
    v = np.array(
        [[-1, g, 0], [1, g, 0], [-1, -g, 0], [1, -g, 0],
         [0, -1, g], [0, 1, g], [0, -1, -g], [0, 1, -g],
         [g, 0, -1], [g, 0, 1], [-g, 0, -1], [-g, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array(
        [[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
         [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
         [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
         [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    verts = [tuple(p) for p in v]
    for _ in range(level):
        cache: dict[tuple[int, int], int] = {}

        def mid(i: int, j: int) -> int:
            key = (i, j) if i < j else (j, i)
            k = cache.get(key)
            if k is None:
                p = (np.asarray(verts[i]) + np.asarray(verts[j])) * 0.5
                p /= np.linalg.norm(p)
                verts.append(tuple(p))
                k = len(verts) - 1
                cache[key] = k
            return k

        nf = []
        for a, b, c in f:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            nf += [[a, ab, ca], [b, bc, ab], [c, ca, bc], [ab, bc, ca]]
        f = np.array(nf, dtype=np.int64)
    return np.asarray(verts, dtype=np.float64) * radius, f


def icosphere_elements(level: int, radius: float = 1.0):
    v, f = icosphere(level, radius)
    verts = np.ascontiguousarray(v[f])            # [nf][3][3]
    etype = np.zeros(len(f), dtype=np.uint8)
    return etype, verts


def cube_surface_rects(nside: int = 32, side: float = 1.0):
    """Surface of the cube [-side/2, side/2]^3 as 6*nside*nside axis-aligned squares."""
    h = side / 2.0
    d = side / nside
    i, j = np.meshgrid(np.arange(nside), np.arange(nside), indexing="ij")
    i = i.ravel().astype(np.float64)
    j = j.ravel().astype(np.float64)
    out = []
    for axis in range(3):
        a1, a2 = (axis + 1) % 3, (axis + 2) % 3
        for sgn in (-1.0, 1.0):
            p0 = np.zeros((nside * nside, 3))
            p0[:, axis] = sgn * h
            p0[:, a1] = -h + i * d
            p0[:, a2] = -h + j * d
            p1 = p0.copy()
            p1[:, a1] += d
            p3 = p0.copy()
            p3[:, a2] += d
            out.append(np.stack([p0, p1, p3], axis=1))
    verts = np.ascontiguousarray(np.concatenate(out, axis=0))
    etype = np.full(len(verts), RECT, dtype=np.uint8)
    return etype, verts


def cylinder_rects(radius: float, z0: float, z1: float, nphi: int, nz: int):
    """Cylinder wall as nphi*nz flat rectangles (chord x dz); vertices lie on the cylinder."""
    ph = 2.0 * np.pi * np.arange(nphi + 1) / nphi
    ph[-1] = 0.0                                   # close the seam exactly
    zz = z0 + (z1 - z0) * np.arange(nz + 1) / nz
    ip, iz = np.meshgrid(np.arange(nphi), np.arange(nz), indexing="ij")
    ip = ip.ravel()
    iz = iz.ravel()
    x0, y0 = radius * np.cos(ph[ip]), radius * np.sin(ph[ip])
    x1, y1 = radius * np.cos(ph[ip + 1]), radius * np.sin(ph[ip + 1])
    p0 = np.stack([x0, y0, zz[iz]], axis=1)
    p1 = np.stack([x1, y1, zz[iz]], axis=1)
    p3 = np.stack([x0, y0, zz[iz + 1]], axis=1)
    verts = np.ascontiguousarray(np.stack([p0, p1, p3], axis=1))
    return np.full(len(verts), RECT, dtype=np.uint8), verts


def cone_tris(r0: float, r1: float, z0: float, z1: float, nphi: int, ns: int):
    """Cone frustum from (r0, z0) to (r1, z1) as nphi*ns quads, each split into 2 triangles."""
    ph = 2.0 * np.pi * np.arange(nphi + 1) / nphi
    ph[-1] = 0.0
    s = np.arange(ns + 1) / ns
    rr = r0 + (r1 - r0) * s
    zz = z0 + (z1 - z0) * s
    ip, js = np.meshgrid(np.arange(nphi), np.arange(ns), indexing="ij")
    ip = ip.ravel()
    js = js.ravel()

    def vtx(i, j):
        return np.stack([rr[j] * np.cos(ph[i]), rr[j] * np.sin(ph[i]), zz[j]], axis=1)

    v00, v10 = vtx(ip, js), vtx(ip + 1, js)
    v01, v11 = vtx(ip, js + 1), vtx(ip + 1, js + 1)
    t1 = np.stack([v00, v10, v11], axis=1)
    t2 = np.stack([v00, v11, v01], axis=1)
    verts = np.empty((2 * len(t1), 3, 3))
    verts[0::2] = t1
    verts[1::2] = t2
    return np.zeros(len(verts), dtype=np.uint8), np.ascontiguousarray(verts)


def element_centroids(etype: np.ndarray, verts: np.ndarray) -> np.ndarray:
    """Geometric centre of each element (mesh bookkeeping for the sigma field below)."""
    tri = verts.mean(axis=1)
    rect = 0.5 * (verts[:, 1] + verts[:, 2])
    return np.where((etype == RECT)[:, None], rect, tri)


# --------------------------------------------------------------------------- configs

def config1(level: int = 3, m: int = 1000, seed: int = SEED_CFG1_PTS):
    """Icosphere R=1 (level 3: 1280 triangles), sigma = 1e-9; m points uniform in volume in
    the shell 1.5 < |r| < 3."""
    etype, verts = icosphere_elements(level, 1.0)
    sigma = np.full(len(etype), 1e-9)
    rng = _rng(seed)
    u = rng.random(m)
    r = np.cbrt(1.5 ** 3 + u * (3.0 ** 3 - 1.5 ** 3))
    pts = isotropic_directions(rng, m) * r[:, None]
    return dict(name="cfg1_icosphere", etype=etype, verts=verts, sigma=sigma,
                pts=np.ascontiguousarray(pts))


def config2(nside: int = 32, m: int = 10000, seed_sigma: int = SEED_CFG2_SIGMA,
            seed_pts: int = SEED_CFG2_PTS):
    """Unit-cube surface, 6*32*32 squares, sigma iid U(-1e-9, 1e-9); m points uniform in
    [-2,2]^3 rejecting points closer than 0.1 to the surface (inside or outside)."""
    etype, verts = cube_surface_rects(nside, 1.0)
    sigma = _rng(seed_sigma).uniform(-1e-9, 1e-9, len(etype))
    rng = _rng(seed_pts)
    pts = np.empty((0, 3))
    while len(pts) < m:
        c = rng.uniform(-2.0, 2.0, (2 * m, 3))
        a = np.abs(c)
        q = np.maximum(a - 0.5, 0.0)
        outside = np.linalg.norm(q, axis=1)
        inside = 0.5 - a.max(axis=1)
        dist = np.where(a.max(axis=1) <= 0.5, inside, outside)
        pts = np.concatenate([pts, c[dist >= 0.1]], axis=0)
    return dict(name="cfg2_cube", etype=etype, verts=verts, sigma=sigma,
                pts=np.ascontiguousarray(pts[:m]))


def config3(level: int = 5):
    """Level-5 icosphere (20480 triangles), unit sigma; field points = centroids (implied)."""
    etype, verts = icosphere_elements(level, 1.0)
    return dict(name="cfg3_matrix", etype=etype, verts=verts,
                sigma=np.ones(len(etype)))


def helical_tracks(ntracks: int, npts: int, seed: int = SEED_CFG4_TRACKS,
                   rmax: float = 4.5, zspan: float = 9.0) -> np.ndarray:
    """ntracks helices of npts points each: gyroradius U(0.01,0.5), guiding centre uniform in
    area with rho_c + r_g <= rmax, z from -zspan to zspan, 5..50 turns."""
    rng = _rng(seed)
    rg = rng.uniform(0.01, 0.5, ntracks)
    rho = (rmax - rg) * np.sqrt(rng.random(ntracks))
    phc = rng.uniform(0.0, 2.0 * np.pi, ntracks)
    turns = rng.uniform(5.0, 50.0, ntracks)
    th0 = rng.uniform(0.0, 2.0 * np.pi, ntracks)
    t = np.arange(npts) / max(npts - 1, 1)
    th = th0[:, None] + 2.0 * np.pi * turns[:, None] * t[None, :]
    x = rho[:, None] * np.cos(phc)[:, None] + rg[:, None] * np.cos(th)
    y = rho[:, None] * np.sin(phc)[:, None] + rg[:, None] * np.sin(th)
    z = np.broadcast_to(-zspan + 2.0 * zspan * t[None, :], x.shape)
    return np.ascontiguousarray(np.stack([x, y, z], axis=2).reshape(-1, 3))


def fourier_sigma(cen: np.ndarray, seed: int = SEED_CFG4_SIGMA, amp: float = 1e-9) -> np.ndarray:
    """Smooth random charge density: 8 seeded Fourier modes in z and azimuth, max|sigma| = amp."""
    rng = _rng(seed)
    a = rng.random(8)
    jm = rng.integers(1, 9, 8)
    nm = rng.integers(0, 5, 8)
    psi = rng.uniform(0.0, 2.0 * np.pi, 8)
    z = cen[:, 2]
    ph = np.arctan2(cen[:, 1], cen[:, 0])
    s = np.zeros(len(cen))
    for k in range(8):
        s += a[k] * np.cos(2.0 * np.pi * jm[k] * z / 40.0 + nm[k] * ph + psi[k])
    return s * (amp / np.abs(s).max())


def config4(scale: float = 1.0, ntracks: int | None = None, npts_per_track: int | None = None):
    """Mixed electrode: cylinder R=5, z in [-10,10] (nphi x nz rectangles) + two end cones
    r 5 -> 0.5 over z in +-[10,15] (triangles); smooth random sigma; helical-track field points.

    scale = 1 gives 8e5 rectangles + 2e5 triangles and 1e6 field points; scale < 1 shrinks
    every mesh dimension by sqrt(scale) and the track/point counts likewise (used by tests).
    """
    f = np.sqrt(scale)
    nphi, nz = max(8, int(round(1000 * f))), max(4, int(round(800 * f)))
    cphi, cs = max(8, int(round(500 * f))), max(2, int(round(100 * f)))
    t_r, v_r = cylinder_rects(5.0, -10.0, 10.0, nphi, nz)
    t_a, v_a = cone_tris(5.0, 0.5, 10.0, 15.0, cphi, cs)
    t_b, v_b = cone_tris(5.0, 0.5, -10.0, -15.0, cphi, cs)
    etype = np.concatenate([t_r, t_a, t_b])
    verts = np.ascontiguousarray(np.concatenate([v_r, v_a, v_b], axis=0))
    sigma = fourier_sigma(element_centroids(etype, verts))
    nt = ntracks if ntracks is not None else max(1, int(round(1000 * f)))
    npt = npts_per_track if npts_per_track is not None else max(2, int(round(1000 * f)))
    pts = helical_tracks(nt, npt)
    return dict(name="cfg4_mixed_electrode", etype=etype, verts=verts, sigma=sigma, pts=pts,
                ntracks=nt, npts_per_track=npt)


CFG5_TRIANGLE = np.array([[[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.3, 0.8, 0.0]]])
CFG5_SQUARE = np.array([[[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.0, 1.0, 0.0]]])


def config5(kind: int, m: int = 1_000_000, seed: int = SEED_CFG5_PTS,
            dr_lo: float = 1.0, dr_hi: float = 1e6):
    """Single triangle (0,0,0),(1,0,0),(0.3,0.8,0) or single unit square, sigma = 1; m field
    points at log-uniform multiples `ratio` in [dr_lo, dr_hi] of the mean side length from the
    element's centre, isotropic directions.  `ratio` is returned for plotting/binning only."""
    verts = (CFG5_TRIANGLE if kind == TRI else CFG5_SQUARE).copy()
    etype = np.array([kind], dtype=np.uint8)
    cen = element_centroids(etype, verts)[0]
    if kind == TRI:
        a, b, c = verts[0]
        mean_side = (np.linalg.norm(b - a) + np.linalg.norm(c - b) + np.linalg.norm(a - c)) / 3.0
    else:
        mean_side = 1.0
    rng = _rng(seed)
    ratio = np.exp(rng.uniform(np.log(dr_lo), np.log(dr_hi), m))
    pts = cen[None, :] + isotropic_directions(rng, m) * (ratio * mean_side)[:, None]
    return dict(name="cfg5_tri" if kind == TRI else "cfg5_square", etype=etype, verts=verts,
                sigma=np.ones(1), pts=np.ascontiguousarray(pts), ratio=ratio)


def random_elements(kind: int, n: int, seed: int):
    """The paper's random-element protocol: corner points uniform in the unit
    cube.  Rectangles: P0 uniform, two orthogonal sides with lengths U(0.1, 1) in a random
    orientation."""
    rng = _rng(seed)
    if kind == TRI:
        verts = rng.random((n, 3, 3))
    else:
        p0 = rng.random((n, 3))
        e1 = isotropic_directions(rng, n)
        t = isotropic_directions(rng, n)
        e2 = np.cross(e1, t)
        e2 /= np.linalg.norm(e2, axis=1, keepdims=True)
        a = rng.uniform(0.1, 1.0, n)
        b = rng.uniform(0.1, 1.0, n)
        verts = np.stack([p0, p0 + a[:, None] * e1, p0 + b[:, None] * e2], axis=1)
    return np.full(n, kind, dtype=np.uint8), np.ascontiguousarray(verts)


def mean_side_and_centre(etype: np.ndarray, verts: np.ndarray):
    """(centre[n][3], mean side length[n]) of each element - used only to PLACE field points at a
    wanted distance ratio; the libraries compute their own."""
    cen = element_centroids(etype, verts)
    a = np.linalg.norm(verts[:, 1] - verts[:, 0], axis=1)
    b = np.linalg.norm(verts[:, 2] - verts[:, 1], axis=1)
    c = np.linalg.norm(verts[:, 0] - verts[:, 2], axis=1)
    tri = (a + b + c) / 3.0
    rect = 0.5 * (a + c)                      # P0->P1 and P0->P3 are the two sides
    return cen, np.where(etype == RECT, rect, tri)


def aspect_ratio(etype: np.ndarray, verts: np.ndarray) -> np.ndarray:
    """Triangle: longest side divided by the corresponding height; rectangle: longer side divided by
    the shorter one."""
    a = np.linalg.norm(verts[:, 1] - verts[:, 0], axis=1)
    b = np.linalg.norm(verts[:, 2] - verts[:, 1], axis=1)
    c = np.linalg.norm(verts[:, 0] - verts[:, 2], axis=1)
    longest = np.maximum(np.maximum(a, b), c)
    area = 0.5 * np.linalg.norm(np.cross(verts[:, 1] - verts[:, 0], verts[:, 2] - verts[:, 0]), axis=1)
    tri = longest / (2.0 * area / longest)
    rect = np.maximum(a, c) / np.minimum(a, c)
    return np.where(etype == RECT, rect, tri)


def random_pairs(kind: int, n: int, ratio, seed: int):
    """The paper's accuracy protocol: n random elements (corners in the unit
    cube), one field point each in a random direction from the element's centre at `ratio` (scalar or
    [n]) mean side lengths.  Returns (etype, verts, pts)."""
    etype, verts = random_elements(kind, n, seed)
    cen, side = mean_side_and_centre(etype, verts)
    dirs = isotropic_directions(_rng(seed + 7919), n)
    pts = cen + dirs * (np.broadcast_to(np.asarray(ratio, dtype=np.float64), (n,)) * side)[:, None]
    return etype, verts, np.ascontiguousarray(pts)


def shard_range(total: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [lo, hi) slice of `total` units owned by `rank` of `world` (sizes differ by
    at most one).  Used to shard field points / matrix rows across GPUs (no collective)."""
    base, rem = divmod(total, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
