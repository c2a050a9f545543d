"""Seeded conforming triangle meshes of a rectangle [0,W]x[0,H].

Every mesh is: float64 vertices [V][2], int32 CCW triangles [R][3], int32
material id per triangle [R].  One triangle = one flat-source region (FSR,
PAPER.md:65).  Non-rectangular cores are embedded in their bounding rectangle
with filler triangles ("bounding box of the whole domain").

No track, ray or transport arithmetic lives here.
"""
from dataclasses import dataclass
import numpy as np


@dataclass
class Mesh:
    xy: np.ndarray         # [V][2] float64
    tri: np.ndarray        # [R][3] int32, counter-clockwise
    material: np.ndarray   # [R] int32
    W: float
    H: float

    @property
    def n_regions(self) -> int:
        return int(self.tri.shape[0])

    def areas(self) -> np.ndarray:
        p = self.xy[self.tri]
        a = p[:, 1] - p[:, 0]
        b = p[:, 2] - p[:, 0]
        return 0.5 * (a[:, 0] * b[:, 1] - a[:, 1] * b[:, 0])


def _orient_ccw(xy, tri):
    p = xy[tri]
    a = p[:, 1] - p[:, 0]
    b = p[:, 2] - p[:, 0]
    sgn = a[:, 0] * b[:, 1] - a[:, 1] * b[:, 0]
    tri = tri.copy()
    flip = sgn < 0
    tri[flip, 1], tri[flip, 2] = tri[flip, 2].copy(), tri[flip, 1].copy()
    return tri


def validate_mesh(mesh: Mesh, rtol: float = 1e-11) -> None:
    """Raise ValueError unless the mesh is a conforming CCW triangulation of the rectangle."""
    xy, tri, W, H = mesh.xy, mesh.tri, mesh.W, mesh.H
    if xy.dtype != np.float64 or tri.dtype != np.int32 or mesh.material.dtype != np.int32:
        raise ValueError("dtype")
    if tri.min() < 0 or tri.max() >= len(xy):
        raise ValueError("vertex index out of range")
    if len(np.unique(tri)) != len(xy):
        raise ValueError("unreferenced vertex")
    area = mesh.areas()
    if not np.all(area > 0):
        raise ValueError(f"{int((area <= 0).sum())} triangles are not CCW with positive area")
    if abs(area.sum() - W * H) > rtol * W * H:
        raise ValueError(f"areas sum to {area.sum()!r}, expected {W * H!r}")
    if xy[:, 0].min() != 0.0 or xy[:, 0].max() != W or xy[:, 1].min() != 0.0 or xy[:, 1].max() != H:
        raise ValueError("vertices do not span the rectangle exactly")
    # conformity: every undirected edge is shared by exactly two triangles, or by one and lies on a side
    e = np.concatenate([tri[:, [0, 1]], tri[:, [1, 2]], tri[:, [2, 0]]]).astype(np.int64)
    lo = np.minimum(e[:, 0], e[:, 1])
    hi = np.maximum(e[:, 0], e[:, 1])
    key = lo * (len(xy) + 1) + hi
    uk, idx, cnt = np.unique(key, return_index=True, return_counts=True)
    if cnt.max() > 2:
        raise ValueError("an edge is shared by more than two triangles")
    b = idx[cnt == 1]
    pa, pb = xy[lo[b]], xy[hi[b]]
    on_side = (((pa[:, 0] == 0.0) & (pb[:, 0] == 0.0)) | ((pa[:, 0] == W) & (pb[:, 0] == W)) |
               ((pa[:, 1] == 0.0) & (pb[:, 1] == 0.0)) | ((pa[:, 1] == H) & (pb[:, 1] == H)))
    if not np.all(on_side):
        raise ValueError("a boundary edge does not lie on a side of the rectangle")
    # directed edges must be unique (orientation consistency)
    dkey = e[:, 0] * (len(xy) + 1) + e[:, 1]
    if len(np.unique(dkey)) != len(dkey):
        raise ValueError("duplicate directed edge")
    # Euler: R = 2V - B - 2 for a triangulated disc
    B = len(b)
    if len(tri) != 2 * len(xy) - B - 2:
        raise ValueError("triangle count violates Euler's formula (hole or overlap)")


# ----------------------------------------------------------------------------------------------
# structured helpers
# ----------------------------------------------------------------------------------------------
def rect_tri_mesh(W, H, nx, ny, seed=None, jitter=0.0, n_materials=1) -> Mesh:
    """nx x ny grid of rectangles, each split into two triangles with alternating diagonals.

    Interior vertices are displaced by `jitter` x cell size (seeded); materials drawn at random
    per triangle when n_materials > 1.  Used for homogeneous / closed-form tests and small cases.
    """
    rng = np.random.default_rng(seed)
    xs = np.linspace(0.0, W, nx + 1)
    ys = np.linspace(0.0, H, ny + 1)
    xs[-1], ys[-1] = W, H
    X, Y = np.meshgrid(xs, ys, indexing="xy")          # [ny+1][nx+1]
    if jitter > 0.0:
        dx, dy = W / nx, H / ny
        jx = (rng.random(X.shape) - 0.5) * 2 * jitter * dx
        jy = (rng.random(Y.shape) - 0.5) * 2 * jitter * dy
        for j in (jx, jy):                      # boundary vertices stay put
            j[0, :] = 0.0
            j[-1, :] = 0.0
            j[:, 0] = 0.0
            j[:, -1] = 0.0
        X = X + jx
        Y = Y + jy
    xy = np.stack([X.ravel(), Y.ravel()], axis=1)
    vid = np.arange((nx + 1) * (ny + 1)).reshape(ny + 1, nx + 1)
    a = vid[:-1, :-1].ravel()
    b = vid[:-1, 1:].ravel()
    c = vid[1:, 1:].ravel()
    d = vid[1:, :-1].ravel()
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    alt = ((ix + iy) % 2 == 0).ravel()
    t1 = np.where(alt[:, None], np.stack([a, b, c], 1), np.stack([a, b, d], 1))
    t2 = np.where(alt[:, None], np.stack([a, c, d], 1), np.stack([b, c, d], 1))
    tri = np.empty((2 * nx * ny, 3), dtype=np.int32)
    tri[0::2] = t1
    tri[1::2] = t2
    tri = _orient_ccw(xy, tri).astype(np.int32)
    if n_materials > 1:
        mat = rng.integers(0, n_materials, size=len(tri)).astype(np.int32)
    else:
        mat = np.zeros(len(tri), dtype=np.int32)
    return Mesh(np.ascontiguousarray(xy), np.ascontiguousarray(tri), mat, float(W), float(H))


def _angles(pts, c):
    return np.mod(np.arctan2(pts[:, 1] - c[1], pts[:, 0] - c[0]), 2 * np.pi)


def _annulus(ia, anga, ib, angb):
    """Triangulate between an inner closed loop (ids ia, angles anga) and an outer loop (ib, angb).

    Both loops are sorted counter-clockwise by angle about a common interior point.  Marches around
    advancing whichever loop has the smaller next angle; returns a list of vertex-id triples.
    """
    na, nb = len(ia), len(ib)
    if na == 1:
        return [(ia[0], ib[j], ib[(j + 1) % nb]) for j in range(nb)]
    # rotate the outer loop so that it starts at the first outer angle >= the first inner angle
    j0 = int(np.searchsorted(angb, anga[0]))
    order = [(j0 + k) % nb for k in range(nb)]
    ib = [ib[k] for k in order]
    ub = np.array([angb[k] for k in order], dtype=np.float64)
    ub = np.where(ub < anga[0], ub + 2 * np.pi, ub)
    ua = np.concatenate([anga, [anga[0] + 2 * np.pi]])
    ub = np.concatenate([ub, [ub[0] + 2 * np.pi]])
    tris = []
    i = j = 0
    while i < na or j < nb:
        nxt_a = ua[i + 1] if i < na else np.inf
        nxt_b = ub[j + 1] if j < nb else np.inf
        if nxt_a <= nxt_b:
            tris.append((ia[i % na], ib[j % nb], ia[(i + 1) % na]))
            i += 1
        else:
            tris.append((ia[i % na], ib[j % nb], ib[(j + 1) % nb]))
            j += 1
    return tris


def _cell_template(w, h, ring_radii, ring_counts, side_div, ring_phase=None, centre_jitter=(0.0, 0.0)):
    """Local mesh of one w x h cell: centre, concentric rings, boundary points (side_div segments per side).

    Returns (pts [n][2], tris [m][3], ring_of_tri [m]) with ring_of_tri = index of the annulus
    (0 = centre fan, k = between ring k-1 and ring k, last = out to the boundary).
    Boundary points come first in a fixed order so that tiling can de-duplicate them.
    """
    cx, cy = 0.5 * w, 0.5 * h
    pts = []
    # boundary loop, counter-clockwise from the lower-left corner
    for k in range(side_div):
        pts.append((w * k / side_div, 0.0))
    for k in range(side_div):
        pts.append((w, h * k / side_div))
    for k in range(side_div):
        pts.append((w - w * k / side_div, h))
    for k in range(side_div):
        pts.append((0.0, h - h * k / side_div))
    nb = len(pts)
    loops = []
    pts.append((cx + centre_jitter[0], cy + centre_jitter[1]))
    loops.append([nb])
    for k, (r, n) in enumerate(zip(ring_radii, ring_counts)):
        ph = 0.0 if ring_phase is None else ring_phase[k]
        ids = []
        for m in range(n):
            a = ph + 2 * np.pi * m / n
            ids.append(len(pts))
            pts.append((cx + r * np.cos(a), cy + r * np.sin(a)))
        loops.append(ids)
    loops.append(list(range(nb)))
    pts = np.array(pts, dtype=np.float64)
    c = np.array([cx, cy])
    tris, ring_of = [], []
    for k in range(len(loops) - 1):
        ia, ib = loops[k], loops[k + 1]
        aa = _angles(pts[ia], c) if len(ia) > 1 else np.array([0.0])
        ab = _angles(pts[ib], c)
        oa = np.argsort(aa, kind="stable")
        ob = np.argsort(ab, kind="stable")
        t = _annulus([ia[q] for q in oa], aa[oa], [ib[q] for q in ob], ab[ob])
        tris += t
        ring_of += [k] * len(t)
    tris = _orient_ccw(pts, np.array(tris, dtype=np.int64))
    return pts, tris, np.array(ring_of, dtype=np.int32), nb


def pin_cell_mesh(pitch=1.26, r_fuel=0.54, seed=0) -> Mesh:
    """Config-1 shape: one square pin cell, 64 triangles.

    Vertices: (jittered) centre, 8 on r = r_fuel/2, 16 on r = r_fuel, 16 on the square
    (4 corners + 3 per side) -> 8 + 24 + 32 = 64 triangles.  Ring phases and the centre jitter
    come from the seed.  Materials by seed: 0 = fuel (inside r_fuel), 1 = clad (outer-zone
    triangles whose centroid radius is below a seeded threshold), 2 = moderator.
    """
    rng = np.random.default_rng(seed)
    ph = [float(rng.uniform(0, 2 * np.pi / 8)), float(rng.uniform(0, 2 * np.pi / 16))]
    cj = tuple((rng.random(2) - 0.5) * 0.08 * pitch)
    pts, tris, ring, _ = _cell_template(pitch, pitch, [0.5 * r_fuel, r_fuel], [8, 16], 4, ph, cj)
    cen = pts[tris].mean(axis=1) - 0.5 * pitch
    rc = np.hypot(cen[:, 0], cen[:, 1])
    mat = np.where(ring <= 1, 0, 2).astype(np.int32)
    thr = float(rng.uniform(0.60, 0.66))
    mat[(ring == 2) & (rc < thr)] = 1
    xy = pts.copy()
    xy[np.abs(xy[:, 0] - pitch) < 1e-12, 0] = pitch
    xy[np.abs(xy[:, 1] - pitch) < 1e-12, 1] = pitch
    xy[np.abs(xy[:, 0]) < 1e-12, 0] = 0.0
    xy[np.abs(xy[:, 1]) < 1e-12, 1] = 0.0
    return Mesh(np.ascontiguousarray(xy), np.ascontiguousarray(tris.astype(np.int32)), mat,
                float(pitch), float(pitch))


def _tile_cells(cells, W, H):
    """Assemble a list of (origin_x, origin_y, pts, tris, mat_per_tri) cells into one mesh.

    Shared boundary points are merged by a 1e-9 cm rounding key; points within 1e-9 of a side of
    the rectangle are snapped onto it exactly.
    """
    all_pts, all_tri, all_mat = [], [], []
    base = 0
    for ox, oy, pts, tris, mat in cells:
        all_pts.append(pts + np.array([ox, oy]))
        all_tri.append(tris + base)
        all_mat.append(mat)
        base += len(pts)
    P = np.concatenate(all_pts)
    T = np.concatenate(all_tri)
    M = np.concatenate(all_mat).astype(np.int32)
    key = np.round(P / 1e-9).astype(np.int64)
    _, first, inv = np.unique(key, axis=0, return_index=True, return_inverse=True)
    inv = inv.reshape(-1)
    xy = P[first].copy()
    tri = inv[T].astype(np.int32)
    for col, lim in ((0, W), (1, H)):
        xy[np.abs(xy[:, col]) < 1e-9, col] = 0.0
        xy[np.abs(xy[:, col] - lim) < 1e-9, col] = lim
    return Mesh(np.ascontiguousarray(xy), np.ascontiguousarray(tri), M, float(W), float(H))


def square_lattice_mesh(pin_material, pitch=1.26, r_fuel=0.54, moderator=None,
                        band_cells=0, band_width=0.0, band_material=None) -> Mesh:
    """Square lattice of pin cells (configs 2 and 3).

    pin_material: int array [ny][nx], material of the pin's fuel zone (inside r_fuel);
    the rest of the cell gets `moderator`.  Per-pin template: centre + 8 on the circle + 8 on the
    cell boundary (corners + mid-sides) -> 8 + 16 = 24 triangles; the template is symmetric so
    neighbours conform.  Optionally a reflector band of `band_cells` cells (total width
    band_width) is appended on the +x and +y sides, meshed with the same 24-triangle template,
    all of material band_material.
    """
    pin_material = np.asarray(pin_material)
    ny, nx = pin_material.shape
    if moderator is None:
        moderator = int(pin_material.max()) + 1
    pts, tris, ring, _ = _cell_template(pitch, pitch, [r_fuel], [8], 2)
    cells = []
    for iy in range(ny):
        for ix in range(nx):
            mat = np.where(ring == 0, int(pin_material[iy, ix]), moderator).astype(np.int32)
            cells.append((ix * pitch, iy * pitch, pts, tris, mat))
    W, H = nx * pitch, ny * pitch
    if band_cells > 0:
        bw = band_width / band_cells
        if band_material is None:
            band_material = moderator
        rr = 0.43 * min(bw, pitch)
        tx = _cell_template(bw, pitch, [rr], [8], 2)       # right band cells
        ty = _cell_template(pitch, bw, [rr], [8], 2)       # top band cells
        tc = _cell_template(bw, bw, [rr], [8], 2)          # corner cells
        for iy in range(ny):
            for k in range(band_cells):
                cells.append((W + k * bw, iy * pitch, tx[0], tx[1],
                              np.full(len(tx[1]), band_material, np.int32)))
        for k in range(band_cells):
            for ix in range(nx):
                cells.append((ix * pitch, H + k * bw, ty[0], ty[1],
                              np.full(len(ty[1]), band_material, np.int32)))
            for k2 in range(band_cells):
                cells.append((W + k2 * bw, H + k * bw, tc[0], tc[1],
                              np.full(len(tc[1]), band_material, np.int32)))
        W, H = W + band_width, H + band_width
    return _tile_cells(cells, W, H)


def _delaunay(points):
    from scipy.spatial import Delaunay
    d = Delaunay(points)
    if d.coplanar.size:
        raise ValueError("Delaunay dropped coplanar points")
    tri = d.simplices.astype(np.int32)
    # remove zero-area hull slivers that Qhull may create from collinear side points
    p = points[tri]
    a = p[:, 1] - p[:, 0]
    b = p[:, 2] - p[:, 0]
    area2 = a[:, 0] * b[:, 1] - a[:, 1] * b[:, 0]
    tri = tri[np.abs(area2) > 1e-14]
    return _orient_ccw(points, tri).astype(np.int32)


def hex_core_mesh(pitch=0.9, rings=9, margin=0.45, seed=0):
    """Config-4 shape: 7 hexagonal assemblies of 3*rings*(rings+1)+1 pins on one global hex lattice.

    Point set = for every hex pin cell of a lattice covering the bounding rectangle: centre,
    6 corners, 6 mid-sides (shared points merged), clipped to the rectangle's interior, plus
    evenly spaced points on the four sides; triangulated by Delaunay.  Cell edges are Gabriel edges
    of this point set, so every full cell is cut into exactly 12 triangles that never straddle a
    cell boundary.  Returns (Mesh, cell_class) where material ids are:
      0..6  assembly index (pin cells within `rings` of an assembly centre),
      7     duct (cells at hex distance rings+1 from an assembly centre),
      8     coolant / filler (everything else out to the bounding rectangle).
    """
    n = rings
    a1 = np.array([pitch, 0.0])
    a2 = np.array([0.5 * pitch, 0.5 * np.sqrt(3.0) * pitch])
    centres_ax = [(0, 0), (n + 1, n + 1), (-(n + 1), 2 * (n + 1)), (-2 * (n + 1), n + 1),
                  (-(n + 1), -(n + 1)), (n + 1, -2 * (n + 1)), (2 * (n + 1), -(n + 1))]

    def hexdist(q, r):
        return np.maximum(np.maximum(np.abs(q), np.abs(r)), np.abs(q + r))

    # bounding rectangle of all assembly cells (+ margin)
    Rc = pitch / np.sqrt(3.0)
    ext_x = ext_y = 0.0
    for (cq, cr) in centres_ax:
        for q in range(-n, n + 1):
            for r in range(-n, n + 1):
                if hexdist(np.array(q), np.array(r)) <= n:
                    c = (cq + q) * a1 + (cr + r) * a2
                    ext_x = max(ext_x, abs(c[0]) + 0.5 * pitch)
                    ext_y = max(ext_y, abs(c[1]) + Rc)
    W = 2 * (ext_x + margin)
    H = 2 * (ext_y + margin)
    org = np.array([0.5 * W, 0.5 * H])
    # lattice cells covering the rectangle
    qmax = int(np.ceil(W / pitch)) + 2
    rmax = int(np.ceil(H / (0.5 * np.sqrt(3.0) * pitch))) + 2
    Q, Rr = np.meshgrid(np.arange(-qmax, qmax + 1), np.arange(-rmax, rmax + 1), indexing="ij")
    Q = Q.ravel()
    Rr = Rr.ravel()
    cen = Q[:, None] * a1 + Rr[:, None] * a2 + org
    ang_c = np.pi / 6 + np.arange(6) * np.pi / 3           # corners (pointy-top hexagon)
    ang_m = np.arange(6) * np.pi / 3                       # mid-sides
    corner = np.stack([Rc * np.cos(ang_c), Rc * np.sin(ang_c)], 1)
    mids = np.stack([0.5 * pitch * np.cos(ang_m), 0.5 * pitch * np.sin(ang_m)], 1)
    local = np.concatenate([np.zeros((1, 2)), corner, mids])
    P = (cen[:, None, :] + local[None, :, :]).reshape(-1, 2)
    key = np.round(P / 1e-7).astype(np.int64)
    _, first = np.unique(key, axis=0, return_index=True)
    P = P[np.sort(first)]
    tol = 0.2 * pitch
    inside = (P[:, 0] > tol) & (P[:, 0] < W - tol) & (P[:, 1] > tol) & (P[:, 1] < H - tol)
    P = P[inside]
    nbx = int(np.ceil(W / (0.5 * pitch)))
    nby = int(np.ceil(H / (0.5 * pitch)))
    bx = np.linspace(0.0, W, nbx + 1)
    by = np.linspace(0.0, H, nby + 1)
    bx[-1], by[-1] = W, H
    side = np.concatenate([
        np.stack([bx, np.zeros_like(bx)], 1), np.stack([bx, np.full_like(bx, H)], 1),
        np.stack([np.zeros_like(by[1:-1]), by[1:-1]], 1), np.stack([np.full_like(by[1:-1], W), by[1:-1]], 1)])
    pts = np.ascontiguousarray(np.concatenate([P, side]))
    tri = _delaunay(pts)
    # material by the hex cell that contains the centroid (nearest lattice centre)
    cg = pts[tri].mean(axis=1) - org
    rf = cg[:, 1] / (0.5 * np.sqrt(3.0) * pitch)
    qf = (cg[:, 0] - 0.5 * pitch * rf) / pitch
    # cube rounding
    x, z = qf, rf
    y = -x - z
    rx, ry, rz = np.round(x), np.round(y), np.round(z)
    dx_, dy_, dz_ = np.abs(rx - x), np.abs(ry - y), np.abs(rz - z)
    fx = (dx_ > dy_) & (dx_ > dz_)
    fz = (~fx) & (dz_ > dy_)
    rx = np.where(fx, -ry - rz, rx)
    rz = np.where(fz, -rx - ry, rz)
    cq_, cr_ = rx.astype(np.int64), rz.astype(np.int64)
    mat = np.full(len(tri), 8, dtype=np.int32)
    dmin = np.full(len(tri), 10 ** 9, dtype=np.int64)
    for k, (aq, ar) in enumerate(centres_ax):
        d = hexdist(cq_ - aq, cr_ - ar)
        mat[d <= n] = k
        dmin = np.minimum(dmin, d)
    mat[(dmin == n + 1)] = 7
    return Mesh(pts, tri, mat, float(W), float(H))


def delaunay_mesh(W, H, n_side, seed=0, n_materials=8, jitter=0.35) -> Mesh:
    """Config-5 shape: Delaunay triangulation of a jittered (n_side-1)^2 interior grid plus
    regular boundary points; ~2*n_side^2 triangles; materials assigned at random per triangle."""
    rng = np.random.default_rng(seed)
    hx, hy = W / n_side, H / n_side
    gx = (np.arange(1, n_side) * hx)
    gy = (np.arange(1, n_side) * hy)
    X, Y = np.meshgrid(gx, gy, indexing="xy")
    X = X + (rng.random(X.shape) - 0.5) * 2 * jitter * hx
    Y = Y + (rng.random(Y.shape) - 0.5) * 2 * jitter * hy
    inner = np.stack([X.ravel(), Y.ravel()], 1)
    bx = np.linspace(0.0, W, n_side + 1)
    by = np.linspace(0.0, H, n_side + 1)
    bx[-1], by[-1] = W, H
    side = np.concatenate([
        np.stack([bx, np.zeros_like(bx)], 1), np.stack([bx, np.full_like(bx, H)], 1),
        np.stack([np.zeros_like(by[1:-1]), by[1:-1]], 1), np.stack([np.full_like(by[1:-1], W), by[1:-1]], 1)])
    pts = np.ascontiguousarray(np.concatenate([inner, side]))
    tri = _delaunay(pts)
    mat = rng.integers(0, n_materials, size=len(tri)).astype(np.int32)
    return Mesh(pts, tri, mat, float(W), float(H))
