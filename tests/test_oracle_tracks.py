"""Pins for the oracle's track laydown (R-T), links (O-3), ray walk (R-W) and track volumes (O-5).

Nothing here re-types the oracle's formulas: the laydown is pinned by integer/geometric invariants,
the walker by brute-force clipping of every track against every triangle.  (CPU only.)
"""
import numpy as np
import pytest

import oracle
from moc_inputs import make_config, rect_tri_mesh, pin_cell_mesh, delaunay_mesh

CASES = [
    ("rect", lambda: rect_tri_mesh(2.0, 1.5, 5, 4, seed=1, jitter=0.3), (0, 0, 0, 0), 16, 0.05),
    ("rect_refl", lambda: rect_tri_mesh(1.3, 2.1, 4, 6, seed=2, jitter=0.25), (1, 1, 1, 1), 32, 0.04),
    ("pin", lambda: pin_cell_mesh(seed=7), (1, 0, 1, 0), 8, 0.1),
    ("delaunay", lambda: delaunay_mesh(3.0, 3.0, 12, seed=5), (1, 1, 0, 0), 24, 0.03),
]


def _gen(case):
    name, mk, bc, na, sp = case
    m = mk()
    return m, bc, na, sp, oracle.generate_tracks(m.xy, m.tri, m.W, m.H, bc, na, sp)


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_laydown_invariants(case):
    m, bc, na, sp, tr = _gen(case)
    nh = na // 2
    T = tr.n_tracks
    assert T == int((tr.azim_nx + tr.azim_ny).sum())
    # azimuthal weights: every track angle stands for two directions; all N_a directions sum to one
    assert abs(2.0 * tr.azim_weight.sum() - 1.0) < 1e-14
    assert np.all(tr.azim_spacing <= sp * (1 + 1e-12))
    d = tr.ends[:, 2:] - tr.ends[:, :2]
    L = np.hypot(d[:, 0], d[:, 1])
    assert np.all(d[:, 1] > 0), "all forward directions point upward"
    for j in range(nh):
        sel = tr.track_azim == j
        # cyclic tracks tile the rectangle: spacing x total length = area, per angle
        assert abs(tr.azim_spacing[j] * L[sel].sum() - m.W * m.H) < 1e-12 * m.W * m.H
        ang = np.arctan2(d[sel, 1], d[sel, 0])
        assert np.allclose(ang, tr.azim_phi[j], atol=1e-12)
        assert np.allclose(tr.track_weight[sel], tr.azim_weight[j] * tr.azim_spacing[j], rtol=1e-15)
        # complement angles mirror each other
        assert abs(tr.azim_phi[j] + tr.azim_phi[nh - 1 - j] - np.pi) < 1e-12
    # no end point is a corner; all end points lie on the sides
    on_side = lambda p: ((p[:, 0] == 0) | (p[:, 0] == m.W)) ^ ((p[:, 1] == 0) | (p[:, 1] == m.H))
    assert np.all(on_side(tr.ends[:, :2])) and np.all(on_side(tr.ends[:, 2:]))


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_links_are_a_perfect_matching(case):
    m, bc, na, sp, tr = _gen(case)
    T = tr.n_tracks
    nh = na // 2
    side_of = lambda p: 0 if p[0] == 0 else 1 if p[0] == m.W else 2 if p[1] == 0 else 3
    targets = set()
    for t in range(T):
        for d in (0, 1):
            lk = int(tr.link[t, d])
            exit_pt = tr.ends[t, 2:] if d == 0 else tr.ends[t, :2]
            if bc[side_of(exit_pt)] == 0:
                assert lk == -1
                continue
            assert 0 <= lk < 2 * T
            t2, d2 = lk // 2, lk % 2
            assert tr.track_azim[t2] == nh - 1 - tr.track_azim[t], "reflection maps an angle to its complement"
            entry_pt = tr.ends[t2, :2] if d2 == 0 else tr.ends[t2, 2:]
            assert np.abs(entry_pt - exit_pt).max() <= 1e-12 * max(m.W, m.H)
            # time reversal: the reversed partner links back to the reversed self
            assert int(tr.link[t2, 1 - d2]) == 2 * t + (1 - d)
            assert lk not in targets
            targets.add(lk)
            # specular reflection: the tangential component is kept, the normal one flips
            u = (tr.ends[t, 2:] - tr.ends[t, :2]) * (1 if d == 0 else -1)
            v = (tr.ends[t2, 2:] - tr.ends[t2, :2]) * (1 if d2 == 0 else -1)
            u, v = u / np.hypot(*u), v / np.hypot(*v)
            if side_of(exit_pt) in (0, 1):
                assert abs(u[0] + v[0]) < 1e-12 and abs(u[1] - v[1]) < 1e-12
            else:
                assert abs(u[0] - v[0]) < 1e-12 and abs(u[1] + v[1]) < 1e-12
    # every incoming end on a reflective side is fed by exactly one outgoing end
    n_refl_ends = 0
    for t in range(T):
        for d in (0, 1):
            entry_pt = tr.ends[t, :2] if d == 0 else tr.ends[t, 2:]
            n_refl_ends += bc[side_of(entry_pt)] != 0
    assert len(targets) == n_refl_ends


def _brute_force_chords(m, p0, p1):
    """Chord of the line p0->p1 inside every triangle by half-plane clipping (independent of any mesh walk)."""
    L = np.hypot(*(p1 - p0))
    u = (p1 - p0) / L
    lo = np.zeros(m.n_regions)
    hi = np.full(m.n_regions, L)
    V = m.xy[m.tri]
    for e in range(3):
        A, B = V[:, e], V[:, (e + 1) % 3]
        E = B - A
        c0 = E[:, 0] * (p0[1] - A[:, 1]) - E[:, 1] * (p0[0] - A[:, 0])
        c1 = E[:, 0] * u[1] - E[:, 1] * u[0]
        with np.errstate(divide="ignore", invalid="ignore"):
            lam = -c0 / c1
        lo = np.where(c1 > 0, np.maximum(lo, lam), lo)
        hi = np.where(c1 < 0, np.minimum(hi, lam), hi)
        hi = np.where((c1 == 0) & (c0 < 0), -1.0, hi)
    return np.maximum(hi - lo, 0.0)


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_ray_walk_against_brute_force_clipping(case):
    m, bc, na, sp, tr = _gen(case)
    worst = 0.0
    for t in range(tr.n_tracks):
        chords = _brute_force_chords(m, tr.ends[t, :2], tr.ends[t, 2:])
        k0, k1 = tr.seg_offset[t], tr.seg_offset[t + 1]
        got = np.zeros(m.n_regions)
        np.add.at(got, tr.seg_region[k0:k1], tr.seg_length[k0:k1])
        worst = max(worst, np.abs(got - chords).max())
        # a convex cell is crossed at most once
        assert len(np.unique(tr.seg_region[k0:k1])) == k1 - k0
        # segments are ordered along the track: cumulative midpoints lie inside their triangles
        assert np.all(tr.seg_length[k0:k1] > 0)
    assert worst < 1e-12


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_segments_are_in_travel_order(case):
    m, bc, na, sp, tr = _gen(case)
    for t in range(0, tr.n_tracks, 3):
        k0, k1 = tr.seg_offset[t], tr.seg_offset[t + 1]
        p0, p1 = tr.ends[t, :2], tr.ends[t, 2:]
        L = np.hypot(*(p1 - p0))
        u = (p1 - p0) / L
        mid = np.cumsum(tr.seg_length[k0:k1]) - 0.5 * tr.seg_length[k0:k1]
        pts = p0[None, :] + mid[:, None] * u[None, :]
        V = m.xy[m.tri[tr.seg_region[k0:k1]]]
        for e in range(3):
            A, B = V[:, e], V[:, (e + 1) % 3]
            cr = (B[:, 0] - A[:, 0]) * (pts[:, 1] - A[:, 1]) - (B[:, 1] - A[:, 1]) * (pts[:, 0] - A[:, 0])
            assert np.all(cr > -1e-12)
        assert abs(tr.seg_length[k0:k1].sum() - L) < 1e-12 * L


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_track_volumes(case):
    m, bc, na, sp, tr = _gen(case)
    assert abs(tr.volume.sum() - m.W * m.H) < 1e-12 * m.W * m.H
    vol = oracle.track_volumes(m.n_regions, tr.seg_offset, tr.seg_region, tr.seg_length, tr.track_weight)
    assert np.array_equal(vol, tr.volume)


def test_track_volumes_converge_to_true_areas():
    m = pin_cell_mesh(seed=3)
    a = m.areas()
    err = []
    for sp in (0.1, 0.02, 0.004):
        tr = oracle.generate_tracks(m.xy, m.tri, m.W, m.H, (1, 1, 1, 1), 16, sp)
        err.append(np.sqrt(np.mean(((tr.volume - a) / a) ** 2)))
    assert err[0] > err[1] > err[2] and err[2] < 5e-3


@pytest.mark.parametrize("idx,rms_max", [(1, 0.15), (2, 0.02)])
def test_config_track_counts_and_volume_error(idx, rms_max):
    """Track counts follow from R-T alone (SURVEY.md section 8 size table: 68 and 8,752)."""
    p = make_config(idx)
    tr = oracle.generate_tracks(p.mesh.xy, p.mesh.tri, p.mesh.W, p.mesh.H, p.bc, p.n_azim, p.spacing)
    assert tr.n_tracks == {1: 68, 2: 8752}[idx]
    a = p.mesh.areas()
    assert np.sqrt(np.mean(((tr.volume - a) / a) ** 2)) < rms_max
    assert np.all(tr.link >= 0)


def test_bad_arguments_are_rejected():
    m = rect_tri_mesh(1.0, 1.0, 2, 2)
    with pytest.raises(RuntimeError):
        oracle.generate_tracks(m.xy, m.tri, m.W, m.H, (1, 1, 1, 1), 6, 0.1)      # N_a not divisible by 4
    with pytest.raises(RuntimeError):
        oracle.generate_tracks(m.xy, m.tri, m.W, m.H, (1, 1, 1, 1), 8, -1.0)
    with pytest.raises(RuntimeError):
        oracle.generate_tracks(m.xy, m.tri[:-1], m.W, m.H, (1, 1, 1, 1), 8, 0.1)  # hole -> interior boundary edge
