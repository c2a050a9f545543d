"""Pins for the oracle's CMFD step (oracle/cmfd.py, moc_oracle.c O-9, C-1..C-9).  CPU only.

The paper names the step (Algorithm 1 line 5) and gives no numbers; what fixes the implementation is
mathematics: exact per-cell balance of the tallied currents, exact coarse balance at the collapsed flux, the closed-form
infinite-medium eigenvalue, a library eigen-decomposition, and the fact that a consistent CMFD leaves the fixed point of
the unaccelerated iteration where it is while reaching it in far fewer sweeps.
"""
import numpy as np
import pytest

import oracle
from oracle import cmfd
from moc_inputs import make_config, rect_tri_mesh, tabuchi_yamamoto, homogeneous_xs, make_xs
from moc_inputs.coarse import cartesian_cells, cartesian_coupling


def _tracks(m, bc, na, sp):
    return oracle.generate_tracks(m.xy, m.tri, m.W, m.H, bc, na, sp)


def _problem(bc, seed, G=3, nx=8, ny=6, W=4.0, H=3.0, n_materials=3, jitter=0.25):
    m = rect_tri_mesh(W, H, nx, ny, seed=seed, jitter=jitter, n_materials=n_materials)
    xs = make_xs(G, [True, False, True][:n_materials], seed, sigt_range=(0.3, 1.2), c_range=(0.5, 0.9), n_up=1)
    tr = _tracks(m, bc, 16, 0.05)
    ps, pw = tabuchi_yamamoto(3)
    return m, xs, tr, ps, pw


@pytest.mark.parametrize("bc", [(1, 1, 1, 1), (0, 0, 0, 0), (0, 1, 1, 0)])
def test_cell_balance_of_the_tallied_currents(bc):
    """C-3: for every coarse cell and group, the tallies of its regions and the net currents through its surfaces and
    boundary ends telescope to zero -- with an arbitrary source and an arbitrary incoming boundary flux."""
    m, xs, tr, ps, pw = _problem(bc, seed=11)
    rng = np.random.default_rng(5)
    R, G, T, P = m.n_regions, xs.n_groups, tr.n_tracks, len(ps)
    Q = rng.uniform(0.05, 1.0, (R, G))
    psi = rng.uniform(0.0, 0.5, (T, 2, P, G))
    cell = cartesian_cells(m, 3, 2)
    lo, hi = cmfd.coarse_surfaces(tr.seg_offset, tr.seg_region, cell, tr.link)
    assert len(lo) >= 7 and np.all(lo < hi)
    _, _, tally = oracle.sweep(m.material, xs.sigma_t, ps, pw, tr.seg_offset, tr.seg_region, tr.seg_length,
                               tr.track_weight, tr.link, tr.volume, Q, psi)
    Js, Jv, Jr = cmfd.sweep_currents(m.material, xs.sigma_t, ps, pw, tr.seg_offset, tr.seg_region, tr.seg_length,
                                     tr.track_weight, tr.link, Q, psi, cell, 6, lo, hi)
    net = np.zeros((6, G))
    np.add.at(net, cell, tally)
    np.add.at(net, lo, Js)
    np.add.at(net, hi, -Js)
    net += Jv + Jr
    scale = np.abs(tally).sum() / 6
    assert np.max(np.abs(net)) < 1e-12 * scale
    # vacuum ends only where a side is vacuum, reflective ends only where one is reflective
    assert (np.abs(Jv).max() > 0) == (0 in bc) and (np.abs(Jr).max() > 0) == (1 in bc)
    # one coarse cell: no interior surface, everything leaves through the boundary ends
    one = np.zeros(R, np.int32)
    l1, h1 = cmfd.coarse_surfaces(tr.seg_offset, tr.seg_region, one, tr.link)
    assert len(l1) == 0
    Js1, Jv1, Jr1 = cmfd.sweep_currents(m.material, xs.sigma_t, ps, pw, tr.seg_offset, tr.seg_region, tr.seg_length,
                                        tr.track_weight, tr.link, Q, psi, one, 1, l1, h1)
    assert np.allclose(tally.sum(0) + Jv1[0] + Jr1[0], 0.0, atol=1e-12 * scale * 6)
    assert np.allclose(Jv1[0] + Jr1[0], (Jv + Jr).sum(0), rtol=1e-11)


def test_coarse_balance_at_the_collapsed_flux():
    """C-4..C-7: applied to the collapsed flux, the coarse operator returns exactly what the fine mesh says -- removal
    minus in-scatter plus the net leakage the sweep tallied (reflective-end imbalance excluded) -- and the fission
    operator returns the fine-mesh emission.  A wrong sign or orientation in D-tilde, a transposed scattering matrix
    or a missing volume fails this."""
    bc = (0, 1, 1, 0)
    m, xs, tr, ps, pw = _problem(bc, seed=23, G=4)
    rng = np.random.default_rng(9)
    R, G, T, P = m.n_regions, xs.n_groups, tr.n_tracks, len(ps)
    phi_old = rng.uniform(0.5, 1.5, (R, G))
    psi = rng.uniform(0.0, 0.3, (T, 2, P, G))
    Q = oracle.source(m.material, xs.sigma_s, xs.nu_sigma_f, xs.chi, phi_old, 0.9)
    phi, _, tally = oracle.sweep(m.material, xs.sigma_t, ps, pw, tr.seg_offset, tr.seg_region, tr.seg_length,
                                 tr.track_weight, tr.link, tr.volume, Q, psi)
    nxc, nyc = 4, 3
    cell = cartesian_cells(m, nxc, nyc)
    NC = nxc * nyc
    lo, hi = cmfd.coarse_surfaces(tr.seg_offset, tr.seg_region, cell, tr.link)
    Js, Jv, Jr = cmfd.sweep_currents(m.material, xs.sigma_t, ps, pw, tr.seg_offset, tr.seg_region, tr.seg_length,
                                     tr.track_weight, tr.link, Q, psi, cell, NC, lo, hi)
    co = cmfd.collapse(m.material, xs.sigma_t, xs.sigma_s, xs.nu_sigma_f, xs.chi, tr.volume, phi, cell, NC)
    A, B, Dhat, Dtil, alpha = cmfd.coarse_operators(co, lo, hi, cartesian_coupling(m, nxc, nyc)(lo, hi), Js, Jv)
    assert np.any(Dhat > 0) and np.all(Dhat >= 0)
    x = co["Phi"].reshape(-1)
    # fine-mesh statement of the same balance
    mat = m.material
    removal = tr.volume[:, None] * xs.sigma_t[mat] * phi
    inscat = tr.volume[:, None] * np.einsum("rgh,rh->rg", xs.sigma_s[mat], phi)
    emission = tr.volume[:, None] * xs.chi[mat] * np.einsum("rg,rg->r", xs.nu_sigma_f[mat], phi)[:, None]
    lhs_fine, rhs_fine = np.zeros((NC, G)), np.zeros((NC, G))
    np.add.at(lhs_fine, cell, removal - inscat - tally)      # -tally = net leakage out of the region
    np.add.at(rhs_fine, cell, emission)
    lhs_fine -= Jr                                            # the coarse system takes reflective ends as J = 0
    scale = np.abs(removal).sum() / NC
    assert np.max(np.abs((A @ x).reshape(NC, G) - lhs_fine)) < 1e-11 * scale
    assert np.max(np.abs((B @ x).reshape(NC, G) - rhs_fine)) < 1e-11 * scale
    assert np.allclose(co["V"].sum(), tr.volume.sum(), rtol=1e-13)


def test_coarse_eigen_against_a_dense_eigendecomposition():
    rng = np.random.default_rng(3)
    n = 24
    A = np.diag(rng.uniform(2.0, 3.0, n)) - rng.uniform(0.0, 0.05, (n, n))
    B = np.outer(rng.uniform(0.1, 1.0, n), rng.uniform(0.1, 1.0, n)) * 0.2 + rng.uniform(0.0, 0.02, (n, n))
    ev, vec = np.linalg.eig(np.linalg.solve(A, B))
    i = int(np.argmax(ev.real))
    k, x = cmfd.coarse_eigen(A, B, np.ones((n, 1)), 1.0)
    assert abs(k - ev[i].real) < 1e-11
    v = np.abs(vec[:, i].real)
    assert np.allclose(x[:, 0] / x[:, 0].sum(), v / v.sum(), rtol=1e-8)
    assert np.isclose(np.sum(B @ x[:, 0]), np.sum(B @ np.ones(n)), rtol=1e-12)     # keeps the fission production


def test_infinite_medium_in_a_handful_of_sweeps():
    """Homogeneous, all sides reflective, ONE coarse cell: the coarse problem is the G x G infinite-medium problem, so
    the first CMFD step already returns k_inf = nuSf^T (diag St - S)^-1 chi (closed form); the plain iteration needs
    hundreds of sweeps for the same digits."""
    G = 5
    xs = homogeneous_xs(G, 105, n_up=2, sigt_range=(0.8, 2.5), c_range=(0.3, 0.8))
    m = rect_tri_mesh(1.0, 0.8, 3, 3, seed=8, jitter=0.2)
    tr = _tracks(m, (1, 1, 1, 1), 8, 0.1)
    ps, pw = tabuchi_yamamoto(2)
    k_inf = float(xs.nu_sigma_f[0] @ np.linalg.solve(np.diag(xs.sigma_t[0]) - xs.sigma_s[0], xs.chi[0]))
    args = (m.material, xs.sigma_t, xs.sigma_s, xs.nu_sigma_f, xs.chi, ps, pw, tr.seg_offset, tr.seg_region,
            tr.seg_length, tr.track_weight, tr.link, tr.volume)
    k, phi, psi, hist = cmfd.power_iteration_cmfd(*args, np.zeros(m.n_regions, np.int32), 1, lambda lo, hi: np.zeros(len(lo)), 3)
    assert abs(hist[0] - k_inf) < 1e-10 and abs(k - k_inf) < 1e-10
    _, _, _, plain = cmfd.power_iteration_cmfd(*args, np.zeros(m.n_regions, np.int32), 1, lambda lo, hi: np.zeros(len(lo)), 3,
                                               accelerate=False)
    assert abs(plain[-1] - k_inf) > 1e-4


@pytest.mark.parametrize("bc,coarse", [((1, 1, 1, 1), (4, 3)), ((0, 1, 1, 0), (8, 6)), ((0, 0, 0, 0), (8, 6))])
def test_cmfd_keeps_the_fixed_point_and_needs_fewer_sweeps(bc, coarse):
    """The accelerated and the plain iteration converge to the same k and the same flux; CMFD gets there in at most a
    third of the sweeps.  The 8 x 6 cm domain has boundary vertices at whole centimetres, where some cyclic tracks end
    exactly: reflective hand-overs between different coarse cells occur and must be counted as surface crossings, or
    the fixed point moves by ~1e-4 in k.  (Coarse cells of 1-2 cm; 4 x 3 cm cells, ~4 mean free paths, make the
    undamped CMFD diverge -- the known limit of the method, not covered here.)"""
    m, xs, tr, ps, pw = _problem(bc, seed=31, G=3, nx=8, ny=6, W=8.0, H=6.0)
    args = (m.material, xs.sigma_t, xs.sigma_s, xs.nu_sigma_f, xs.chi, ps, pw, tr.seg_offset, tr.seg_region,
            tr.seg_length, tr.track_weight, tr.link, tr.volume)
    cell = cartesian_cells(m, *coarse)
    coup = cartesian_coupling(m, *coarse)
    kp, phip, _, hp = cmfd.power_iteration_cmfd(*args, cell, coarse[0] * coarse[1], coup, 3000, accelerate=False, tol_k=1e-11)
    # the plain loop is O-8 itself
    k8, phi8, _, h8 = oracle.power_iteration(*args, 25)
    assert np.allclose(hp[:25], h8, rtol=0, atol=1e-13)
    ka, phia, _, ha = cmfd.power_iteration_cmfd(*args, cell, coarse[0] * coarse[1], coup, 3000, accelerate=True, tol_k=1e-11)
    assert abs(ka - kp) < 2e-9, (ka, kp)
    fa = phia / oracle.fission_rate(m.material, xs.nu_sigma_f, tr.volume, phia)
    fp = phip / oracle.fission_rate(m.material, xs.nu_sigma_f, tr.volume, phip)
    assert np.max(np.abs(fa - fp) / fp) < 2e-6
    assert len(ha) * 3 <= len(hp), (len(ha), len(hp))


def test_boundary_flux_prolongation_uses_the_cell_the_chain_enters():
    """The psi half of C-9: after one accelerated iteration the stored boundary flux of chain (t, d) -- the flux that will
    ENTER track t travelling in direction d -- is the plain iteration's value times the flux ratio of the coarse cell that
    GEOMETRICALLY contains the chain's entry point (the start point of the track for d = 0, its end point for d = 1).
    The cell is located here from the track end coordinates, not from the segment list, on a mesh whose grid lines
    coincide with the overlay (no jitter), and the ratio is read off the oracle's own phi (accelerated / plain).  A chain
    scaled with the cell at its other end, or with the cell its feeding chain came from, fails."""
    bc = (1, 0, 1, 1)                                   # reflective left, bottom, top; vacuum right
    W, H, nx, ny = 4.0, 3.0, 8, 6
    m = rect_tri_mesh(W, H, nx, ny, seed=41, jitter=0.0, n_materials=3)
    xs = make_xs(3, [True, False, True], 41, sigt_range=(0.3, 1.2), c_range=(0.5, 0.9), n_up=1)
    tr = _tracks(m, bc, 16, 0.05)
    ps, pw = tabuchi_yamamoto(3)
    ncx, ncy = 4, 3                                     # overlay lines on mesh grid lines: every triangle lies in one cell
    cell = cartesian_cells(m, ncx, ncy)
    args = (m.material, xs.sigma_t, xs.sigma_s, xs.nu_sigma_f, xs.chi, ps, pw, tr.seg_offset, tr.seg_region, tr.seg_length,
            tr.track_weight, tr.link, tr.volume, cell, ncx * ncy, cartesian_coupling(m, ncx, ncy))
    # a state three plain iterations from the flat start: the flux is far from converged, so the ratios differ by cell
    k0, phi0, psi0, _ = cmfd.power_iteration_cmfd(*args, 3, accelerate=False)
    _, phi_p, psi_p, _ = cmfd.power_iteration_cmfd(*args, 1, state=(k0, phi0, psi0), accelerate=False)
    _, phi_a, psi_a, _ = cmfd.power_iteration_cmfd(*args, 1, state=(k0, phi0, psi0), accelerate=True)
    ratio_r = phi_a / phi_p                              # the phi half of C-9: constant inside a coarse cell
    ratio_c = np.zeros((ncx * ncy, xs.n_groups))
    for c in range(ncx * ncy):
        rr = ratio_r[cell == c]
        assert len(rr) > 0 and np.abs(rr - rr[0]).max() < 1e-12
        ratio_c[c] = rr[0]
    assert (ratio_c.max(0) - ratio_c.min(0)).min() > 1e-3, "the cells' ratios must differ for the pin to bite"
    # entry point of chain (t, d), nudged into the domain along the direction of travel
    e = tr.ends
    u = e[:, 2:] - e[:, :2]
    u /= np.linalg.norm(u, axis=1)[:, None]
    eps = 1e-7
    pts = np.stack([e[:, :2] + eps * u, e[:, 2:] - eps * u], 1)             # [T][2][xy]
    cx = np.clip((pts[..., 0] / W * ncx).astype(int), 0, ncx - 1)
    cy = np.clip((pts[..., 1] / H * ncy).astype(int), 0, ncy - 1)
    cell_geo = cy * ncx + cx                                                   # [T][2]
    # a track end that sits ON an overlay line (a mesh vertex on the boundary) has no unique geometric cell: left out
    fx, fy = pts[..., 0] / W * ncx, pts[..., 1] / H * ncy
    clear = (np.abs(fx - np.round(fx)) > 1e-5) & (np.abs(fy - np.round(fy)) > 1e-5) | \
            ((np.abs(fx - np.round(fx)) > 1e-5) & ((np.round(fy) == 0) | (np.round(fy) == ncy))) | \
            ((np.abs(fy - np.round(fy)) > 1e-5) & ((np.round(fx) == 0) | (np.round(fx) == ncx)))
    assert clear.mean() > 0.98
    expect = psi_p * ratio_c[cell_geo][:, :, None, :]
    scale = np.abs(psi_p).max()
    assert scale > 0 and np.abs(psi_a - expect)[clear].max() < 1e-12 * scale
    # the pin bites: scaling with the cell at the chain's OTHER end is off by orders of magnitude more than the bar
    wrong = psi_p * ratio_c[cell_geo[:, ::-1]][:, :, None, :]
    assert np.abs(psi_a - wrong)[clear].max() > 1e-6 * scale
