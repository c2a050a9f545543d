"""Input generators: meshes are valid conforming triangulations; quadrature constants obey what the
mathematics fixes; cross sections are physically sane.  (CPU only.)"""
import numpy as np
import pytest
from scipy import integrate

from moc_inputs import (make_config, validate_mesh, rect_tri_mesh, tabuchi_yamamoto, delaunay_mesh,
                        homogeneous_xs)


@pytest.mark.parametrize("idx,scale,expect_R", [(1, 1.0, 64), (2, 1.0, 6936), (3, 1.0, 38400), (4, 1.0, None),
                                                (5, 0.02, None)])
def test_config_meshes_valid(idx, scale, expect_R):
    p = make_config(idx, scale)
    validate_mesh(p.mesh)
    if expect_R is not None:
        assert p.mesh.n_regions == expect_R
    assert p.mesh.material.min() >= 0 and p.mesh.material.max() < p.xs.n_materials
    assert len(p.bc) == 4 and p.n_azim % 4 == 0


def test_config4_pins_have_12_triangles_each():
    p = make_config(4)
    # 7 assemblies x 271 pins x 12 triangles, none straddling a cell (materials 0..6 are the assemblies)
    counts = np.bincount(p.mesh.material, minlength=9)
    assert np.all(counts[:7] == 271 * 12)


def test_generators_are_seeded():
    a, b = make_config(2), make_config(2)
    assert np.array_equal(a.mesh.xy, b.mesh.xy) and np.array_equal(a.xs.sigma_s, b.xs.sigma_s)
    m1, m2 = delaunay_mesh(5, 5, 20, seed=3), delaunay_mesh(5, 5, 20, seed=3)
    assert np.array_equal(m1.tri, m2.tri)


def test_validate_mesh_rejects_broken_meshes():
    m = rect_tri_mesh(1.0, 1.0, 3, 3)
    validate_mesh(m)
    bad = rect_tri_mesh(1.0, 1.0, 3, 3)
    bad.tri[0, [1, 2]] = bad.tri[0, [2, 1]]          # clockwise triangle
    with pytest.raises(ValueError):
        validate_mesh(bad)
    hole = rect_tri_mesh(1.0, 1.0, 3, 3)
    hole.tri = hole.tri[1:].copy()
    hole.material = hole.material[1:].copy()
    with pytest.raises(ValueError):
        validate_mesh(hole)


@pytest.mark.parametrize("P,tol", [(2, 6e-4), (3, 6e-5)])
def test_polar_quadrature_matches_bickley_ki3(P, tol):
    s, w = tabuchi_yamamoto(P)
    assert abs(w.sum() - 1.0) < 1e-14
    assert np.all((s > 0) & (s <= 1))
    assert abs((w * s).sum() - np.pi / 4) < 1e-3
    for x in (0.01, 0.1, 0.5, 1.0, 2.0, 5.0):
        ki3, _ = integrate.quad(lambda th: np.sin(th) ** 2 * np.exp(-x / np.sin(th)), 0.0, np.pi / 2)
        assert abs((w * s * np.exp(-x / s)).sum() - ki3) < tol


@pytest.mark.parametrize("idx", [1, 2, 4, 5])
def test_cross_sections_are_physical(idx):
    xs = make_config(idx, 0.02 if idx == 5 else 1.0).xs
    assert np.all(xs.sigma_t > 0) and np.all(xs.sigma_s >= 0) and np.all(xs.nu_sigma_f >= 0)
    out_scatter = xs.sigma_s.sum(axis=1)              # column sums: total scattering out of g'
    assert np.all(out_scatter < xs.sigma_t)           # scattering ratio < 1 -> subcritical without fission
    fissile = xs.nu_sigma_f.sum(axis=1) > 0
    assert fissile.any()
    assert np.allclose(xs.chi[fissile].sum(axis=1), 1.0)
    if idx == 1:
        assert np.all(np.triu(xs.sigma_s, 1) == 0)    # [g_to][g_from]: no upscatter = nothing above the diagonal
        assert np.array_equal(xs.chi[0], [1.0, 0.0])


def test_homogeneous_xs_has_upscatter_when_asked():
    xs = homogeneous_xs(7, 5, n_up=3)
    assert (np.triu(xs.sigma_s[0], 1) > 0).any()
