"""GPU ray walk (nd_tracks_generate_device) against the oracle's own tracer and the library's host
tracer: tracks, segments, links and volumes must agree BYTE FOR BYTE (rule R-T / R-W)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
import paper_2607_01591_b200 as nd
from moc_inputs import make_config, rect_tri_mesh

pytestmark = pytest.mark.gpu

FIELDS_O = ("seg_offset", "seg_region", "seg_length", "track_weight", "link", "volume")


def _same(a, b, fields):
    for f in fields:
        assert getattr(a, f).tobytes() == getattr(b, f).tobytes(), f"{f} differs"


@pytest.mark.parametrize("idx,scale", [(1, 1.0), (2, 0.3), (3, 0.05), (4, 0.1), (5, 0.002)])
def test_device_walk_is_bit_exact_against_oracle_and_host(idx, scale):
    prob = make_config(idx, scale=scale)
    m = prob.mesh
    o = oracle.generate_tracks(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    h = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    d = nd.nd_tracks_generate_device(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    try:
        assert d.n_segments == o.n_segs == h.n_segments
        _same(d, o, FIELDS_O)
        _same(d, h, FIELDS_O + ("track_azim", "ends", "azim_phi", "azim_weight", "azim_spacing"))
    finally:
        h.destroy()
        d.destroy()


def test_device_walk_in_many_small_batches_and_degenerate_hits():
    # a jittered grid mesh with tracks through vertices' neighbourhoods; a tiny workspace forces many fill batches
    mesh = rect_tri_mesh(2.3, 1.7, 9, 7, seed=5, jitter=0.35)
    bc = (1, 0, 0, 1)
    h = nd.nd_tracks_generate(mesh.xy, mesh.tri, mesh.W, mesh.H, bc, 32, 0.0004)
    d = nd.nd_tracks_generate_device(mesh.xy, mesh.tri, mesh.W, mesh.H, bc, 32, 0.0004, segment_capacity=0)
    try:
        _same(d, h, FIELDS_O)
        assert d.timing["batches"] >= 2 and d.timing["n_segments"] == h.n_segments
    finally:
        h.destroy()
        d.destroy()


def test_device_walk_rejects_a_bad_mesh_and_a_small_workspace():
    mesh = rect_tri_mesh(1.0, 1.0, 3, 3, seed=1, jitter=0.1)
    tri = mesh.tri.copy()
    tri[0] = tri[0][::-1]                      # one clockwise triangle: not a conforming CCW mesh
    with pytest.raises(nd.NdError, match="ND_ERR_MESH"):
        nd.nd_tracks_generate_device(mesh.xy, tri, mesh.W, mesh.H, (1, 1, 1, 1), 8, 0.1)
