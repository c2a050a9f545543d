"""CPU-only checks of the product library: it loads, exports every symbol include/nd.h declares, validates
its inputs, and its host ray tracer (nd_tracks_generate) is BIT-EXACT against the independent oracle tracer.
No compute entry point is called here (no GPU)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
import paper_2607_01591_b200 as nd
from moc_inputs import make_config, rect_tri_mesh, pin_cell_mesh, delaunay_mesh, tabuchi_yamamoto, homogeneous_xs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "nd.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nd_[a-z_0-9]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    L = nd.lib()
    for name in sorted(declared):
        assert hasattr(L, name), f"{name} is declared in include/nd.h but not exported"
    assert declared == set(nd.EXPORTS), declared ^ set(nd.EXPORTS)
    assert nd.nd_version() >> 16 == 2


def test_no_product_file_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_01591_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                txt = open(os.path.join(base, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "moc_oracle" not in txt, f


CASES = [
    ("rect", lambda: rect_tri_mesh(2.0, 1.5, 5, 4, seed=1, jitter=0.3), (0, 0, 0, 0), 16, 0.05),
    ("rect_refl", lambda: rect_tri_mesh(1.3, 2.1, 4, 6, seed=2, jitter=0.25), (1, 1, 1, 1), 32, 0.04),
    ("pin", lambda: pin_cell_mesh(seed=7), (1, 0, 1, 0), 8, 0.1),
    ("delaunay", lambda: delaunay_mesh(3.0, 3.0, 12, seed=5), (1, 1, 0, 0), 24, 0.03),
    ("cfg1", lambda: make_config(1).mesh, (1, 1, 1, 1), 8, 0.1),
    ("cfg2_small", lambda: make_config(2, scale=0.1).mesh, (1, 1, 1, 1), 32, 0.05),
    ("cfg3_small", lambda: make_config(3, scale=0.05).mesh, (1, 0, 1, 0), 64, 0.02),
    ("cfg4_small", lambda: make_config(4, scale=0.08).mesh, (0, 0, 0, 0), 48, 0.03),
    ("cfg5_small", lambda: make_config(5, scale=0.002).mesh, (1, 0, 1, 0), 64, 0.01),
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_tracks_bit_exact_against_oracle(case):
    _, mk, bc, na, sp = case
    m = mk()
    a = oracle.generate_tracks(m.xy, m.tri, m.W, m.H, bc, na, sp)
    b = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, bc, na, sp)
    assert b.n_tracks == a.n_tracks and b.n_segments == a.n_segs
    for name_b, name_a in [("seg_offset", "seg_offset"), ("seg_region", "seg_region"), ("seg_length", "seg_length"),
                           ("track_weight", "track_weight"), ("link", "link"), ("track_azim", "track_azim"),
                           ("ends", "ends"), ("volume", "volume"), ("azim_phi", "azim_phi"),
                           ("azim_weight", "azim_weight"), ("azim_spacing", "azim_spacing")]:
        x, y = getattr(b, name_b), getattr(a, name_a)
        assert x.dtype == y.dtype and x.shape == y.shape, name_b
        assert x.tobytes() == y.tobytes(), f"{name_b} differs from the oracle"
    b.destroy()


def test_tracks_thread_count_does_not_change_bits():
    m = delaunay_mesh(3.0, 3.0, 12, seed=5)
    a = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, (1, 1, 0, 0), 24, 0.03, n_threads=1)
    b = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, (1, 1, 0, 0), 24, 0.03, n_threads=4)
    assert a.seg_length.tobytes() == b.seg_length.tobytes() and a.seg_region.tobytes() == b.seg_region.tobytes()


def test_tracks_generate_rejects_bad_input():
    m = rect_tri_mesh(2.0, 1.5, 3, 3, seed=1)
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, (0, 0, 0, 0), 6, 0.05)        # n_azim not a multiple of 4
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, (0, 0, 0, 0), 8, -1.0)
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, (0, 2, 0, 0), 8, 0.05)
    bad = m.tri.copy()
    bad = bad[:-1]                                                                  # a hole: interior edges become boundary
    with pytest.raises(nd.NdError, match="ND_ERR_MESH"):
        nd.nd_tracks_generate(m.xy, bad, m.W, m.H, (0, 0, 0, 0), 8, 0.05)
    flipped = m.tri.copy()
    flipped[0] = flipped[0, ::-1]                                                   # one clockwise triangle
    with pytest.raises(nd.NdError, match="ND_ERR_MESH"):
        nd.nd_tracks_generate(m.xy, flipped, m.W, m.H, (0, 0, 0, 0), 8, 0.05)


def _desc_for(m, xs, tr, P=2):
    s, w = tabuchi_yamamoto(P)
    keep = dict(rm=m.material.astype(np.int32), st=xs.sigma_t, ss=xs.sigma_s, nf=xs.nu_sigma_f, ch=xs.chi, ps=s, pw=w,
                so=tr.seg_offset.copy(), sr=tr.seg_region.copy(), sl=tr.seg_length.copy(), tw=tr.track_weight.copy(),
                lk=tr.link.copy())
    d = nd.nd_problem_desc(len(keep["rm"]), xs.n_materials, xs.n_groups, P, tr.n_tracks,
                           *[keep[k].ctypes.data for k in ("rm", "st", "ss", "nf", "ch", "ps", "pw", "so", "sr", "sl", "tw", "lk")],
                           None, None)
    return d, keep


def test_workspace_bytes_and_host_validation_without_a_gpu():
    m = rect_tri_mesh(2.0, 1.5, 3, 3, seed=1)
    m.material[:] = 0
    xs = homogeneous_xs(3, 5)
    tr = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, (1, 1, 1, 1), 8, 0.2)
    d, keep = _desc_for(m, xs, tr)
    L = nd.lib()
    n = C.c_size_t()
    assert L.nd_workspace_bytes(C.byref(d), None, C.byref(n)) == nd.ND_OK
    S, T, R, G, P = tr.n_segments, tr.n_tracks, len(m.tri), 3, 2
    assert n.value >= 8 * S + 2 * 4 * T * 2 * P * G + 12 * R * G
    assert L.nd_workspace_bytes(C.byref(d), None, None) == 1                          # ND_ERR_NULL
    # host-side validation happens before any CUDA call: these fail identically on a CPU box
    h = C.c_void_p()
    fake_ws = C.c_void_p(256 * 4096)
    assert L.nd_problem_create(C.byref(d), None, fake_ws, 16, None, C.byref(h)) == 4  # ND_ERR_WORKSPACE (too small)
    assert L.nd_problem_create(C.byref(d), None, C.c_void_p(256 * 4096 + 8), n.value, None, C.byref(h)) == 4  # misaligned
    keep["sr"][0] = R + 5
    assert L.nd_problem_create(C.byref(d), None, fake_ws, n.value, None, C.byref(h)) == 3  # ND_ERR_RANGE
    assert b"seg_region" in L.nd_last_error(None)
    keep["sr"][0] = 0
    keep["st"][0, 0] = -1.0
    assert L.nd_problem_create(C.byref(d), None, fake_ws, n.value, None, C.byref(h)) == 2  # ND_ERR_INVALID
    keep["st"][0, 0] = 1.0
    keep["lk"][0, 0] = keep["lk"][1, 0] = 2                                             # two ends feed one entry
    assert L.nd_problem_create(C.byref(d), None, fake_ws, n.value, None, C.byref(h)) == 2
    keep["so"][1] = keep["so"][2] + 1                                                   # non-monotone offsets
    assert L.nd_workspace_bytes(C.byref(d), None, C.byref(n)) == 2
    assert h.value is None


def test_cmfd_plan_entry_points_reject_null_arguments_without_a_gpu():
    """Argument checks of the nd_cmfd_* calls (include/nd.h) come before any CUDA call, so they run without a GPU."""
    L = nd.lib()
    n = C.c_size_t()
    k = C.c_double()
    assert L.nd_status_string(L.nd_cmfd_workspace_bytes(None, None, 1, None, 0, C.byref(n))) == b"ND_ERR_NULL"
    assert L.nd_status_string(L.nd_cmfd_workspace_bytes(None, None, 1, None, 0, None)) == b"ND_ERR_NULL"
    h = C.c_void_p()
    ws = (C.c_char * 512)()
    assert L.nd_status_string(L.nd_cmfd_create(None, None, 1, None, 0, None, None, None, None, ws, 512, None, C.byref(h))) == b"ND_ERR_NULL"
    assert L.nd_status_string(L.nd_cmfd_iteration(None, 1, C.byref(k), None, None)) == b"ND_ERR_NULL"
    assert L.nd_status_string(L.nd_cmfd_sweep(None, None, None, None)) == b"ND_ERR_NULL"
    assert L.nd_status_string(L.nd_cmfd_solve(None, 1.0, C.byref(k), None, None, None)) == b"ND_ERR_NULL"
    assert L.nd_status_string(L.nd_cmfd_collapse(None, None, None)) == b"ND_ERR_NULL"
    assert L.nd_status_string(L.nd_cmfd_prolong(None, None)) == b"ND_ERR_NULL"
    assert L.nd_cmfd_destroy(None) == 0
    assert b"NULL" in L.nd_last_error(None)


def test_round2_entry_points_check_their_arguments_without_a_gpu():
    """nd_tracks_generate_resident / nd_tracks_materialise / nd_problem_stream_view / nd_fission_rate_static and the
    seg_on_device field of the descriptor: the argument checks come before any CUDA call."""
    L = nd.lib()
    name = lambda rc: L.nd_status_string(rc)
    assert name(L.nd_tracks_generate_resident(None, 8, 0.1, None, 0, None, None, None, None)) == b"ND_ERR_NULL"
    assert name(L.nd_tracks_materialise(None, None)) == b"ND_ERR_NULL"
    assert name(L.nd_problem_stream_view(None, None)) == b"ND_ERR_NULL"
    one = C.c_void_p(4096)
    assert name(L.nd_fission_rate_static(4, 2, None, one, one, one, one, None)) == b"ND_ERR_NULL"
    assert name(L.nd_fission_rate_static(0, 2, one, one, one, one, one, None)) == b"ND_ERR_INVALID"
    assert name(L.nd_fission_rate_static((1 << 27) + 1, 1, one, one, one, one, one, None)) == b"ND_ERR_RANGE"
    assert b"ND_STATIC_FISSION_MAX_ELEMENTS" in L.nd_last_error(None)
    # host tracks have no device arrays, and materialising them is a no-op
    m = rect_tri_mesh(2.0, 1.5, 3, 3, seed=1)
    m.material[:] = 0
    tr = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, (1, 1, 1, 1), 8, 0.2)
    assert tr.seg_device is None and tr.on_host
    assert L.nd_tracks_materialise(tr._h, None) == nd.ND_OK
    # the descriptor's seg_on_device: 0 or 1, and 1 needs the track geometry
    xs = homogeneous_xs(3, 5)
    d, keep = _desc_for(m, xs, tr)
    h, n = C.c_void_p(), C.c_size_t()
    assert L.nd_workspace_bytes(C.byref(d), None, C.byref(n)) == nd.ND_OK
    fake_ws = C.c_void_p(256 * 4096)
    d.seg_on_device = 2
    assert name(L.nd_problem_create(C.byref(d), None, fake_ws, n.value, None, C.byref(h))) == b"ND_ERR_INVALID"
    d.seg_on_device = 1                                  # _desc_for passes no track_azim / track_ends
    assert name(L.nd_problem_create(C.byref(d), None, fake_ws, n.value, None, C.byref(h))) == b"ND_ERR_INVALID"
    assert b"geometry" in L.nd_last_error(None)
    d.seg_on_device, d.reserved = 0, 7
    assert name(L.nd_problem_create(C.byref(d), None, fake_ws, n.value, None, C.byref(h))) == b"ND_ERR_INVALID"
    assert h.value is None
    tr.destroy()
