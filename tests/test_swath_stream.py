"""Host logic of row A1 (no GPU): the swath/tile chunk stream of ND_SWEEP_SWATH, decoded chunk by chunk.

Checks the format csrc/nd_swath.h documents and the properties the kernel relies on: every segment of the
descriptor appears exactly once, in track order, with its FP32 length and its q / Sigma_t / delta row offsets; every
delta-buffer row is owned by exactly one segment and lies in the contiguous row range of that segment's region; the limits
(Kmax, Lmax, head and record capacity) hold; work items cover every (swath, direction) once, in the documented order."""
import numpy as np
import pytest

import paper_2607_01591_b200 as nd
from moc_inputs import make_config


def _decode_and_check(st, mat, seg_offset, seg_region, seg_length, NT, Kmax, Lmax, NC, row_bytes, item_order=0, azim=None):
    blob, ref = st["blob"], st["tile_ref"].astype(np.int64) * 16
    line = NC * row_bytes           # stride of the Sigma_t rows; q rows use one copy per region here (NCq = NC in this builder call)
    T = len(seg_offset) - 1
    cursor = seg_offset[:-1].copy()
    tracks_seen = np.zeros(T, bool)
    total = 0
    for sw in range(st["n_swaths"]):
        trk = st["swath_track"][sw]
        for b in trk[trk >= 0]:
            assert not tracks_seen[b]
            tracks_seen[b] = True
        for ti in range(st["swath_tile0"][sw], st["swath_tile0"][sw + 1]):
            c = blob[ref[ti, 0]:ref[ti + 1, 0]]
            hdr = c[:16].view(np.uint32)
            L, nseg = int(hdr[0] & 0xffff), int(hdr[0] >> 16)
            o_rg = 16 * int(hdr[1])
            head = int(hdr[2])
            assert head == ref[ti, 1] and head % 16 == 0 and head <= st["max_head_bytes"]
            assert hdr[3] == len(c) == head + 16 * nseg and 16 * nseg <= st["max_rec_bytes"]
            assert 1 <= L <= Lmax and 1 <= nseg <= NT * Kmax
            ss = c[16:16 + 2 * (NT + 1)].view(np.uint16).astype(np.int64)
            rg = c[o_rg:o_rg + 8 * L].view(np.uint32).reshape(L, 2).astype(np.int64)
            regions = rg[:, 0]
            co = np.concatenate([rg[:, 1] & 0xffff, [rg[-1, 1] >> 16]])
            assert np.array_equal(rg[:, 1] >> 16, co[1:]), "row ranges of consecutive regions are contiguous"
            assert o_rg + 8 * L <= head
            assert np.all(np.diff(np.diff(co)) <= 0), "regions in descending order of their row counts"
            rec = c[head:head + 16 * nseg].view(np.uint32).reshape(nseg, 4)
            assert ss[0] == 0 and ss[NT] == nseg and np.all(np.diff(ss) >= 0) and np.all(np.diff(ss) <= Kmax)
            assert len(np.unique(regions)) == L
            assert co[0] == 0 and co[L] == nseg and np.all(np.diff(co) >= 1)
            row_region = np.repeat(regions, np.diff(co))          # region-major delta rows: region l owns rows co[l]..co[l+1]-1
            rows_seen = np.zeros(nseg, bool)
            last_row_of_region = {}
            for b in range(NT):
                n = ss[b + 1] - ss[b]
                if trk[b] < 0:
                    assert n == 0
                    continue
                k0 = cursor[trk[b]]
                assert k0 + n <= seg_offset[trk[b] + 1]
                for j in range(n):
                    r = seg_region[k0 + j]
                    lenbits, qoff, soff, doff = rec[ss[b] + j]
                    assert np.uint32(lenbits).view(np.float32) == np.float32(seg_length[k0 + j])
                    assert qoff % line == 0 and regions[qoff // line] == r
                    assert soff == mat[r] * line
                    assert doff % row_bytes == 0
                    row = doff // row_bytes
                    assert row < nseg and not rows_seen[row] and row_region[row] == r
                    rows_seen[row] = True
                    assert last_row_of_region.get(r, -1) < row, "rows of a region in (slot, position) order"
                    last_row_of_region[r] = row
                cursor[trk[b]] += n
            assert rows_seen.all()
            total += nseg
    assert tracks_seen.all()
    assert np.array_equal(cursor, seg_offset[1:]), "every segment exactly once, in order"
    assert total == seg_offset[-1]
    items = st["items"]
    assert len(items) == 2 * st["n_swaths"]
    assert sorted(map(tuple, items[:, :2])) == sorted((s, d) for s in range(st["n_swaths"]) for d in (0, 1))
    if item_order == 0:
        assert np.all(np.diff(items[:, 2]) <= 0), "most expensive first"
    else:
        # angle by angle; inside an angle every forward item in swath order, then every backward item
        sw_angle = np.array([azim[t[t >= 0][0]] if azim is not None and (t >= 0).any() else 0 for t in st["swath_track"]])
        key = [(sw_angle[s], d, s) for s, d in items[:, :2]]
        assert key == sorted(key)


@pytest.mark.parametrize("lag,item_order", [(-1.0, 0), (0.0, 1), (4.0, 0), (1e9, 1)])
@pytest.mark.parametrize("NT,Kmax,Lmax,NC,row_bytes", [(19, 16, 64, 1, 208), (64, 8, 96, 4, 32), (28, 16, 92, 1, 144), (3, 2, 4, 1, 16)])
def test_stream_of_a_traced_problem(NT, Kmax, Lmax, NC, row_bytes, lag, item_order):
    prob = make_config(2, scale=0.12)
    m = prob.mesh
    tr = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    st = nd.nd_swath_stream_build(m.material, prob.xs.sigma_t.shape[0], tr.seg_offset, tr.seg_region, tr.seg_length,
                                  NT, Kmax, Lmax, NC, row_bytes, tr.track_azim, tr.ends, lag_segments=lag, item_order=item_order)
    _decode_and_check(st, m.material, tr.seg_offset, tr.seg_region, tr.seg_length, NT, Kmax, Lmax, NC, row_bytes, item_order, tr.track_azim)
    assert 0.3 < st["lockstep_efficiency"] <= 1.0
    # swaths hold tracks of ONE angle, adjacent in the perpendicular coordinate
    for trk in st["swath_track"]:
        t = trk[trk >= 0]
        assert len(set(tr.track_azim[t])) == 1
    tr.destroy()


def test_stream_without_geometry_and_with_degenerate_tracks():
    rng = np.random.default_rng(4)
    R, T = 5, 23
    counts = rng.integers(0, 40, size=T)
    counts[[0, 7, 22]] = 0
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    seg_region = rng.integers(0, R, size=off[-1]).astype(np.int32)      # a track may re-enter a region
    seg_length = rng.uniform(1e-3, 1.0, size=off[-1])
    mat = rng.integers(0, 3, size=R).astype(np.int32)
    for NT, Kmax, Lmax, NC in [(8, 4, 3, 1), (8, 16, 5, 4), (1, 1, 1, 1)]:
        for lag in (-1.0, 2.0):
            st = nd.nd_swath_stream_build(mat, 3, off, seg_region, seg_length, NT, Kmax, Lmax, NC, 32, lag_segments=lag)
            _decode_and_check(st, mat, off, seg_region, seg_length, NT, Kmax, Lmax, NC, 32)


def test_stream_rejects_bad_parameters():
    off = np.array([0, 2], np.int64)
    args = (np.zeros(1, np.int32), 1, off, np.zeros(2, np.int32), np.ones(2))
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        nd.nd_swath_stream_build(*args, 6, 4, 4, 4, 32)        # NT % NC != 0
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        nd.nd_swath_stream_build(*args, 8, 4, 70000, 1, 208)   # region window exceeds 16 bits
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        nd.nd_swath_stream_build(*args, 8, 4, 4, 1, 20)        # row_bytes not a multiple of 16
