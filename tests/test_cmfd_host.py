"""Host logic of the CMFD step (no GPU): nd_cmfd_surfaces (C-2 of DESIGN.md 8d) against the oracle's list and against
a brute-force enumeration, and its argument checks."""
import numpy as np
import pytest

import oracle
from oracle import cmfd
import paper_2607_01591_b200 as nd
from moc_inputs import make_config, rect_tri_mesh
from moc_inputs.coarse import cartesian_cells

CASES = [(1, 1.0, 2, 2, None), (2, 0.15, 4, 3, None), (3, 0.03, 5, 5, None), (4, 0.06, 3, 4, None), (5, 0.0008, 6, 6, None),
         (2, 0.15, 1, 1, None), (2, 0.15, 3, 3, (0, 0, 0, 0)), (3, 0.03, 4, 2, (1, 1, 1, 1))]


@pytest.mark.parametrize("idx,scale,nx,ny,bc", CASES)
def test_surfaces_equal_the_oracles(idx, scale, nx, ny, bc):
    prob = make_config(idx, scale=scale)
    m = prob.mesh
    bc = bc or prob.bc
    otr = oracle.generate_tracks(m.xy, m.tri, m.W, m.H, bc, prob.n_azim, prob.spacing)
    gtr = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, bc, prob.n_azim, prob.spacing)
    cell = cartesian_cells(m, nx, ny)
    lo, hi = nd.nd_cmfd_surfaces(gtr.seg_offset, gtr.seg_region, gtr.link, cell, nx * ny)
    olo, ohi = cmfd.coarse_surfaces(otr.seg_offset, otr.seg_region, cell, otr.link)
    assert np.array_equal(lo, olo) and np.array_equal(hi, ohi)
    assert np.all(lo < hi) and (len(lo) > 0) == (nx * ny > 1)
    gtr.destroy()


def test_surfaces_by_brute_force_with_hand_overs_and_empty_tracks():
    """Random segment lists (no geometry): plain loops over every consecutive pair and every linked hand-over."""
    rng = np.random.default_rng(12)
    R, T, C = 40, 30, 7
    counts = rng.integers(0, 25, size=T)
    counts[[3, 11]] = 0
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    sr = rng.integers(0, R, size=off[-1]).astype(np.int32)
    cell = rng.integers(0, C, size=R).astype(np.int32)
    perm = rng.permutation(2 * T)
    link = np.full(2 * T, -1, np.int32)
    link[perm[:25]] = perm[30:55][rng.permutation(25)].astype(np.int32)         # 25 linked exits, distinct targets
    want = set()
    for t in range(T):
        for k in range(off[t] + 1, off[t + 1]):
            a, b = cell[sr[k - 1]], cell[sr[k]]
            if a != b:
                want.add((min(a, b), max(a, b)))
        if off[t + 1] > off[t]:
            for d in (0, 1):
                lk = link[2 * t + d]
                if lk < 0:
                    continue
                t2, d2 = lk // 2, lk % 2
                if off[t2 + 1] == off[t2]:
                    continue
                a = cell[sr[off[t + 1] - 1 if d == 0 else off[t]]]
                b = cell[sr[off[t2] if d2 == 0 else off[t2 + 1] - 1]]
                if a != b:
                    want.add((min(a, b), max(a, b)))
    lo, hi = nd.nd_cmfd_surfaces(off, sr, link.reshape(T, 2), cell, C, n_regions=R)
    assert list(zip(lo.tolist(), hi.tolist())) == sorted(want)


def test_surfaces_argument_checks():
    off = np.array([0, 2, 3], np.int64)
    sr = np.array([0, 1, 1], np.int32)
    link = np.full((2, 2), -1, np.int32)
    cell = np.array([0, 1], np.int32)
    lo, hi = nd.nd_cmfd_surfaces(off, sr, link, cell, 2)
    assert lo.tolist() == [0] and hi.tolist() == [1]
    with pytest.raises(nd.NdError, match="ND_ERR_RANGE"):
        nd.nd_cmfd_surfaces(off, sr, link, np.array([0, 2], np.int32), 2)
    with pytest.raises(nd.NdError, match="ND_ERR_RANGE"):
        nd.nd_cmfd_surfaces(off, np.array([0, 5, 1], np.int32), link, cell, 2)
    with pytest.raises(nd.NdError, match="ND_ERR_RANGE"):
        nd.nd_cmfd_surfaces(off, sr, np.array([[9, -1], [-1, -1]], np.int32), cell, 2)
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        nd.nd_cmfd_surfaces(off, sr, link, cell, 0)
