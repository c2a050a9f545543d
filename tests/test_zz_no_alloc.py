"""nd_fission_rate_static (include/nd.h): the allocation-free fission rate, whose partial sums live in a file-scope __device__
array of the library, against the existing path (nd_source_update's d_fission_rate_out, partial sums in the problem's
workspace) and against the plain FP64 sum, on calls in a row that share the static array.  Collected last on purpose (the
file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import paper_2607_01591_b200 as nd
from gpu_common import make_pair

pytestmark = pytest.mark.gpu

F_RTOL = 1e-12      # the same FP64 products added in another order (the bar of the other FP64 re-ordering checks)


def _inputs(pair, seed):
    p = pair.prob
    rng = np.random.default_rng(seed)
    phi = rng.uniform(0.1, 2.0, size=(pair.R, pair.G))
    vol = pair.gpu.nd_track_volume_get()
    dev = dict(phi=torch.from_numpy(phi).cuda(), mat=torch.from_numpy(np.ascontiguousarray(p.mesh.material, np.int32)).cuda(),
               nusf=torch.from_numpy(np.ascontiguousarray(p.xs.nu_sigma_f, np.float64)).cuda(), vol=torch.from_numpy(vol).cuda())
    plain = float((vol[:, None] * p.xs.nu_sigma_f[p.mesh.material] * phi).sum())
    return dev, plain


def _existing(pair, d_phi):
    _, dF = pair.gpu.nd_source_update(d_phi, 1.0, want_fission_rate=True)
    return float(dF.cpu()[0])


def test_static_fission_rate_matches_the_workspace_path_on_calls_in_a_row():
    big = make_pair(4, 0.1)        # 33 groups, several thousand regions: many partial sums
    small = make_pair(1, 1.0)      # 64 regions x 2 groups: ONE partial sum; the array still holds the big call's others
    try:
        a, plain_a = _inputs(big, 1)
        b, plain_b = _inputs(small, 2)
        assert big.R * big.G > 8 * 4096 and small.R * small.G < 4096
        out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
        results = []
        for dev, pair, plain in ((a, big, plain_a), (b, small, plain_b), (a, big, plain_a), (b, small, plain_b)):
            nd.nd_fission_rate_static(dev["phi"], dev["mat"], dev["nusf"], dev["vol"], d_out=out)
            got = float(out.cpu()[0])
            ref = _existing(pair, dev["phi"])
            assert plain > 0 and abs(got - ref) <= F_RTOL * abs(ref), (got, ref)
            assert abs(got - plain) <= F_RTOL * abs(plain), (got, plain)
            results.append(got)
        # a fixed decomposition: the same input gives the same bits, whatever ran in between
        assert results[0] == results[2] and results[1] == results[3]
    finally:
        big.close()
        small.close()


def test_static_fission_rate_rejects_sizes_beyond_its_scratch_and_bad_arguments():
    t = torch.ones(8, dtype=torch.float64, device="cuda")
    m = torch.zeros(8, dtype=torch.int32, device="cuda")
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    L = nd.lib()
    args = lambda R, G: (R, G, t.data_ptr(), m.data_ptr(), t.data_ptr(), t.data_ptr(), out.data_ptr(), None)
    R_max = nd.ND_STATIC_FISSION_MAX_ELEMENTS
    assert L.nd_fission_rate_static(*args(R_max + 1, 1)) == 3                      # ND_ERR_RANGE
    assert b"ND_STATIC_FISSION_MAX_ELEMENTS" in L.nd_last_error(None)
    assert L.nd_fission_rate_static(*args((R_max >> 5) + 1, 32)) == 3
    assert L.nd_fission_rate_static(*args(0, 1)) == 2                              # ND_ERR_INVALID
    assert L.nd_fission_rate_static(8, 1, None, m.data_ptr(), t.data_ptr(), t.data_ptr(), out.data_ptr(), None) == 1   # ND_ERR_NULL
    torch.cuda.synchronize()
    assert float(out.cpu()[0]) == 7.0, "a rejected call launches nothing"
    assert L.nd_fission_rate_static(*args(8, 1)) == 0
    assert float(out.cpu()[0]) == 8.0                                              # sum of 1 * 1 * 1 over 8 regions
