"""GPU parity of NEXT-3, step C-3: nd_sweep_currents (through the C ABI) against orc_sweep_currents
(oracle/moc_oracle.c, FP64) on the same seeded Q, boundary flux and coarse overlay, plus the exact per-cell balance of
the currents with the tallies of the GPU's own sweep.  Run with  pytest -m gpu  on a B200."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import paper_2607_01591_b200 as nd
from oracle import cmfd
from moc_inputs.coarse import cartesian_cells
from gpu_common import make_pair, seeded_sweep_inputs, phi_rel_err, PHI_RTOL

pytestmark = pytest.mark.gpu

# FP32 chains against FP64.  A net current is a difference of one-way currents, so the bar is relative to the largest
# net current of the array.  Measured on the five cases: 4e-8 .. 7e-7 (the FP32 rounding of psi, averaged over the tracks
# of a surface); the bar leaves a factor of ~7.  The C-3 balance of the GPU's own numbers: measured 4e-9 .. 1.2e-7.
J_RTOL = 5e-6
BALANCE_RTOL = 2e-6
# (config, scale, coarse nx, ny): reflective, vacuum and mixed boundaries; G = 7 .. 51, ragged group tails (G % 32 != 0)
CASES = [(1, 1.0, 3, 2), (2, 0.15, 4, 3), (3, 0.03, 5, 4), (4, 0.06, 6, 5), (5, 0.0008, 4, 4)]


def _oracle_currents(pair, Q, psi, cell, n_cells, lo, hi):
    p, t = pair.prob, pair.o_tr
    return cmfd.sweep_currents(p.mesh.material, p.xs.sigma_t, p.polar_sin, p.polar_weight, t.seg_offset, t.seg_region,
                               t.seg_length, t.track_weight, t.link, Q, psi.astype(np.float64), cell, n_cells, lo, hi)


@pytest.mark.parametrize("case", CASES, ids=[f"cfg{c[0]}x{c[1]}" for c in CASES])
def test_currents_match_oracle_and_balance(case):
    idx, scale, nx, ny = case
    pair = make_pair(idx, scale, sweep_kernel=nd.ND_SWEEP_ATOMIC)
    try:
        Q, psi = seeded_sweep_inputs(pair, seed=300 + idx)
        n_cells = nx * ny
        cell = cartesian_cells(pair.prob.mesh, nx, ny)
        lo, hi = cmfd.coarse_surfaces(pair.o_tr.seg_offset, pair.o_tr.seg_region, cell, pair.o_tr.link)
        assert len(lo) >= nx * (ny - 1) + ny * (nx - 1) - 1
        Js_o, Jv_o, Jr_o = _oracle_currents(pair, Q, psi, cell, n_cells, lo, hi)
        # the library takes the surfaces in any order
        perm = np.random.default_rng(7).permutation(len(lo))
        dQ = torch.from_numpy(Q).cuda()
        pair.gpu.nd_boundary_flux_set(psi)
        Js_g, Jv_g, Jr_g = pair.gpu.nd_sweep_currents(dQ, cell, n_cells, lo[perm], hi[perm])
        Js_back = np.empty_like(Js_g)
        Js_back[perm] = Js_g
        for name, g, o in (("J_surf", Js_back, Js_o), ("J_vac", Jv_g, Jv_o), ("J_ref", Jr_g, Jr_o)):
            ref = np.abs(o).max()
            err = np.abs(g - o).max()
            print(f"cfg{idx} {name}: max|J| {ref:.4e} err {err:.3e} ratio {err / max(ref, 1e-300):.3e}")
            if ref == 0.0:
                assert err == 0.0, name      # no vacuum (or no reflective) side: nothing may be written there
            else:
                assert err <= J_RTOL * ref, name
        # the call leaves the state alone: same boundary flux, and the sweep that follows is the oracle's sweep
        assert np.array_equal(pair.gpu.nd_boundary_flux_get(), psi)
        phi_g = pair.gpu.nd_transport_sweep(dQ).cpu().numpy()
        tally_g = pair.gpu.nd_tally_get().cpu().numpy()
        phi_o, _, tally_o = pair.oracle_sweep(Q, psi.astype(np.float64))
        assert phi_rel_err(phi_g, phi_o) <= PHI_RTOL
        # C-3 identity on the GPU's own numbers: tallies + surface currents + boundary ends telescope to zero per cell
        net = np.zeros((n_cells, pair.G))
        np.add.at(net, cell, tally_g)
        np.add.at(net, lo, Js_back)
        np.add.at(net, hi, -Js_back)
        net += Jv_g + Jr_g
        gross = np.zeros((n_cells, pair.G))
        np.add.at(gross, cell, np.abs(tally_o))
        print(f"cfg{idx} balance: {np.abs(net).max() / gross.max():.3e}")
        assert np.abs(net).max() <= BALANCE_RTOL * gross.max()
    finally:
        pair.close()


def test_one_cell_has_no_surface_and_all_leakage_at_the_ends():
    pair = make_pair(2, 0.15, sweep_kernel=nd.ND_SWEEP_ATOMIC)
    try:
        Q, psi = seeded_sweep_inputs(pair, seed=41)
        dQ = torch.from_numpy(Q).cuda()
        pair.gpu.nd_boundary_flux_set(psi)
        one = np.zeros(pair.R, np.int32)
        none = np.zeros(0, np.int32)
        Js, Jv, Jr = pair.gpu.nd_sweep_currents(dQ, one, 1, none, none)
        assert Js.shape == (0, pair.G)
        _, Jv_o, Jr_o = _oracle_currents(pair, Q, psi, one, 1, none, none)
        assert np.abs(Jv - Jv_o).max() <= J_RTOL * max(np.abs(Jv_o).max(), 1e-300) or np.abs(Jv_o).max() == 0.0
        assert np.abs(Jr - Jr_o).max() <= J_RTOL * max(np.abs(Jr_o).max(), 1e-300) or np.abs(Jr_o).max() == 0.0
        pair.gpu.nd_transport_sweep(dQ)
        tally = pair.gpu.nd_tally_get().cpu().numpy()
        assert np.abs(tally.sum(0) + Jv[0] + Jr[0]).max() <= BALANCE_RTOL * np.abs(tally).sum(0).max()
    finally:
        pair.close()


def test_errors_are_reported():
    pair = make_pair(1, 1.0, sweep_kernel=nd.ND_SWEEP_ATOMIC)
    swath = make_pair(1, 1.0, sweep_kernel=nd.ND_SWEEP_SWATH)
    try:
        Q, psi = seeded_sweep_inputs(pair, seed=5)
        dQ = torch.from_numpy(Q).cuda()
        cell = cartesian_cells(pair.prob.mesh, 3, 2)
        lo, hi = cmfd.coarse_surfaces(pair.o_tr.seg_offset, pair.o_tr.seg_region, cell, pair.o_tr.link)
        with pytest.raises(nd.NdError, match="ND_SWEEP_ATOMIC"):       # the tiled kernels carry no SoA stream
            swath.gpu.nd_sweep_currents(dQ, cell, 6, lo, hi)
        with pytest.raises(nd.NdError, match="not a listed surface"):  # a crossing without its surface
            pair.gpu.nd_sweep_currents(dQ, cell, 6, lo[1:], hi[1:])
        with pytest.raises(nd.NdError, match="listed twice"):
            pair.gpu.nd_sweep_currents(dQ, cell, 6, np.r_[lo, lo[:1]], np.r_[hi, hi[:1]])
        with pytest.raises(nd.NdError, match="out of"):
            pair.gpu.nd_sweep_currents(dQ, cell, 5, lo, hi)            # cell 5 >= n_cells
        with pytest.raises(nd.NdError, match="lo < hi"):
            pair.gpu.nd_sweep_currents(dQ, cell, 6, hi, lo)
        # and the problem still works afterwards
        Js, Jv, Jr = pair.gpu.nd_sweep_currents(dQ, cell, 6, lo, hi)
        assert np.isfinite(Js).all() and np.isfinite(Jv).all() and np.isfinite(Jr).all()
    finally:
        pair.close()
        swath.close()
