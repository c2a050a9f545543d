"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default options, the
kernel ND_SWEEP_AUTO selects).

configs 2-4: the whole problem against the oracle (one seeded sweep element by element, then a short power
iteration), and the library's tracks against the oracle's, byte for byte.
config 5 (1e6 regions, 4.9e8 segments, 1.5e11 updates per sweep): the oracle computes SAMPLED outputs one by
one -- the outgoing angular flux of sampled tracks, and the tally / scalar flux of sampled regions from the sub-set
of tracks that cross them -- all with the bars of the small cases."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
import paper_2607_01591_b200 as nd
from moc_inputs import make_config
from gpu_common import make_pair, seeded_sweep_inputs, phi_rel_err, PHI_RTOL, K_PCM, PSI_ATOL_REL

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("idx,n_it", [(2, 10), (3, 4), (4, 4)], ids=["cfg2", "cfg3", "cfg4"])
def test_full_config_against_the_oracle(idx, n_it):
    pair = make_pair(idx, 1.0)
    try:
        o, g = pair.o_tr, pair.g_tr
        for name in ("seg_offset", "seg_region", "seg_length", "track_weight", "link"):
            assert getattr(o, name).tobytes() == getattr(g, name).tobytes(), f"{name} not bit-exact"
        assert pair.gpu.nd_problem_info_get()["sweep_kernel"] == nd.ND_SWEEP_SWATH
        Q, psi = seeded_sweep_inputs(pair, 40 + idx)
        pair.gpu.nd_boundary_flux_set(psi)
        phi_g = pair.gpu.nd_transport_sweep(torch.from_numpy(Q).cuda()).cpu().numpy()
        psi_g = pair.gpu.nd_boundary_flux_get()
        phi_o, psi_o, _ = pair.oracle_sweep(Q, psi.astype(np.float64))
        assert phi_rel_err(phi_g, phi_o) <= PHI_RTOL
        assert np.abs(psi_g - psi_o).max() <= PSI_ATOL_REL * np.abs(psi_o).max()
        pair.gpu.nd_state_reset()
        ko, phio, _, _ = pair.oracle_power(n_it)
        dphi = torch.empty((pair.R, pair.G), dtype=torch.float64, device="cuda")
        out = pair.gpu.nd_power_iteration(n_it, d_phi_out=dphi)
        assert abs(out["k_eff"] - ko) * 1e5 <= K_PCM
        assert phi_rel_err(dphi.cpu().numpy(), phio) <= PHI_RTOL
    finally:
        pair.close()


def _subset(tr, tracks):
    """CSR of a sub-set of tracks (links cut), for the oracle."""
    counts = (tr.seg_offset[tracks + 1] - tr.seg_offset[tracks]).astype(np.int64)
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    idx = np.concatenate([np.arange(tr.seg_offset[t], tr.seg_offset[t + 1]) for t in tracks]) if len(tracks) else np.zeros(0, np.int64)
    return off, np.ascontiguousarray(tr.seg_region[idx]), np.ascontiguousarray(tr.seg_length[idx]), np.ascontiguousarray(tr.track_weight[tracks])


def test_config5_full_size_sampled_outputs():
    prob = make_config(5, scale=1.0)
    m = prob.mesh
    tr = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    gp = nd.nd_problem_create(prob.xs, prob.polar_sin, prob.polar_weight, m.material, tr)
    try:
        R, G, P, T = m.n_regions, prob.n_groups, prob.n_polar, tr.n_tracks
        info = gp.nd_problem_info_get()
        assert info["sweep_kernel"] == nd.ND_SWEEP_SWATH and info["n_segments"] == tr.n_segments
        rng = np.random.default_rng(505)
        Q = rng.uniform(0.05, 1.0, size=(R, G))
        psi = rng.uniform(0.0, 2.0, size=(T, 2, P, G)).astype(np.float32)
        gp.nd_boundary_flux_set(psi)
        phi_g = gp.nd_transport_sweep(torch.from_numpy(Q).cuda()).cpu().numpy()
        tally_g = gp.nd_tally_get().cpu().numpy()
        psi_g = gp.nd_boundary_flux_get().reshape(2 * T, P, G)
        vol = gp.nd_track_volume_get()
        assert np.isfinite(phi_g).all() and (phi_g > 0).all()
        # (0) telescoping balance over the WHOLE problem, per group: what the chains lost is what the regions tallied
        psi_exit_all = gp.nd_outgoing_flux_get().astype(np.float64)
        w_tp = 4.0 * np.pi * tr.track_weight[:, None] * (prob.polar_weight * prob.polar_sin)[None, :]      # [T][P]
        lost = np.einsum("tp,tdpg->g", w_tp, psi.astype(np.float64) - psi_exit_all)
        assert np.abs(tally_g.sum(axis=0) - lost).max() <= 2e-5 * np.abs(lost).max()
        del psi_exit_all
        # (a) sampled tracks: the oracle's chain along each track alone; compare where the exit is linked
        tracks = np.unique(np.concatenate([rng.integers(0, T, size=96), [0, T - 1]])).astype(np.int64)
        off, sr, sl, tw = _subset(tr, tracks)
        link_id = np.arange(2 * len(tracks), dtype=np.int32).reshape(len(tracks), 2)   # exit (i,d) -> entry 2i+d of the sub-set
        _, psi_exit, _ = oracle.sweep(m.material, prob.xs.sigma_t, prob.polar_sin, prob.polar_weight, off, sr, sl, tw,
                                      link_id, vol, Q, psi[tracks].astype(np.float64))
        psi_exit = psi_exit.reshape(2 * len(tracks), P, G)
        n_cmp = 0
        for i, t in enumerate(tracks):
            for d in (0, 1):
                lk = tr.link[t, d]
                if lk >= 0:
                    ref = psi_exit[2 * i + d]
                    assert np.abs(psi_g[lk] - ref).max() <= PSI_ATOL_REL * max(np.abs(ref).max(), 1.0)
                    n_cmp += 1
        assert n_cmp > 50
        # vacuum entries stay exactly zero
        fed = np.zeros(2 * T, bool)
        fed[tr.link[tr.link >= 0]] = True
        assert np.all(psi_g[~fed] == 0.0)
        # (b) sampled regions: all tracks that cross them, swept by the oracle -> their tally rows and scalar flux
        regions = np.unique(rng.integers(0, R, size=6))
        hit = np.flatnonzero(np.isin(tr.seg_region, regions))
        crossing = np.unique(np.searchsorted(tr.seg_offset, hit, side="right") - 1).astype(np.int64)
        off, sr, sl, tw = _subset(tr, crossing)
        phi_o, _, tally_o = oracle.sweep(m.material, prob.xs.sigma_t, prob.polar_sin, prob.polar_weight, off, sr, sl, tw,
                                         np.full((len(crossing), 2), -1, np.int32), vol, Q, psi[crossing].astype(np.float64))
        for r in regions:
            assert np.abs(tally_g[r] - tally_o[r]).max() <= 2e-4 * np.abs(tally_o[r]).max()
            assert phi_rel_err(phi_g[r:r + 1], phi_o[r:r + 1]) <= PHI_RTOL
    finally:
        gp.destroy()
        tr.destroy()


def test_config5_full_size_whole_sweep_against_the_oracle():
    """ONE oracle sweep (O-6) at config 5's full size, compared element by element with the CUDA path in the launch
    configuration bench.py times: every phi[r][g] (1e-4), every tally (2e-4 of the largest), every boundary psi (2e-5).
    About 1.5e11 FP64 updates on the host cores (minutes) and ~10 GB of host arrays."""
    prob = make_config(5, scale=1.0)
    m = prob.mesh
    tr = nd.nd_tracks_generate_device(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing, segment_capacity=1 << 28)
    gp = nd.nd_problem_create(prob.xs, prob.polar_sin, prob.polar_weight, m.material, tr)
    try:
        R, G, P, T = m.n_regions, prob.n_groups, prob.n_polar, tr.n_tracks
        info = gp.nd_problem_info_get()
        assert info["sweep_kernel"] == nd.ND_SWEEP_SWATH and info["n_segments"] == tr.n_segments
        rng = np.random.default_rng(515)
        Q = rng.uniform(0.05, 1.0, size=(R, G))
        psi = rng.uniform(0.0, 2.0, size=(T, 2, P, G)).astype(np.float32)
        gp.nd_boundary_flux_set(psi)
        phi_g = gp.nd_transport_sweep(torch.from_numpy(Q).cuda()).cpu().numpy()
        tally_g = gp.nd_tally_get().cpu().numpy()
        psi_g = gp.nd_boundary_flux_get()
        vol = gp.nd_track_volume_get()
        # the oracle on the library's (bit-exact, tests/test_gpu_trace.py) segment arrays; its own volumes from them
        vol_o = oracle.track_volumes(R, tr.seg_offset, tr.seg_region, tr.seg_length, tr.track_weight)
        assert np.abs(vol - vol_o).max() <= 1e-12 * vol_o.max()
        psi64 = psi.astype(np.float64)
        del psi
        phi_o, psi_o, tally_o = oracle.sweep(m.material, prob.xs.sigma_t, prob.polar_sin, prob.polar_weight, tr.seg_offset,
                                             tr.seg_region, tr.seg_length, tr.track_weight, tr.link, vol_o, Q, psi64)
        del psi64
        err_phi = phi_rel_err(phi_g, phi_o)
        err_tally = float(np.abs(tally_g - tally_o).max() / np.abs(tally_o).max())
        err_psi = float(np.abs(psi_g - psi_o).max() / np.abs(psi_o).max())
        print(f"config 5 full sweep: phi rel err {err_phi:.3e}, tally {err_tally:.3e}, psi {err_psi:.3e}")
        assert err_phi <= PHI_RTOL
        assert err_tally <= 2e-4
        assert err_psi <= PSI_ATOL_REL
    finally:
        gp.destroy()
        tr.destroy()


def test_config5_tenth_scale_twin_power_iteration():
    """k_eff, k history and phi after 20 power iterations on config 5's 0.1-scale twin (~1e5 FSRs, 51 groups, the
    production tile / swath shapes): SURVEY 8(d) 'k_eff parity ... on a stated 10x-down-scaled twin'."""
    pair = make_pair(5, 0.1)
    try:
        assert pair.R > 90_000 and pair.gpu.nd_problem_info_get()["sweep_kernel"] == nd.ND_SWEEP_SWATH
        n_it = 20
        ko, phio, psio, hist = pair.oracle_power(n_it)
        dphi = torch.empty((pair.R, pair.G), dtype=torch.float64, device="cuda")
        out = pair.gpu.nd_power_iteration(n_it, d_phi_out=dphi, want_stats=True)
        kg = np.array([s["k_eff"] for s in out["stats"]])
        print(f"config 5 x0.1 twin: k_gpu {out['k_eff']:.8f} k_oracle {ko:.8f}, max history diff {np.abs(kg - hist).max() * 1e5:.3f} pcm")
        assert np.abs(kg - hist).max() * 1e5 <= K_PCM
        assert abs(out["k_eff"] - ko) * 1e5 <= K_PCM
        assert phi_rel_err(dphi.cpu().numpy(), phio) <= PHI_RTOL
        psi_g = pair.gpu.nd_boundary_flux_get()
        assert np.abs(psi_g - psio).max() <= 5 * PSI_ATOL_REL * np.abs(psio).max()   # the bar of test_power_iteration_matches_oracle
    finally:
        pair.close()
