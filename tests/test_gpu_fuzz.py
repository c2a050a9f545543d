"""Seeded random shapes through the swath kernel: meshes, group counts (every lanes-per-slot count from 1 to 16 and the
fallback beyond 128 groups), polar sets of 1-4 angles, boundary conditions, ray densities, and tile shapes / cut rules /
buffer options of nd_options -- one sweep against the oracle (Eq. (5)) and a few power iterations against
the atomic kernel.  The ragged cases (slots without a track, tiles with one segment, windows of 16 regions, tracks of one
segment) come from the small meshes and the tiny tile shapes."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import paper_2607_01591_b200 as nd
from gpu_common import Pair, seeded_sweep_inputs, phi_rel_err, PHI_RTOL, PSI_ATOL_REL
from moc_inputs import Problem, make_xs, rect_tri_mesh, tabuchi_yamamoto

pytestmark = pytest.mark.gpu

GROUPS = [1, 2, 3, 4, 5, 7, 8, 9, 12, 13, 16, 17, 20, 24, 28, 29, 33, 36, 40, 44, 47, 51, 56, 60, 64, 70, 130]


def _random_problem(seed):
    rng = np.random.default_rng(1000 + seed)
    G = GROUPS[seed % len(GROUPS)]
    P = int(rng.integers(1, 5))
    if P <= 3:
        s, w = tabuchi_yamamoto(P)
    else:
        s = np.array([0.21, 0.48, 0.79, 0.96])
        w = np.array([0.1, 0.2, 0.3, 0.4])
    nx, ny = int(rng.integers(2, 9)), int(rng.integers(2, 9))
    M = int(rng.integers(1, 5))
    mesh = rect_tri_mesh(float(rng.uniform(1.0, 4.0)), float(rng.uniform(1.0, 4.0)), nx, ny, seed=seed, jitter=float(rng.uniform(0.0, 0.4)),
                         n_materials=M)
    xs = make_xs(G, [bool(m % 2 == 0) for m in range(M)], seed, sigt_range=(0.1, 2.5), c_range=(0.3, 0.9), n_up=min(2, G - 1) if G > 1 else 0)
    bc = tuple(int(b) for b in rng.integers(0, 2, 4))
    n_azim = int(rng.choice([4, 8, 16, 32]))
    spacing = float(rng.choice([0.2, 0.07, 0.03, 0.011]))
    return Problem(f"fuzz{seed}", mesh, xs, n_azim, spacing, s, w, bc, 5, "seeded random shape")


def _random_options(seed):
    rng = np.random.default_rng(5000 + seed)
    o = {}
    if rng.random() < 0.6:
        o["block_warps"] = int(rng.choice([1, 2, 4, 8]))
    if rng.random() < 0.6:
        o["tile_segments"] = int(rng.choice([1, 2, 3, 5, 8, 13]))
    if rng.random() < 0.5:
        o["window_regions"] = int(rng.choice([16, 17, 24, 40]))
    if rng.random() < 0.5:
        o["tile_lag"] = int(rng.choice([-1, 1, 4, 16]))
    if rng.random() < 0.3:
        o["q_copies"] = int(rng.choice([1, 2, 8]))
    if rng.random() < 0.3:
        o["delta_buffers"] = 2
    if rng.random() < 0.3:
        o["item_order"] = 1
    if rng.random() < 0.2:
        o["p1_stream"] = 1
    return o


@pytest.mark.parametrize("seed", range(len(GROUPS) + 9))
def test_random_shapes_against_the_oracle_and_the_atomic_kernel(seed):
    prob = _random_problem(seed)
    opts = _random_options(seed)
    try:
        pair = Pair(prob, sweep_kernel=nd.ND_SWEEP_SWATH, **opts)
    except nd.NdError as e:            # a shape the shared memory cannot hold is refused at create, never mis-run
        assert "ND_ERR_INVALID" in str(e) or "ND_ERR_WORKSPACE" in str(e), str(e)
        pytest.skip(f"options {opts} refused for G = {prob.n_groups}: {e}")
    ref = Pair(prob, sweep_kernel=nd.ND_SWEEP_ATOMIC)
    try:
        info = pair.gpu.nd_problem_info_get()
        assert info["sweep_kernel"] == (nd.ND_SWEEP_SWATH if prob.n_groups <= 128 else nd.ND_SWEEP_ATOMIC)
        Q, psi = seeded_sweep_inputs(pair, seed)
        dQ = torch.from_numpy(Q).cuda()
        phi_o, psi_o, _ = pair.oracle_sweep(Q, psi.astype(np.float64))
        for p in (pair, ref):
            p.gpu.nd_boundary_flux_set(psi)
            phi = p.gpu.nd_transport_sweep(dQ).cpu().numpy()
            assert phi_rel_err(phi, phi_o) <= PHI_RTOL, (prob.n_groups, prob.n_polar, opts)
            assert np.abs(p.gpu.nd_boundary_flux_get() - psi_o).max() <= PSI_ATOL_REL * max(np.abs(psi_o).max(), 1e-30)
        if seed % 2 == 0 and info["sweep_kernel"] == nd.ND_SWEEP_SWATH:
            # the same shape with the segments left on the GPU: the device builder's chunk stream, byte for byte
            m = prob.mesh
            tr = nd.nd_tracks_generate_resident(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
            g = nd.nd_problem_create(prob.xs, prob.polar_sin, prob.polar_weight, m.material, tr, sweep_kernel=nd.ND_SWEEP_SWATH, **opts)
            try:
                a, b = g.nd_problem_stream_view(), pair.gpu.nd_problem_stream_view()
                assert a["built_on_device"] and not b["built_on_device"]
                for f in ("blob", "tile_ref", "swath_tile0", "swath_track", "items"):
                    assert a[f].tobytes() == b[f].tobytes(), (f, prob.n_groups, opts)
            finally:
                g.destroy()
                tr.destroy()
        for p in (pair, ref):
            p.gpu.nd_state_reset()
        ka, kb = pair.gpu.nd_power_iteration(5)["k_eff"], ref.gpu.nd_power_iteration(5)["k_eff"]
        assert abs(ka - kb) <= 2e-6 * abs(kb), (ka, kb, prob.n_groups, opts)
    finally:
        pair.close()
        ref.close()
