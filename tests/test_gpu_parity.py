"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle, element by element, on the same
seeded inputs.  Bars (BASELINE.json north_star): phi max rel err <= 1e-4 per sweep, k_eff within 5 pcm after a
fixed iteration count.  Run with  pytest -m gpu  on a B200."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
import paper_2607_01591_b200 as nd
from moc_inputs import make_config, rect_tri_mesh, homogeneous_xs, tabuchi_yamamoto, make_xs
from moc_inputs.configs import Problem as InputProblem
from gpu_common import Pair, make_pair, seeded_sweep_inputs, phi_rel_err, PHI_RTOL, K_PCM, PSI_ATOL_REL

pytestmark = pytest.mark.gpu

KERNELS = [pytest.param(nd.ND_SWEEP_ATOMIC, id="atomic"), pytest.param(nd.ND_SWEEP_SWATH, id="swath")]

# (config index, scale): sizes the oracle finishes in seconds, spanning several tiles and ragged tails
SWEEP_CASES = [(1, 1.0), (2, 0.15), (2, 1.0), (3, 0.03), (4, 0.06), (5, 0.0008)]


def _check_sweep(pair, seed, n_sweeps=2):
    Q, psi = seeded_sweep_inputs(pair, seed)
    dQ = torch.from_numpy(Q).cuda()
    pair.gpu.nd_boundary_flux_set(psi)
    psi_o = psi.astype(np.float64)
    for _ in range(n_sweeps):  # the second sweep starts from the exchanged boundary flux
        phi_g = pair.gpu.nd_transport_sweep(dQ).cpu().numpy()
        tally_g = pair.gpu.nd_tally_get().cpu().numpy()
        psi_g = pair.gpu.nd_boundary_flux_get()
        phi_o, psi_o, tally_o = pair.oracle_sweep(Q, psi_o)
        assert phi_rel_err(phi_g, phi_o) <= PHI_RTOL
        assert np.abs(psi_g - psi_o).max() <= PSI_ATOL_REL * np.abs(psi_o).max()
        # telescoping invariant on the GPU result itself (exact up to FP32 rounding of the chain)
        if _ == 0:
            w_tp = 4.0 * np.pi * pair.o_tr.track_weight[:, None] * (pair.prob.polar_weight * pair.prob.polar_sin)[None, :]
            lost = np.einsum("tp,tdpg->g", w_tp, psi.astype(np.float64) - pair.gpu.nd_outgoing_flux_get().astype(np.float64))
            assert np.abs(tally_g.sum(axis=0) - lost).max() <= 2e-5 * max(np.abs(lost).max(), 1e-30)
        scale = np.abs(tally_o).max()
        assert np.abs(tally_g - tally_o).max() <= 2e-4 * scale


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("case", SWEEP_CASES, ids=[f"cfg{c[0]}x{c[1]}" for c in SWEEP_CASES])
def test_sweep_matches_oracle(case, kernel):
    pair = make_pair(case[0], case[1], sweep_kernel=kernel)
    try:
        _check_sweep(pair, seed=100 + case[0])
    finally:
        pair.close()


SHAPES = [dict(block_warps=1), dict(block_warps=3, tile_segments=2, window_regions=5), dict(block_warps=8, tile_segments=16),
          dict(block_warps=16, tile_segments=5, delta_buffers=2), dict(block_warps=8, tile_lag=-1), dict(block_warps=4, tile_lag=1000),
          dict(block_warps=12, tile_segments=12, blocks_per_sm=1), dict(block_warps=4, q_copies=4), dict(block_warps=2, q_copies=2),
          dict(block_warps=4, q_copies=3, tile_segments=6)]


@pytest.mark.parametrize("case", [(2, 0.15), (4, 0.06), (5, 0.0008)], ids=["cfg2", "cfg4", "cfg5"])
@pytest.mark.parametrize("shape", SHAPES, ids=[str(i) for i in range(len(SHAPES))])
def test_swath_block_and_tile_shapes(case, shape):
    """The swath kernel's tuning options (block size, tile length, region window, delta buffers, tile policy) never
    change the result beyond summation order."""
    pair = make_pair(case[0], case[1], sweep_kernel=nd.ND_SWEEP_SWATH, **shape)
    try:
        info = pair.gpu.nd_problem_info_get()
        assert info["sweep_kernel"] == nd.ND_SWEEP_SWATH and 32 <= info["block_threads"] <= 32 * shape["block_warps"]
        _check_sweep(pair, seed=300 + case[0])
    finally:
        pair.close()


@pytest.mark.parametrize("exp_mode", [nd.ND_EXP_FAST, nd.ND_EXP_EXPM1])
def test_sweep_exp_modes(exp_mode):
    pair = make_pair(2, 0.15, exp_mode=exp_mode)
    try:
        _check_sweep(pair, seed=7, n_sweeps=1)
    finally:
        pair.close()


def _custom_pair(G, P, bc, n_azim=16, spacing=0.07, seed=3, n_materials=3, **options):
    mesh = rect_tri_mesh(2.3, 1.7, 7, 5, seed=seed, jitter=0.3)
    rng = np.random.default_rng(seed)
    mesh.material[:] = rng.integers(0, n_materials, size=mesh.n_regions).astype(np.int32)
    xs = make_xs(G, [True] + [False] * (n_materials - 1), seed, n_up=min(2, G - 1))
    if P <= 3:
        s, w = tabuchi_yamamoto(P)
    else:  # any valid quadrature is an input; 4-point Gauss-Legendre in mu on (0,1)
        mu, w = np.polynomial.legendre.leggauss(4)
        mu, w = 0.5 * (mu + 1.0), 0.5 * w
        s = np.sqrt(1.0 - mu * mu)
    prob = InputProblem(f"custom_G{G}_P{P}", mesh, xs, n_azim, spacing, s, w, bc, 10)
    return Pair(prob, **options)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("G,P", [(1, 1), (2, 2), (3, 3), (5, 4), (8, 3), (31, 3), (32, 2), (33, 3), (51, 3), (64, 1), (70, 3), (128, 2), (129, 1), (200, 3)])
def test_sweep_group_and_polar_shapes(G, P, kernel):
    pair = _custom_pair(G, P, (1, 0, 0, 1), sweep_kernel=kernel)
    try:
        _check_sweep(pair, seed=G * 10 + P)
    finally:
        pair.close()


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("bc", [(0, 0, 0, 0), (1, 1, 1, 1), (0, 1, 1, 0)])
def test_sweep_boundary_conditions(bc, kernel):
    pair = _custom_pair(7, 3, bc, sweep_kernel=kernel)
    try:
        _check_sweep(pair, seed=11, n_sweeps=3)
        psi = pair.gpu.nd_boundary_flux_get()
        lk = pair.o_tr.link
        fed = np.zeros(2 * pair.T, bool)
        fed[lk[lk >= 0]] = True
        assert np.all(psi.reshape(2 * pair.T, -1)[~fed] == 0.0), "vacuum entries must stay exactly zero"
    finally:
        pair.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_sweep_with_empty_and_single_segment_tracks(kernel):
    """Degenerate descriptor: tracks with zero segments pass their flux through unchanged."""
    G, P, R, T = 5, 2, 4, 6
    rng = np.random.default_rng(5)
    xs = make_xs(G, [True, False], 9)
    s, w = tabuchi_yamamoto(P)
    counts = np.array([0, 1, 3, 0, 9, 2])
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    seg_region = rng.integers(0, R, size=off[-1]).astype(np.int32)
    seg_length = rng.uniform(0.01, 0.8, size=off[-1])
    tw = rng.uniform(0.001, 0.01, size=T)
    link = np.array([[2, 1], [0, 3], [-1, 5], [7, -1], [9, 8], [11, 10]], np.int32)
    mat = np.array([0, 1, 1, 0], np.int32)
    gp = nd.Problem(mat, xs.sigma_t, xs.sigma_s, xs.nu_sigma_f, xs.chi, s, w, off, seg_region, seg_length, tw, link,
                    sweep_kernel=kernel)
    vol = oracle.track_volumes(R, off, seg_region, seg_length, tw)
    assert np.allclose(gp.nd_track_volume_get(), vol, rtol=1e-15)
    Q = rng.uniform(0.1, 1.0, size=(R, G))
    psi = rng.uniform(0, 2, size=(T, 2, P, G)).astype(np.float32)
    gp.nd_boundary_flux_set(psi)
    phi_g = gp.nd_transport_sweep(torch.from_numpy(Q).cuda()).cpu().numpy()
    psi_g = gp.nd_boundary_flux_get()
    phi_o, psi_o, _ = oracle.sweep(mat, xs.sigma_t, s, w, off, seg_region, seg_length, tw, link, vol, Q, psi.astype(np.float64))
    assert phi_rel_err(phi_g, phi_o) <= PHI_RTOL
    assert np.abs(psi_g - psi_o).max() <= PSI_ATOL_REL * np.abs(psi_o).max()
    assert np.array_equal(psi_g[1, 0], psi[0, 0]), "empty track 0 forwards its flux bit-exactly into entry 2"
    gp.destroy()


def test_source_update_matches_oracle():
    for idx, scale in [(1, 1.0), (4, 0.06), (5, 0.0008)]:
        pair = make_pair(idx, scale)
        try:
            rng = np.random.default_rng(idx)
            phi = rng.uniform(0.1, 3.0, size=(pair.R, pair.G))
            k = 0.9 + 0.3 * rng.random()
            Qg, Fg = pair.gpu.nd_source_update(torch.from_numpy(phi).cuda(), k, want_fission_rate=True)
            p = pair.prob
            Qo = oracle.source(p.mesh.material, p.xs.sigma_s, p.xs.nu_sigma_f, p.xs.chi, phi, k)
            Fo = oracle.fission_rate(p.mesh.material, p.xs.nu_sigma_f, pair.o_tr.volume, phi)
            assert np.abs(Qg.cpu().numpy() - Qo).max() <= 1e-13 * np.abs(Qo).max()
            assert abs(Fg.item() - Fo) <= 1e-12 * abs(Fo)
        finally:
            pair.close()


def test_source_update_alternating_between_live_problems_of_different_size():
    # the source kernel's dynamic shared-memory limit is an attribute of the KERNEL: a small problem created after a large one
    # must not lower it under the large one's feet (G = 33 stages a 57 KB tile, G = 2 a few hundred bytes)
    big, small = make_pair(4, 0.06), make_pair(1, 1.0)
    try:
        for pair in (big, small, big, small, big):
            rng = np.random.default_rng(pair.G)
            phi = rng.uniform(0.1, 3.0, size=(pair.R, pair.G))
            Qg = pair.gpu.nd_source_update(torch.from_numpy(phi).cuda(), 1.1)
            p = pair.prob
            Qo = oracle.source(p.mesh.material, p.xs.sigma_s, p.xs.nu_sigma_f, p.xs.chi, phi, 1.1)
            assert np.abs(Qg.cpu().numpy() - Qo).max() <= 1e-13 * np.abs(Qo).max()
    finally:
        big.close()
        small.close()


POWER_CASES = [(1, 1.0, 50), (2, 0.15, 20), (2, 1.0, 20), (3, 0.03, 20), (4, 0.06, 20), (5, 0.0008, 20)]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("case", POWER_CASES, ids=[f"cfg{c[0]}x{c[1]}" for c in POWER_CASES])
def test_power_iteration_matches_oracle(case, kernel):
    idx, scale, n_it = case
    pair = make_pair(idx, scale, sweep_kernel=kernel)
    try:
        ko, phio, psio, hist = pair.oracle_power(n_it)
        dphi = torch.empty((pair.R, pair.G), dtype=torch.float64, device="cuda")
        out = pair.gpu.nd_power_iteration(n_it, d_phi_out=dphi, want_stats=True)
        assert out["iters"] == n_it
        assert abs(out["k_eff"] - ko) * 1e5 <= K_PCM
        kh = np.array([s["k_eff"] for s in out["stats"]])
        assert np.abs(kh - hist).max() * 1e5 <= K_PCM, "k history"
        assert phi_rel_err(dphi.cpu().numpy(), phio) <= PHI_RTOL
        psi_g = pair.gpu.nd_boundary_flux_get()
        assert np.abs(psi_g - psio).max() <= 5 * PSI_ATOL_REL * np.abs(psio).max()
        # resume: state get/set round trip continues the same iteration
        out2 = pair.gpu.nd_power_iteration(3)
        ko2, *_ = pair.oracle_power(3, state=(ko, phio, psio))
        assert abs(out2["k_eff"] - ko2) * 1e5 <= K_PCM
    finally:
        pair.close()


@pytest.mark.parametrize("case", [(3, 0.03), (4, 0.06), (2, 0.15)], ids=["cfg3", "cfg4", "cfg2"])
def test_iteration_stats_leakage_and_balance_residual(case):
    """nd_iter_stats.leakage against the oracle's telescoping identity (sum of the tallies = what entered - what left
    through the track ends, tests/test_oracle_sweep.py): leakage = in - sum(tally) - what left through LINKED ends, all from
    the oracle's own sweep; balance_residual is that identity evaluated on the GPU's own numbers (FP32 chain rounding)."""
    pair = make_pair(*case)
    try:
        p, t = pair.prob, pair.o_tr
        n_it = 4
        out = pair.gpu.nd_power_iteration(n_it, want_stats=True)
        w_tp = 4.0 * np.pi * t.track_weight[:, None] * (p.polar_weight * p.polar_sin)[None, :]          # [T][P]
        k, phi, psi = 1.0, np.ones((pair.R, pair.G)), np.zeros((pair.T, 2, pair.P, pair.G))
        fed = t.link.reshape(-1)
        fed = fed[fed >= 0]                                                                               # entries a linked exit feeds
        for it in range(n_it):
            F = oracle.fission_rate(p.mesh.material, p.xs.nu_sigma_f, t.volume, phi)
            phi, psi = phi / F, psi / F
            Q = oracle.source(p.mesh.material, p.xs.sigma_s, p.xs.nu_sigma_f, p.xs.chi, phi, k)
            phi_new, psi_next, tally = pair.oracle_sweep(Q, psi)
            w_e = np.repeat(w_tp, 2, axis=0).reshape(pair.T, 2, pair.P)                                  # weight of entry (t, d)
            s_in = np.einsum("tdp,tdpg->", w_e, psi)
            out_linked = np.einsum("ep,epg->", w_e.reshape(-1, pair.P)[fed], psi_next.reshape(-1, pair.P, pair.G)[fed])
            leak_o = s_in - tally.sum() - out_linked
            k *= oracle.fission_rate(p.mesh.material, p.xs.nu_sigma_f, t.volume, phi_new)
            phi, psi = phi_new, psi_next
            st = out["stats"][it]
            assert abs(st["k_eff"] - k) * 1e5 <= K_PCM
            if 0 in p.bc:
                assert leak_o > 0 and abs(st["leakage"] - leak_o) <= 2e-5 * leak_o, (it, st["leakage"], leak_o)
            else:
                assert st["leakage"] == 0.0 and abs(leak_o) <= 1e-9 * max(abs(tally.sum()), 1e-30)
            assert abs(st["balance_residual"]) <= 2e-6, st["balance_residual"]
    finally:
        pair.close()


def test_iteration_stats_beyond_one_ring():
    """More iterations than the device ring of stats records holds (4096): every record is delivered."""
    pair = make_pair(1, 1.0)
    try:
        n = 4096 + 700
        out = pair.gpu.nd_power_iteration(n, want_stats=True)
        ks = np.array([s["k_eff"] for s in out["stats"]])
        assert out["iters"] == n and len(ks) == n and np.all(ks > 0)
        assert ks[-1] == out["k_eff"]
        ko, _, _, hist = pair.oracle_power(60)
        assert np.abs(ks[:60] - hist).max() * 1e5 <= K_PCM
        assert abs(ks[4095] - ks[4096]) < 1e-7 and abs(ks[-1] - ks[4096]) < 1e-7    # converged long before (FP32 chains: ~1e-9 jitter); no seam at the ring edge
    finally:
        pair.close()


def test_power_iteration_tolerance_mode_and_reset():
    pair = make_pair(1, 1.0)
    try:
        out = pair.gpu.nd_power_iteration(2000, tol_k=1e-7, tol_phi=1e-6)
        assert out["converged"] and out["iters"] < 2000
        k1 = out["k_eff"]
        out_nc = pair.gpu.nd_power_iteration(1, tol_k=1e-30)
        assert not out_nc["converged"]
        pair.gpu.nd_state_reset()
        out = pair.gpu.nd_power_iteration(50)
        ko, *_ = pair.oracle_power(50)
        assert abs(out["k_eff"] - ko) * 1e5 <= K_PCM
        assert abs(k1 - ko) < 5e-3
    finally:
        pair.close()


@pytest.mark.parametrize("case", [(1, 1.0), (2, 0.15), (4, 0.06)], ids=["cfg1", "cfg2", "cfg4"])
def test_power_iteration_graph_replay_matches_plain_launches(case):
    """Fixed-count calls of >= 4 iterations replay a CUDA graph of two iterations (nd_options.graph_mode 0); the result,
    the iteration count and the launch count are those of the plain launches (graph_mode 1), also when plain and
    replayed calls are mixed so that an odd iteration comes first, and after a reset."""
    import time
    import torch
    a = make_pair(case[0], case[1])
    b = make_pair(case[0], case[1], graph_mode=1)
    try:
        for g in (a.gpu, b.gpu):
            g.nd_profile_enable(0)
        seq = [3, 9, 4, 1, 6]                     # 3 plain, odd start + pairs, pairs, plain, pairs
        for n in seq:
            oa, ob = a.gpu.nd_power_iteration(n), b.gpu.nd_power_iteration(n)
            assert oa["iters"] == ob["iters"] == n
            assert abs(oa["k_eff"] - ob["k_eff"]) < 1e-9 * abs(ob["k_eff"])
        pa, pb = a.gpu.nd_flux_get().cpu().numpy(), b.gpu.nd_flux_get().cpu().numpy()
        assert np.max(np.abs(pa - pb) / np.maximum(np.abs(pb), 1e-6 * np.abs(pb).max())) < 1e-6
        assert a.gpu.nd_profile_read()["kernels_launched"] == b.gpu.nd_profile_read()["kernels_launched"] > 0
        ko, *_ = a.oracle_power(sum(seq))
        assert abs(oa["k_eff"] - ko) * 1e5 <= K_PCM
        for g in (a.gpu, b.gpu):
            g.nd_state_reset()
        assert abs(a.gpu.nd_power_iteration(8)["k_eff"] - b.gpu.nd_power_iteration(8)["k_eff"]) < 1e-9
        a.gpu.nd_profile_enable(1)                # profiling on: plain launches again, sweep events recorded
        a.gpu.nd_power_iteration(6)
        assert a.gpu.nd_profile_read()["sweep_launches"] == 6
        a.gpu.nd_profile_enable(0)
        t = []
        for g in (a.gpu, b.gpu):
            g.nd_power_iteration(40)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            g.nd_power_iteration(200)
            torch.cuda.synchronize()
            t.append((time.perf_counter() - t0) / 200 * 1e3)
        print(f"cfg{case[0]}: {t[0]:.4f} ms / iteration replayed, {t[1]:.4f} ms plain")
    finally:
        a.close()
        b.close()


def test_infinite_medium_closed_form_on_gpu():
    """Homogeneous reflective rectangle: k -> nuSf^T (diag(St) - S)^-1 chi (closed form, not the oracle)."""
    mesh = rect_tri_mesh(1.5, 1.5, 4, 4, seed=2, jitter=0.2)
    mesh.material[:] = 0
    xs = homogeneous_xs(4, 21, n_up=2)
    s, w = tabuchi_yamamoto(3)
    tr = nd.nd_tracks_generate(mesh.xy, mesh.tri, mesh.W, mesh.H, (1, 1, 1, 1), 8, 0.1)
    gp = nd.nd_problem_create(xs, s, w, mesh.material, tr)
    out = gp.nd_power_iteration(3000, tol_k=1e-9, tol_phi=1e-7)
    A = np.diag(xs.sigma_t[0]) - xs.sigma_s[0]
    k_inf = float(xs.nu_sigma_f[0] @ np.linalg.solve(A, xs.chi[0]))
    assert abs(out["k_eff"] - k_inf) * 1e5 <= K_PCM
    gp.destroy()


def test_problem_create_rejects_on_device_side_errors():
    pair = make_pair(1, 1.0)
    try:
        with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
            pair.gpu.nd_source_update(torch.ones((pair.R, pair.G), dtype=torch.float64, device="cuda"), -1.0)
        info = pair.gpu.nd_problem_info_get()
        assert info["n_segments"] == pair.o_tr.n_segs
        assert info["updates_per_sweep"] == 2 * pair.o_tr.n_segs * pair.P * pair.G
    finally:
        pair.close()


def test_pure_absorber_fixed_source_closed_form_on_gpu():
    """Fixed-source mode against mathematics, not the oracle: pure absorber (Sigma_s = 0), uniform isotropic emission
    density q0, reflective box -> phi = q0 / Sigma_a in every region and group once the boundary flux has converged."""
    mesh = rect_tri_mesh(1.3, 0.9, 5, 4, seed=8, jitter=0.25)
    mesh.material[:] = 0
    G = 3
    xs = homogeneous_xs(G, 5)
    xs.sigma_s[:] = 0.0
    xs.nu_sigma_f[:] = 0.0
    s, w = tabuchi_yamamoto(3)
    tr = nd.nd_tracks_generate(mesh.xy, mesh.tri, mesh.W, mesh.H, (1, 1, 1, 1), 16, 0.03)
    gp = nd.nd_problem_create(xs, s, w, mesh.material, tr)
    try:
        q0 = np.array([1.0, 0.4, 2.5])
        Q = torch.from_numpy(np.tile(q0 / (4.0 * np.pi), (mesh.n_regions, 1))).cuda()
        gp.nd_boundary_flux_fill(0.0)
        for _ in range(400):                       # the boundary flux advances one track per sweep
            phi = gp.nd_transport_sweep(Q)
        expect = q0 / xs.sigma_t[0]
        assert np.abs(phi.cpu().numpy() / expect - 1.0).max() <= 2e-5
    finally:
        gp.destroy()
        tr.destroy()


def test_vacuum_rectangle_worked_example_on_gpu():
    """The worked example of tests/golden/vacuum_rectangle.txt through the CUDA path: homogeneous 2 x 1.5 cm
    rectangle, Sigma_t = Sigma_a = 1, unit emission density, vacuum on all sides, N_a = 64, 0.01 cm, TY-3, one sweep:
    the track-volume weighted mean flux is 0.57485289 whatever the triangulation."""
    import os
    golden = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "vacuum_rectangle.txt")):
        if line.strip() and not line.lstrip().startswith("#"):
            k, v = line.split()[:2]
            golden[k] = float(v)
    target = golden["phi_bar"]
    assert (golden["W"], golden["H"], golden["n_azim"], golden["spacing"], golden["n_polar"]) == (2.0, 1.5, 64, 0.01, 3)
    mesh = rect_tri_mesh(2.0, 1.5, 6, 5, seed=4, jitter=0.3)
    mesh.material[:] = 0
    xs = homogeneous_xs(1, 1)
    xs.sigma_t[:] = 1.0
    xs.sigma_s[:] = 0.0
    xs.nu_sigma_f[:] = 0.0
    s, w = tabuchi_yamamoto(3)
    tr = nd.nd_tracks_generate(mesh.xy, mesh.tri, mesh.W, mesh.H, (0, 0, 0, 0), 64, 0.01)
    gp = nd.nd_problem_create(xs, s, w, mesh.material, tr)
    try:
        Q = torch.full((mesh.n_regions, 1), 1.0 / (4.0 * np.pi), dtype=torch.float64, device="cuda")
        phi = gp.nd_transport_sweep(Q).cpu().numpy()[:, 0]
        vol = gp.nd_track_volume_get()
        assert abs(float((phi * vol).sum() / vol.sum()) - target) <= 2e-6
    finally:
        gp.destroy()
        tr.destroy()


@pytest.mark.parametrize("case", [(3, 0.3, {}), (4, 0.5, {}), (5, 0.02, {}), (5, 0.01, dict(block_warps=16, tile_segments=6, delta_buffers=2))],
                         ids=["cfg3", "cfg4", "cfg5", "cfg5-2buf"])
def test_swath_sweep_is_reproducible(case):
    """Race check by repetition: the segment chains and the per-tile FP32 sums have a fixed order, so the boundary flux
    must come back BIT-identical run after run and the tally may differ only by the order of the FP64 REDs.  A
    shared-memory hazard (staging buffers, delta buffer, barriers) would show up here as run-to-run differences."""
    idx, scale, opts = case
    prob = make_config(idx, scale=scale)
    m = prob.mesh
    tr = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    gp = nd.nd_problem_create(prob.xs, prob.polar_sin, prob.polar_weight, m.material, tr, sweep_kernel=nd.ND_SWEEP_SWATH, **opts)
    try:
        rng = np.random.default_rng(77)
        Q = torch.from_numpy(rng.uniform(0.05, 1.0, size=(m.n_regions, prob.n_groups))).cuda()
        psi0 = rng.uniform(0.0, 2.0, size=(tr.n_tracks, 2, prob.n_polar, prob.n_groups)).astype(np.float32)
        ref_psi = ref_tally = None
        for _ in range(6):
            gp.nd_boundary_flux_set(psi0)
            gp.nd_transport_sweep(Q)
            psi = gp.nd_boundary_flux_get()
            tally = gp.nd_tally_get().cpu().numpy()
            if ref_psi is None:
                ref_psi, ref_tally = psi, tally
            else:
                assert np.array_equal(psi, ref_psi), "boundary flux differs between identical runs"
                assert np.abs(tally - ref_tally).max() <= 1e-12 * np.abs(ref_tally).max()
    finally:
        gp.destroy()
        tr.destroy()


def test_phase_profile_of_the_instrumented_swath_kernel():
    pair = make_pair(4, 0.06, sweep_kernel=nd.ND_SWEEP_SWATH)
    try:
        with pytest.raises(nd.NdError, match="ND_ERR_STATE"):
            pair.gpu.nd_sweep_phases_get()
        ko, *_ = pair.oracle_power(4)
        pair.gpu.nd_profile_enable(2)
        out = pair.gpu.nd_power_iteration(4)           # the instrumented build computes the same thing
        assert abs(out["k_eff"] - ko) * 1e5 <= K_PCM
        ph = pair.gpu.nd_sweep_phases_get()
        assert abs(sum(ph.values()) - 1.0) < 1e-9 and all(v >= 0.0 for v in ph.values())
        assert ph["segment_loop"] == max(ph.values())
        pair.gpu.nd_profile_enable(0)
    finally:
        pair.close()
