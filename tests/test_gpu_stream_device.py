"""SURVEY 8(f) NEXT-1, second half: the set-up with NO segment on the host.  nd_tracks_generate_resident leaves the traced
segments in device memory; nd_problem_create (nd_problem_desc.seg_on_device = 1) validates them, forms A~_r and builds the
kernels' segment streams on the GPU.  Checked here:
  - the resident segments equal the host tracer's and the oracle's tracer's bit for bit, the atomically summed areas to
    rounding;
  - the chunk stream of the device builder equals the host builder's BYTE FOR BYTE (blob, tile references, swath table, work
    items), over tile shapes, cut rules and configurations -- the host builder is itself decoded against the descriptor in
    tests/test_swath_stream.py;
  - sweeps and power iterations of a device-built problem against the oracle and against the host-built problem;
  - the error paths (bad region id, bad length, missing geometry, workspace too small) and the consumers of host segments
    (CMFD surfaces, shards) through nd_tracks_materialise."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
import paper_2607_01591_b200 as nd
from gpu_common import make_pair, seeded_sweep_inputs, phi_rel_err, PHI_RTOL, K_PCM
from moc_inputs import make_config, rect_tri_mesh

pytestmark = pytest.mark.gpu


def _resident(prob, **kw):
    m = prob.mesh
    return nd.nd_tracks_generate_resident(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing, **kw)


def _create(prob, tracks, **options):
    return nd.nd_problem_create(prob.xs, prob.polar_sin, prob.polar_weight, prob.mesh.material, tracks, **options)


@pytest.mark.parametrize("idx,scale", [(1, 1.0), (2, 0.3), (3, 0.05), (4, 0.1), (5, 0.002)])
def test_resident_segments_are_bit_exact(idx, scale):
    prob = make_config(idx, scale=scale)
    m = prob.mesh
    o = oracle.generate_tracks(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    h = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    d = _resident(prob)
    try:
        assert d.seg_device is not None and not d.on_host
        assert d.n_segments == o.n_segs == h.n_segments
        for f in ("seg_offset", "track_weight", "link", "track_azim", "ends", "azim_phi", "azim_weight", "azim_spacing"):
            assert getattr(d, f).tobytes() == getattr(h, f).tobytes(), f
        # the areas: FP64 atomics in an order that differs from the canonical one
        assert np.abs(d.volume - h.volume).max() <= 1e-13 * h.volume.max()
        # straight from device memory, before anything is materialised
        S = d.n_segments
        ws, base = d.device_workspace, d.device_workspace.data_ptr()
        reg = ws[d.seg_device[0] - base:d.seg_device[0] - base + 4 * S].cpu().numpy().view(np.int32)
        length = ws[d.seg_device[1] - base:d.seg_device[1] - base + 8 * S].cpu().numpy().view(np.float64)
        assert reg.tobytes() == o.seg_region.tobytes() == h.seg_region.tobytes()
        assert length.tobytes() == o.seg_length.tobytes() == h.seg_length.tobytes()
        assert not d.on_host
        assert d.seg_region.tobytes() == h.seg_region.tobytes() and d.seg_length.tobytes() == h.seg_length.tobytes()   # materialises
        assert d.on_host
    finally:
        h.destroy()
        d.destroy()


def test_resident_workspace_is_sized_by_a_second_call():
    prob = make_config(3, scale=0.2)             # 6e6 segments: more than the 2^20 the minimum workspace holds
    a = _resident(prob)
    b = _resident(prob, segment_estimate=1)      # far too small: ND_ERR_WORKSPACE reports the size, the binding retries
    try:
        assert a.n_segments > 1 << 21
        assert a.timing["attempts"] == 1, "the mean-chord estimate should suffice"
        assert b.timing["attempts"] == 2
        assert a.seg_region.tobytes() == b.seg_region.tobytes() and a.seg_length.tobytes() == b.seg_length.tobytes()
    finally:
        a.destroy()
        b.destroy()


STREAM_FIELDS = ("blob", "tile_ref", "swath_tile0", "swath_track", "items")
STREAM_CASES = [
    ((1, 1.0), {}),
    ((2, 0.3), {}),
    ((3, 0.05), {}),
    ((3, 0.05), dict(tile_lag=-1)),                        # always geometric cuts
    ((3, 0.03), dict(block_warps=4, tile_segments=6, window_regions=24)),
    ((4, 0.1), {}),
    ((4, 0.1), dict(cmfd_stream=1)),
    ((4, 0.06), dict(item_order=1)),
    ((5, 0.002), {}),
    ((5, 0.002), dict(q_copies=1, tile_lag=3)),
    ((3, 0.05), dict(p1_stream=1)),                        # the larger shared-memory layout of the P_1 sweep: shorter tiles
    ((5, 0.002), dict(p1_stream=1)),
]


@pytest.mark.parametrize("case,opts", STREAM_CASES, ids=[f"cfg{c[0]}-{'-'.join(f'{k}{v}' for k, v in o.items()) or 'default'}" for c, o in STREAM_CASES])
def test_device_built_stream_equals_the_host_built_stream_byte_for_byte(case, opts):
    prob = make_config(case[0], scale=case[1])
    tr = _resident(prob)
    g_dev = _create(prob, tr, sweep_kernel=nd.ND_SWEEP_SWATH, **opts)
    g_host = _create(prob, tr, sweep_kernel=nd.ND_SWEEP_SWATH, host_build=True, **opts)   # materialises, host builder
    try:
        a, b = g_dev.nd_problem_stream_view(), g_host.nd_problem_stream_view()
        assert a["built_on_device"] and not b["built_on_device"]
        assert a["n_tiles"] == b["n_tiles"] > 0 and a["n_swaths"] == b["n_swaths"] > 0
        for f in STREAM_FIELDS:
            assert a[f].shape == b[f].shape, f
            assert a[f].tobytes() == b[f].tobytes(), f"{f} differs"
        ia, ib = g_dev.nd_problem_info_get(), g_host.nd_problem_info_get()
        for f in ("n_batches", "mean_regions_per_tile", "mean_segments_per_tile", "lockstep_efficiency", "smem_bytes", "grid_blocks"):
            assert ia[f] == ib[f], f
    finally:
        g_dev.destroy(); g_host.destroy(); tr.destroy()


@pytest.mark.parametrize("kernel", [nd.ND_SWEEP_ATOMIC, nd.ND_SWEEP_SWATH], ids=["atomic", "swath"])
@pytest.mark.parametrize("case", [(3, 0.05), (4, 0.1), (5, 0.002)], ids=["cfg3", "cfg4", "cfg5"])
def test_device_built_problem_sweeps_like_the_oracle_and_the_host_built_problem(case, kernel):
    pair = make_pair(*case, sweep_kernel=kernel)
    tr = _resident(pair.prob)
    g = _create(pair.prob, tr, sweep_kernel=kernel)
    try:
        assert np.abs(g.nd_track_volume_get() - pair.gpu.nd_track_volume_get()).max() <= 1e-13 * pair.gpu.nd_track_volume_get().max()
        Q, psi = seeded_sweep_inputs(pair, 11)
        dQ = torch.from_numpy(Q).cuda()
        g.nd_boundary_flux_set(psi)
        pair.gpu.nd_boundary_flux_set(psi)
        phi_d = g.nd_transport_sweep(dQ).cpu().numpy()
        phi_h = pair.gpu.nd_transport_sweep(dQ).cpu().numpy()
        # the same stream, the same FP32 arithmetic: the boundary fluxes are bit-equal, the flux differs by the order of the
        # FP64 tally atomics and by the last bits of A~_r
        assert g.nd_boundary_flux_get().tobytes() == pair.gpu.nd_boundary_flux_get().tobytes()
        assert np.abs(phi_d - phi_h).max() <= 1e-11 * np.abs(phi_h).max()
        phi_o, _, _ = pair.oracle_sweep(Q, psi.astype(np.float64))
        assert phi_rel_err(phi_d, phi_o) <= PHI_RTOL
    finally:
        g.destroy(); tr.destroy(); pair.close()


def test_device_built_problem_power_iteration_against_the_oracle():
    pair = make_pair(3, 0.05)
    tr = _resident(pair.prob)
    g = _create(pair.prob, tr)                       # ND_SWEEP_AUTO: the swath kernel (geometry present)
    try:
        assert g.nd_problem_info_get()["sweep_kernel"] == nd.ND_SWEEP_SWATH
        n = 12
        out = g.nd_power_iteration(n, want_stats=True)
        ko, *_ = pair.oracle_power(n)
        assert abs(out["k_eff"] - ko) * 1e5 <= K_PCM
        host = pair.gpu.nd_power_iteration(n)
        assert abs(out["k_eff"] - host["k_eff"]) <= 1e-9
    finally:
        g.destroy(); tr.destroy(); pair.close()


def test_volume_formed_on_the_device_when_the_descriptor_brings_none():
    prob = make_config(4, scale=0.06)
    tr = _resident(prob)
    h = nd.nd_tracks_generate(prob.mesh.xy, prob.mesh.tri, prob.mesh.W, prob.mesh.H, prob.bc, prob.n_azim, prob.spacing)
    xs, m = prob.xs, prob.mesh
    g = nd.Problem(m.material, xs.sigma_t, xs.sigma_s, xs.nu_sigma_f, xs.chi, prob.polar_sin, prob.polar_weight, tr.seg_offset,
                   None, None, tr.track_weight, tr.link, track_azim=tr.track_azim, track_ends=tr.ends, seg_device=tr.seg_device)
    try:
        v = g.nd_track_volume_get()
        assert np.abs(v - h.volume).max() <= 1e-13 * h.volume.max() and v.min() > 0
    finally:
        g.destroy(); tr.destroy(); h.destroy()


def test_device_segments_are_validated_on_the_device():
    prob = make_config(1)
    tr = _resident(prob)
    S = tr.n_segments
    ws, base = tr.device_workspace, tr.device_workspace.data_ptr()
    reg = ws[tr.seg_device[0] - base:tr.seg_device[0] - base + 4 * S].view(torch.int32)
    length = ws[tr.seg_device[1] - base:tr.seg_device[1] - base + 8 * S].view(torch.float64)
    try:
        for kernel in (nd.ND_SWEEP_ATOMIC, nd.ND_SWEEP_SWATH):
            keep = int(reg[S // 2])
            reg[S // 2] = prob.mesh.n_regions
            with pytest.raises(nd.NdError, match="ND_ERR_RANGE"):
                _create(prob, tr, sweep_kernel=kernel)
            reg[S // 2] = -1
            with pytest.raises(nd.NdError, match="ND_ERR_RANGE"):
                _create(prob, tr, sweep_kernel=kernel)
            reg[S // 2] = keep
            keep = float(length[S - 1])
            for bad in (0.0, -1.0, float("nan"), float("inf")):
                length[S - 1] = bad
                with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
                    _create(prob, tr, sweep_kernel=kernel)
            length[S - 1] = keep
            _create(prob, tr, sweep_kernel=kernel).destroy()
        xs, m = prob.xs, prob.mesh
        with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):      # no geometry
            nd.Problem(m.material, xs.sigma_t, xs.sigma_s, xs.nu_sigma_f, xs.chi, prob.polar_sin, prob.polar_weight, tr.seg_offset,
                       None, None, tr.track_weight, tr.link, seg_device=tr.seg_device)
    finally:
        tr.destroy()


def test_cmfd_and_shards_on_resident_tracks():
    # the consumers of HOST segments (nd_cmfd_surfaces, nd_cmfd_create, nd_tracks_shard) behind nd_tracks_materialise; the
    # crossing lists of the current tally come from the slot_start arrays the DEVICE builder wrote
    from moc_inputs.coarse import cartesian_cells
    pair = make_pair(4, 0.1, sweep_kernel=nd.ND_SWEEP_SWATH, cmfd_stream=1)
    tr = _resident(pair.prob)
    g = _create(pair.prob, tr, sweep_kernel=nd.ND_SWEEP_SWATH, cmfd_stream=1)
    try:
        assert g.nd_problem_stream_view()["built_on_device"] and not tr.on_host
        n_cells = 36
        cell = cartesian_cells(pair.prob.mesh, 6, 6)
        lo, hi = nd.nd_cmfd_surfaces(tr.seg_offset, tr.seg_region, tr.link, cell, n_cells)
        assert tr.on_host
        hlo, hhi = nd.nd_cmfd_surfaces(pair.g_tr.seg_offset, pair.g_tr.seg_region, pair.g_tr.link, cell, n_cells)
        assert np.array_equal(lo, hlo) and np.array_equal(hi, hhi)
        plans = [p.nd_cmfd_create(t.seg_offset, t.seg_region, t.link, cell, n_cells, lo, hi, np.zeros(len(lo)))
                 for p, t in ((g, tr), (pair.gpu, pair.g_tr))]
        Q, psi = seeded_sweep_inputs(pair, 3)
        dQ = torch.from_numpy(Q).cuda()
        J = []
        for p, plan in zip((g, pair.gpu), plans):
            p.nd_boundary_flux_set(psi)
            plan.nd_cmfd_sweep(dQ)
            J.append(plan.nd_cmfd_currents_get())
        for a, b in zip(J[0], J[1]):
            assert np.abs(a - b).max() <= 1e-11 * max(np.abs(b).max(), 1e-300)
        sh = tr.shard(2, 1)
        sh_h = pair.g_tr.shard(2, 1)
        assert sh.seg_region.tobytes() == sh_h.seg_region.tobytes() and sh.seg_length.tobytes() == sh_h.seg_length.tobytes()
        sh.destroy(); sh_h.destroy()
        for plan in plans:
            plan.destroy()
    finally:
        g.destroy(); tr.destroy(); pair.close()
