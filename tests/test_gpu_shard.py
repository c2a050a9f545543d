"""NEXT-2 on ONE GPU: problems built from the shards of an angle-pair partition against the unsharded
problem and against the oracle.  (i) the shards' tallies of one sweep add up to the unsharded tally, every boundary flux
bit-equal; (ii) the reducer hook sits between the sweep and the flux; (iii) two shard problems iterated in lock step --
one host thread each, the reducer a host barrier that adds the two tallies -- follow the unsharded k history and the
oracle's.  No kernel waits for another kernel: the threads meet on the host after synchronising their streams."""
import threading

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import paper_2607_01591_b200 as nd
from gpu_common import make_pair, seeded_sweep_inputs, phi_rel_err, PHI_RTOL, K_PCM

pytestmark = pytest.mark.gpu


def _shard_problems(pair, n_shards, **options):
    p = pair.prob
    out = []
    for s in range(n_shards):
        tr = pair.g_tr.shard(n_shards, s)
        out.append((tr, nd.nd_problem_create(p.xs, p.polar_sin, p.polar_weight, p.mesh.material, tr, **options)))
    return out


@pytest.mark.parametrize("kernel,opts", [(nd.ND_SWEEP_ATOMIC, {}), (nd.ND_SWEEP_SWATH, dict(block_warps=4))], ids=["atomic", "swath"])
@pytest.mark.parametrize("case,n_shards", [((3, 0.03), 2), ((4, 0.06), 3), ((5, 0.0008), 4)], ids=["cfg3", "cfg4", "cfg5"])
def test_shard_tallies_add_up_to_the_unsharded_sweep(case, n_shards, kernel, opts):
    pair = make_pair(*case, sweep_kernel=kernel, **opts)
    shards = _shard_problems(pair, n_shards, sweep_kernel=kernel, **opts)
    try:
        Q, psi = seeded_sweep_inputs(pair, 77)
        dQ = torch.from_numpy(Q).cuda()
        pair.gpu.nd_boundary_flux_set(psi)
        phi_full = pair.gpu.nd_transport_sweep(dQ).cpu().numpy()
        tally_full = pair.gpu.nd_tally_get().cpu().numpy()
        psi_full = pair.gpu.nd_boundary_flux_get()
        tally_sum = np.zeros_like(tally_full)
        for tr, gp in shards:
            assert gp.nd_track_volume_get().tobytes() == pair.gpu.nd_track_volume_get().tobytes()
            gp.nd_boundary_flux_set(psi[tr.track_global])
            gp.nd_transport_sweep(dQ)
            tally_sum += gp.nd_tally_get().cpu().numpy()
            assert gp.nd_boundary_flux_get().tobytes() == psi_full[tr.track_global].tobytes(), "boundary flux bit-equal"
        # atomic kernel: the same FP32 contributions summed in FP64 in another order.  Swath kernel: a tile's FP32 partial sums
        # depend on where the tiles are cut, and the cut rule looks at the mean segment length of the problem's own tracks
        tol = 1e-12 if kernel == nd.ND_SWEEP_ATOMIC else 2e-7
        assert np.abs(tally_sum - tally_full).max() <= tol * np.abs(tally_full).max()
        phi_o, _, _ = pair.oracle_sweep(Q, psi.astype(np.float64))
        assert phi_rel_err(phi_full, phi_o) <= PHI_RTOL
    finally:
        for tr, gp in shards:
            gp.destroy(); tr.destroy()
        pair.close()


def test_reducer_is_called_between_the_sweep_and_the_flux():
    pair = make_pair(3, 0.03, block_warps=4)            # the same tile shapes in every problem: identical FP32 partial sums
    shards = _shard_problems(pair, 2, block_warps=4)
    try:
        Q, psi = seeded_sweep_inputs(pair, 5)
        dQ = torch.from_numpy(Q).cuda()
        pair.gpu.nd_boundary_flux_set(psi)
        phi_full = pair.gpu.nd_transport_sweep(dQ).cpu().numpy()
        (tr0, g0), (tr1, g1) = shards
        g1.nd_boundary_flux_set(psi[tr1.track_global])
        g1.nd_transport_sweep(dQ)
        calls = []

        def add_other(tally):            # what an all-reduce does for shard 0: add shard 1's tally, in stream order
            calls.append(tally.numel())
            tally += other
        g0.nd_boundary_flux_set(psi[tr0.track_global])
        g0.nd_transport_sweep(dQ)        # no reducer yet: the partial flux
        Gs = (pair.G + 3) // 4 * 4
        other = torch.zeros(pair.R * Gs, dtype=torch.float64, device="cuda")
        other.view(pair.R, Gs)[:, :pair.G] = g1.nd_tally_get()
        g0.nd_tally_reducer_set(add_other)
        g0.nd_boundary_flux_set(psi[tr0.track_global])
        phi0 = g0.nd_transport_sweep(dQ).cpu().numpy()
        assert calls == [pair.R * Gs]
        assert phi_rel_err(phi0, phi_full) <= 2e-7       # FP32 partial sums of differently cut tiles
        g0.nd_tally_reducer_set(None)
        g0.nd_boundary_flux_set(psi[tr0.track_global])
        phi_part = g0.nd_transport_sweep(dQ).cpu().numpy()
        assert len(calls) == 1 and np.abs(phi_part - phi_full).max() > 1e-3 * np.abs(phi_full).max()
    finally:
        for tr, gp in shards:
            gp.destroy(); tr.destroy()
        pair.close()


@pytest.mark.parametrize("case", [(3, 0.03), (2, 0.15)], ids=["cfg3", "cfg2"])
def test_two_shards_iterate_in_lock_step(case):
    pair = make_pair(*case, block_warps=4)
    shards = _shard_problems(pair, 2, block_warps=4)
    try:
        n_it = 12
        barrier = threading.Barrier(2)
        views = [None, None]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        results = [None, None]
        errors = []

        def make_reducer(i):
            def reduce(tally):
                views[i] = tally
                torch.cuda.current_stream().synchronize()      # my sweep is done
                barrier.wait()
                total = views[0] + views[1]                    # both threads form the same sum from the same two arrays
                torch.cuda.current_stream().synchronize()
                barrier.wait()                                 # nobody overwrites before both have read
                tally.copy_(total)
            return reduce

        def run(i):
            try:
                with torch.cuda.stream(streams[i]):
                    gp = shards[i][1]
                    gp.nd_tally_reducer_set(make_reducer(i))
                    dphi = torch.empty((pair.R, pair.G), dtype=torch.float64, device="cuda")
                    out = gp.nd_power_iteration(n_it, d_phi_out=dphi, want_stats=True)
                    torch.cuda.current_stream().synchronize()
                    results[i] = (out, dphi.cpu().numpy())
            except Exception as e:                             # pragma: no cover
                errors.append(e)
                barrier.abort()
        th = [threading.Thread(target=run, args=(i,)) for i in range(2)]
        for t in th:
            t.start()
        for t in th:
            t.join(timeout=300)
        assert not errors, errors
        ref = pair.gpu.nd_power_iteration(n_it, want_stats=True)
        ko, phio, _, hist = pair.oracle_power(n_it)
        k_ref = np.array([s["k_eff"] for s in ref["stats"]])
        for out, phi in results:
            ks = np.array([s["k_eff"] for s in out["stats"]])
            assert np.abs(ks - k_ref).max() < 2e-7, "sharded = unsharded up to the summation order of the tallies"
            assert np.abs(ks - hist).max() * 1e5 <= K_PCM
            assert phi_rel_err(phi, phio) <= PHI_RTOL
        assert results[0][0]["k_eff"] == results[1][0]["k_eff"], "every shard computes the same k from the same reduced tally"
        assert np.array_equal(results[0][1], results[1][1])
    finally:
        for tr, gp in shards:
            gp.nd_tally_reducer_set(None)
            gp.destroy(); tr.destroy()
        pair.close()
