"""Host logic of NEXT-2 (angle-pair sharding; no GPU): nd_tracks_shard partitions a cyclic laydown into
shards that own whole angle pairs {j, N_a/2-1-j}, so no link leaves a shard; and the world_size-2 gloo check that the sum
of the shards' tallies, each swept by the ORACLE on its own shard, equals the unsharded tally after one FP64 all-reduce --
the only collective the sharded path has."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import paper_2607_01591_b200 as nd
from moc_inputs import make_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("idx,scale,n_shards", [(2, 0.15, 2), (3, 0.03, 4), (4, 0.06, 3), (5, 0.0008, 16), (1, 1.0, 2)])
def test_shards_partition_the_laydown(idx, scale, n_shards):
    prob = make_config(idx, scale=scale)
    m = prob.mesh
    full = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    nh = full.n_half
    seen = np.zeros(full.n_tracks, int)
    seg_per_shard = []
    for s in range(n_shards):
        sh = full.shard(n_shards, s)
        g = sh.track_global
        assert sh.n_tracks == len(g) > 0 and np.all(np.diff(g) > 0), "canonical order kept"
        seen[g] += 1
        # whole angle pairs
        ang = set(full.track_azim[g].tolist())
        assert all((nh - 1 - j) in ang for j in ang)
        assert np.array_equal(np.isin(full.track_azim, list(ang)), np.isin(np.arange(full.n_tracks), g))
        # per-track data copied, links remapped and closed inside the shard
        assert np.array_equal(sh.track_weight, full.track_weight[g]) and np.array_equal(sh.track_azim, full.track_azim[g])
        assert np.array_equal(sh.ends, full.ends[g])
        for lt, t in enumerate(g):
            k0, k1 = full.seg_offset[t], full.seg_offset[t + 1]
            a0, a1 = sh.seg_offset[lt], sh.seg_offset[lt + 1]
            assert a1 - a0 == k1 - k0
            assert np.array_equal(sh.seg_region[a0:a1], full.seg_region[k0:k1])
            assert sh.seg_length[a0:a1].tobytes() == full.seg_length[k0:k1].tobytes()
        lk_full = full.link[g]                                            # [n][2] global chain ids or -1
        lk = sh.link
        assert np.array_equal(lk < 0, lk_full < 0)
        ok = lk >= 0
        assert np.array_equal(g[lk[ok] // 2] * 2 + lk[ok] % 2, lk_full[ok])
        # the areas of the WHOLE laydown
        assert sh.volume.tobytes() == full.volume.tobytes()
        seg_per_shard.append(sh.n_segments)
        sh.destroy()
    assert np.all(seen == 1), "every track in exactly one shard"
    assert sum(seg_per_shard) == full.n_segments
    # balance: longest-first dealing keeps the largest shard within one pair's worth of the mean
    pair_seg = np.zeros(nh // 2)
    np.add.at(pair_seg, np.minimum(full.track_azim, nh - 1 - full.track_azim), np.diff(full.seg_offset))
    assert max(seg_per_shard) <= full.n_segments / n_shards + pair_seg.max()
    full.destroy()


def test_shard_argument_checks():
    prob = make_config(1, 1.0)                       # N_a = 8: two angle pairs
    m = prob.mesh
    full = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        full.shard(3, 0)                             # more shards than pairs
    with pytest.raises(nd.NdError, match="ND_ERR_INVALID"):
        full.shard(2, 2)
    sh = full.shard(2, 1)
    with pytest.raises(nd.NdError, match="ND_ERR_STATE"):
        sh.shard(2, 0)                               # a shard cannot be sharded again
    one = full.shard(1, 0)
    assert one.n_tracks == full.n_tracks and np.array_equal(one.link, full.link)


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import oracle, paper_2607_01591_b200 as nd
from moc_inputs import make_config
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
prob = make_config(3, scale=0.03)
m = prob.mesh
full = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
sh = full.shard(2, rank)
rng = np.random.default_rng(7)
R, G, P = m.n_regions, prob.n_groups, prob.n_polar
Q = rng.uniform(0.05, 1.0, (R, G))
psi_full = rng.uniform(0.0, 1.0, (full.n_tracks, 2, P, G))
def sweep(tr, psi, vol):
    return oracle.sweep(m.material, prob.xs.sigma_t, prob.polar_sin, prob.polar_weight, tr.seg_offset, tr.seg_region,
                        tr.seg_length, tr.track_weight, tr.link, vol, Q, psi)
_, psi_s, tally_s = sweep(sh, psi_full[sh.track_global], full.volume)
t = torch.from_numpy(tally_s.copy())
dist.all_reduce(t)                                   # the one collective of the sharded path: FP64 sum of the tally
phi_f, psi_f, tally_f = sweep(full, psi_full, full.volume)
st = prob.xs.sigma_t[m.material]
phi_s = 4 * np.pi * Q / st + t.numpy() / (st * full.volume[:, None])      # O-6 finalise with the reduced tally
out = dict(rank=rank, tally=float(np.abs(t.numpy() - tally_f).max() / np.abs(tally_f).max()),
           phi=float(np.abs(phi_s - phi_f).max() / np.abs(phi_f).max()),
           psi=bool(np.array_equal(psi_s, psi_f[sh.track_global])), n=int(sh.n_tracks))
dist.barrier(); dist.destroy_process_group()
print(json.dumps(out))
"""


def test_two_gloo_ranks_sum_their_shards_tallies_to_the_unsharded_sweep(tmp_path):
    port = 31000 + os.getpid() % 2000
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(os.environ, RANK=str(r), WORLD_SIZE="2", OMP_NUM_THREADS="2"),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    n = 0
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
        res = json.loads(o.strip().splitlines()[-1])
        assert res["tally"] < 1e-13 and res["phi"] < 1e-13 and res["psi"], res
        n += res["n"]
    assert n > 0
