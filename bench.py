#!/usr/bin/env python
"""bench.py -- the planar-MOC hot path on synthetic problems shaped like the paper's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--scale s] [--impl ours|reference]

A STEP is one pass of the whole hot path (DESIGN.md rows A2-A7): source update -> transport sweep -> link swap
-> flux finalise -> fission-rate reduction and k update, i.e. one power iteration, through the C ABI.
metric = segment-group-polar updates per second (U = 2*S*P*G per sweep, both directions counted).
Prints ONE JSON line.  Multi-GPU (N > 1): the angle pairs of the laydown are sharded over the ranks
(nd_tracks_shard; reflective links never leave a pair, so no boundary flux is exchanged) and the ranks share ONE collective
per sweep, an FP64 NCCL all-reduce of the tally (nd_tally_reducer_set): strong scaling of one problem.  --replicas runs N
independent copies instead (weak scaling, no collective).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "moc_segment_group_polar_updates_per_s"
UNIT = "updates/s"
L2_BYTES = 126 * 1024 * 1024


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config index 1..5 (default: the largest)")
    ap.add_argument("--scale", type=float, default=1.0, help="down-scaled twin of the config (1.0 = full size)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", type=int, default=0, help="ND_SWEEP_* (0 auto)")
    ap.add_argument("--exp-mode", type=int, default=0)
    for name in ("window-regions", "block-warps", "tile-segments", "delta-buffers", "blocks-per-sm", "tile-lag", "q-copies", "item-order"):
        ap.add_argument("--" + name, type=int, default=0, help="nd_options tuning field (0 = library default)")
    ap.add_argument("--cpu-seconds", type=float, default=None,
                    help="target CPU time of one oracle sample (default: 15 s for cpu_baseline; --impl reference: 150 s / steps, 2..30 s)")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: run N independent replicas (weak scaling) instead of sharding the angle pairs over the ranks")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(p.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", 1965.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


def build_inputs(args, tracer="device"):
    """Seeded synthetic problem + ray tracing (not timed).  tracer = "device": the library's GPU ray walk (row NEXT-1,
    segments bit-identical to its host tracer's and to the oracle's) with the segments left in device memory; "oracle": the oracle's own tracer (reference arm: nothing of
    the library runs there)."""
    from moc_inputs import make_config
    t0 = time.time()
    prob = make_config(args.config, scale=args.scale)
    m = prob.mesh
    t1 = time.time()
    if tracer == "oracle":
        import oracle
        tr = oracle.generate_tracks(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
        tr.n_segments = tr.n_segs
    else:
        import paper_2607_01591_b200 as nd
        local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        # the segments stay on the GPU: nd_problem_create builds its streams there (no segment crosses PCIe); the oracle legs
        # and the sharded run copy them back on first use (nd_tracks_materialise)
        tr = nd.nd_tracks_generate_resident(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing, device=f"cuda:{local_rank}")
        tracer = "device-resident"
    t2 = time.time()
    return prob, tr, {"mesh_s": round(t1 - t0, 2), "trace_s": round(t2 - t1, 2), "tracer": tracer}


def oracle_sample(prob, tr, cpu_seconds):
    """The oracle sweep (O-6), as it stands, on contiguous samples of the workload's tracks.  Sampled tracks keep their
    segments; their links are cut (vacuum), which does not change the work per update.

    Every orc_sweep call allocates, zeroes and reduces one private tally array per thread (threads x R x G doubles: 6.5 GB
    at config 5 with 16 threads) whatever the sample holds -- a cost of SAMPLING that a full sweep pays once per 1.5e11
    updates.  So two samples of different size are timed (about 1/3 and 2/3 of `cpu_seconds`) and the MARGINAL rate
    (u2 - u1) / (t2 - t1) is reported as `value`; the raw rates of both samples are reported beside it."""
    import oracle
    nth = oracle.num_threads()
    G, P, T = prob.n_groups, prob.n_polar, tr.n_tracks
    rate_guess = 6.0e7 * nth                         # FP64 updates/s, glibc expm1; refined by a pilot run
    rng = np.random.default_rng(1)
    Q = rng.uniform(0.05, 1.0, size=(prob.mesh.n_regions, G))

    def run(t0, t1):
        so = tr.seg_offset[t0:t1 + 1] - tr.seg_offset[t0]
        k0, k1 = int(tr.seg_offset[t0]), int(tr.seg_offset[t1])
        n = t1 - t0
        link = np.full((n, 2), -1, np.int32)
        psi = np.zeros((n, 2, P, G))
        vol = oracle.track_volumes(prob.mesh.n_regions, so, tr.seg_region[k0:k1], tr.seg_length[k0:k1], tr.track_weight[t0:t1])
        t_a = time.perf_counter()
        oracle.sweep(prob.mesh.material, prob.xs.sigma_t, prob.polar_sin, prob.polar_weight, so, tr.seg_region[k0:k1],
                     tr.seg_length[k0:k1], tr.track_weight[t0:t1], link, vol, Q, psi)
        dt = time.perf_counter() - t_a
        return 2 * (k1 - k0) * P * G, dt

    def pick(n_updates):
        # tracks from the middle of the canonical order (typical lengths), enough for n_updates
        per_track = 2.0 * tr.n_segments / T * P * G
        n = int(min(T, max(1, n_updates / per_track)))
        t0 = max(0, T // 2 - n // 2)
        return t0, t0 + n

    u0, dt0 = run(*pick(rate_guess * 0.5))           # pilot ~0.5 s (includes the fixed cost)
    rate = u0 / dt0
    u1, dt1 = run(*pick(rate * cpu_seconds / 3.0))
    u2, dt2 = run(*pick(rate * cpu_seconds * 2.0 / 3.0))
    U = 2.0 * tr.n_segments * P * G
    if u2 > u1 and dt2 > dt1:
        value, fixed = (u2 - u1) / (dt2 - dt1), max(0.0, dt1 - u1 * (dt2 - dt1) / (u2 - u1))
    else:                                            # the whole workload fits the smaller sample (tiny configs)
        value, fixed = u2 / dt2, 0.0
    return {"value": value, "unit": UNIT, "cores": nth, "kind": "oracle",
            "raw_rates": [u1 / dt1, u2 / dt2], "fixed_cost_s_per_call": fixed,
            "sample": f"oracle O-6 sweep (FP64, OpenMP), marginal rate between two contiguous track samples holding "
                      f"{u1 / U:.4%} and {u2 / U:.4%} of the workload's updates ({u1:.3e} updates in {dt1:.1f} s, {u2:.3e} in "
                      f"{dt2:.1f} s; {fixed:.2f} s per call is the per-thread tally set-up of orc_sweep, paid once per full sweep)"}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on this box's host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    prob, tr, setup = build_inputs(args, tracer="oracle")
    per_step = args.cpu_seconds if args.cpu_seconds else max(2.0, min(30.0, 150.0 / max(1, args.steps + args.warmup)))
    vals, times = [], []
    cb = None
    for i in range(args.warmup + args.steps):
        cb = oracle_sample(prob, tr, per_step)
        if i >= args.warmup:
            vals.append(cb["value"])
    value = float(np.mean(vals))
    # ms_per_step: time the oracle would need for one full sweep of the workload at the sampled rate
    U = 2.0 * tr.n_segments * prob.n_polar * prob.n_groups
    cb["value"] = value
    line = {"metric": METRIC, "value": value, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": U / value * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, prob, tr), "cpu_baseline": cb,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "note": "oracle O-6 sweep on a bounded track sample per step; ms_per_step extrapolates "
                                       "the sampled rate to one full sweep"}
    print(json.dumps(line), flush=True)


def workload_config(args, prob, tr):
    return {"workload": f"BASELINE.json configs[{args.config - 1}] ({prob.name})" + (f" down-scaled x{args.scale}" if args.scale != 1.0 else ""),
            "n_regions": int(prob.mesh.n_regions), "n_groups": int(prob.n_groups), "n_polar": int(prob.n_polar),
            "n_azim": int(prob.n_azim), "spacing_cm": float(prob.spacing), "n_tracks": int(tr.n_tracks),
            "n_segments": int(tr.n_segments), "updates_per_sweep": int(2 * tr.n_segments * prob.n_polar * prob.n_groups),
            "bc_left_right_bottom_top": list(prob.bc), "step": "one power iteration (source, sweep, link swap, finalise, k)",
            "parallelism": ("single GPU" if args.gpus <= 1 else f"replicas x{args.gpus}" if args.replicas else
                            f"angle pairs sharded over {args.gpus} ranks, one FP64 all-reduce of the tally per sweep")}


def aggregate(ms_local: float, units_local: float):
    """MAX time over ranks and SUM of units over ranks (torch.distributed if initialised; gloo on CPU, nccl on GPU)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return ms_local, units_local
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    u = torch.tensor([units_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    import torch
    import torch.distributed as dist
    import paper_2607_01591_b200 as nd

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the MOC hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    prob, tr_full, setup = build_inputs(args)
    sharded = world > 1 and not args.replicas
    tr = tr_full.shard(world, rank) if sharded else tr_full     # NEXT-2: this rank's angle pairs (areas of the whole laydown)
    t0 = time.time()
    gp = nd.nd_problem_create(prob.xs, prob.polar_sin, prob.polar_weight, prob.mesh.material, tr, device=str(dev),
                              sweep_kernel=args.kernel, exp_mode=args.exp_mode,
                              window_regions=args.window_regions, block_warps=args.block_warps,
                              tile_segments=args.tile_segments, delta_buffers=args.delta_buffers,
                              blocks_per_sm=args.blocks_per_sm, tile_lag=args.tile_lag, item_order=args.item_order,
                              q_copies=args.q_copies)
    setup["create_s"] = round(time.time() - t0, 2)
    if sharded:
        gp.nd_tally_reducer_set(lambda tally: dist.all_reduce(tally))   # the one collective of the path: sum of the shards' tallies
    info = gp.nd_problem_info_get()
    R, G = prob.mesh.n_regions, prob.n_groups
    U = info["updates_per_sweep"]
    resident = info["n_segments_padded"] * 8 + 2 * 4 * tr.n_tracks * 2 * prob.n_polar * G + 20 * R * G
    need_flush = resident < 2 * L2_BYTES
    flush_buf = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev) if need_flush else None
    stream = torch.cuda.current_stream(dev)

    def step():
        gp.nd_power_iteration(1)

    def sync_all():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize(dev)

    for _ in range(max(3, args.warmup)):
        step()
    sync_all()

    # ---- device-resident timing: K steps, CUDA events on the launching stream, L2 flushed between steps if small ----
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    gp.nd_profile_enable(True)
    with ClockSampler(local_rank) as clocks:
        sync_all()
        for a, b in evs:
            if flush_buf is not None:
                flush_buf.fill_(1)
            a.record(stream)
            step()
            b.record(stream)
        sync_all()
    prof = gp.nd_profile_read()
    gp.nd_profile_enable(False)
    ms_local = sum(a.elapsed_time(b) for a, b in evs)
    ms_total, units = aggregate(ms_local, float(U) * args.steps)
    ms_per_step = ms_total / args.steps
    value = units / (ms_total * 1e-3)

    # ---- end to end through the C ABI with HOST buffers: H2D phi -> nd_flux_set -> one power iteration -> D2H phi ----
    e2e = None
    if not args.no_e2e:
        h_bufs = [torch.ones((R, G), dtype=torch.float64).pin_memory(), torch.empty((R, G), dtype=torch.float64).pin_memory()]
        d_in = torch.empty((R, G), dtype=torch.float64, device=dev)
        d_out = torch.empty((R, G), dtype=torch.float64, device=dev)
        k_host = 1.0

        def e2e_step(k):
            h_in, h_out = h_bufs
            d_in.copy_(h_in, non_blocking=True)
            gp.nd_flux_set(d_in, k)
            out = gp.nd_power_iteration(1, d_phi_out=d_out)
            h_out.copy_(d_out, non_blocking=True)
            torch.cuda.synchronize(dev)
            h_bufs.reverse()                       # next step starts from this step's result (the state lives on the host)
            return out["k_eff"]

        for _ in range(2):
            k_host = e2e_step(k_host)
        sync_all()
        t_a = time.perf_counter()
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ea.record(stream)
        for _ in range(args.steps):
            if flush_buf is not None:
                flush_buf.fill_(1)
            k_host = e2e_step(k_host)
        eb.record(stream)
        sync_all()
        e_ms, e_units = aggregate(ea.elapsed_time(eb), float(U) * args.steps)
        e2e = {"value": e_units / (e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(R * G * 8 + 8),
               "d2h_bytes_per_step": int(R * G * 8 + 16), "ms_per_step": e_ms / args.steps,
               "what": "pinned host phi -> device, nd_flux_set, nd_power_iteration(1), phi + k -> pinned host"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_peak, peak_src, sm_max = peaks()
    sweep_ms = prof["sweep_ms"] / max(1, prof["sweep_launches"])
    achieved = info["algorithmic_bytes"] / (sweep_ms * 1e-3) / 1e9
    # DRAM bytes of one sweep launch as ncu saw them: profiles/r02_traffic_cfg<config>_<build id>.csv, the log of the ncu
    # command in profiles/r02_traffic.md.  Only a capture of THIS build (nd_build_id) is quoted; otherwise null.
    build_id = nd.nd_build_id()
    traffic, traffic_src = None, f"no ncu capture of build {build_id} under profiles/ (see profiles/r02_traffic.md)"
    tpath = os.path.join(ROOT, "profiles", f"r02_traffic_cfg{args.config}_{build_id}.csv")
    if os.path.exists(tpath) and args.scale == 1.0 and info["sweep_kernel"] == 3:
        import csv
        tot = 0
        for row in csv.reader(open(tpath)):
            if len(row) > 14 and "k_sweep_swath" in row[4] and row[12] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                tot += int(float(row[14]))
        if tot > 0:
            traffic, traffic_src = tot, os.path.relpath(tpath, ROOT)
    mb = None
    try:
        mb = nd.nd_microbench(device=str(dev))
    except nd.NdError as e:                          # diagnostics only: the bench line does not depend on it
        mb = {"error": str(e)}
    # The sweep is bound by the exp pipe, not by HBM: one update = one MUFU.EX2, and the SM issues
    # 16 of them per clock -> peak = 148 SMs x 16 x max SM clock.  The HBM view (algorithmic bytes / kernel time against
    # the measured copy bandwidth, and the DRAM traffic ncu saw) is reported beside it.
    mufu_peak = 148 * 16 * sm_max * 1e6
    upd_rate = U / (sweep_ms * 1e-3)
    roofline = {"bound": "alu", "achieved": upd_rate / 1e9, "peak": mufu_peak / 1e9, "unit": "Gupdate/s (1 MUFU.EX2 each)",
                "frac": upd_rate / mufu_peak, "traffic": traffic, "kernel": "k_sweep_swath" if info["sweep_kernel"] == 3 else "sweep",
                "kernel_ms": sweep_ms, "kernel_share_of_step": sweep_ms / (ms_local / args.steps),
                "peak_source": f"derived: 148 SMs x 16 MUFU.EX2/clk/SM x {sm_max:.0f} MHz max SM clock (DESIGN.md section 5); "
                               "nd_microbench measured in this run: see roofline.microbench",
                "microbench": mb, "traffic_source": traffic_src, "build_id": build_id,
                "hbm": {"bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s", "frac": achieved / hbm_peak,
                        "algorithmic_bytes_per_launch": int(info["algorithmic_bytes"]), "peak_source": peak_src,
                        "dram_traffic_GBps": (traffic / (sweep_ms * 1e-3) / 1e9) if traffic else None}}
    cb = None
    if not args.no_cpu_baseline:
        cb = oracle_sample(prob, tr_full, args.cpu_seconds or 15.0)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms_per_step, "ms_per_sweep": sweep_ms, "higher_is_better": True,
            "scaling": "strong" if sharded else "weak",
            "vs_baseline": None, "dtype": "f32 (segment arithmetic) + f64 (tallies, flux, source, k)", "data": "synthetic",
            "config": dict(workload_config(args, prob, tr_full), l2="L2 flushed between steps" if need_flush else "inputs larger than L2",
                           sweep_kernel=info["sweep_kernel"], setup_s=setup,
                           launch={k: info[k] for k in ("block_threads", "smem_bytes", "grid_blocks", "tracks_per_block", "n_batches",
                                                        "mean_regions_per_tile", "mean_segments_per_tile", "lockstep_efficiency")}),
            "e2e": e2e, "gpu_launches": int(prof["kernels_launched"]), "roofline": roofline, "cpu_baseline": cb,
            "clocks": clocks.summary(), "k_eff": k_host if e2e else None}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
