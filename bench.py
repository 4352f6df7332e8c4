#!/usr/bin/env python
"""bench.py -- throughput of the per-frame particle pipeline of arXiv 2311.15088 on B200 (sm_100a).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is ONE FRAME of the whole hot path on BASELINE.json's headline
workload (config 4: 1 048 576 fluid particles, 4 096 boids, 256^3 voxel corners):
neighbour grid -> SPH density / forces / integration -> boid update with two-way coupling -> grid on the new
positions -> voxel signed distance -> marching cubes.  All of it runs in libsphboid's CUDA kernels through the
C ABI; torch supplies device memory, streams and events only.  One JSON line is printed by rank 0.

  value      particle-updates/s over the whole frame = N * K / t, inputs resident in HBM
  parts      the two halves BASELINE.json's metric names: SPH+boid particle-updates/s (S1-S13) and MC voxels/s
             (S14-S17), each with its algorithmic GB/s and fraction of the measured HBM peak
  e2e        the same frame through sph_simulate_host with pinned HOST buffers, copies inside the timed region
  roofline   the dominant kernel on the roofline that binds it: binary32 arithmetic (algorithmic flops of the true
             pairs / its average CUDA-event duration against the FMA peak), with its HBM coordinates under "hbm"
  kernels    every kernel: launches, average us, share of the step, algorithmic GB/s (event pairs around every launch,
             in a second run of the same K frames so that the pairs do not sit inside the region `value` is timed on)
  cpu_baseline  the CPU oracle (oracle/, test infrastructure) timed on this box's host cores on the same workload

--impl reference times the oracle alone (this tier has no reference implementation to install).
--gpus N > 1 (under torchrun): N independent replicas, no data-path collective ("replicas only").
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle-updates/s (whole frame: grid + SPH + boids + voxel SDF + marching cubes)"
L2_BYTES = 126e6


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md, clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except Exception:
                self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1]))
                smax.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(smax), reasons=sorted(reasons), samples=len(sm))
        return out


def workload_config(cfg, world):
    """The `config` object of the JSON line: the workload only, identical for the GPU arm and the --impl reference arm
    (run-specific facts -- frame loop, grid cells, triangle count -- go under `run`)."""
    n, nb, G = cfg["n"], cfg["n_boid"], cfg["G"]
    state_bytes = 32 * n * 2 + 16 * n + 4 * G ** 3
    return {"workload": cfg["name"], "particles": n, "boids": nb, "mc_points_per_axis": G,
            "parallelism": "replicas x%d" % world,
            "l2": ("no explicit flush: the frame's working set (%.0f MB of state, sorted copies and phi) exceeds the %.0f MB "
                   "L2 and the state changes every step" if state_bytes > L2_BYTES else
                   "no explicit flush, and this workload's working set (%.0f MB) FITS the %.0f MB L2: an L2-resident "
                   "figure (the headline workload, config4, exceeds it)") % (state_bytes / 1e6, L2_BYTES / 1e6)}


def oracle_frame(R, W, cfg, mp, state):
    """One frame on the CPU oracle (same order as Frame.frame).  state = [pos, vel, bpos, bvel]; returns n_tris."""
    pos, vel, bpos, bvel = state
    ref = R.step(cfg["sph"], pos, vel, bpos, bvel, cfg["boid"])
    refb = R.boid_step(cfg["sph"], cfg["boid"], pos, vel, ref["density"], bpos, bvel)
    state[:] = [ref["pos"], ref["vel"], refb["bpos"], refb["bvel"]]
    phi = R.voxel_sdf(cfg["sph"], mp, state[0])
    _, nt, _ = R.mc_polygonise(mp, phi)
    return nt


def time_oracle(cfg, mp, min_seconds, max_frames):
    from oracle import refbind as R
    from paper_2311_15088_b200 import workloads as W
    state = [cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"]]
    frames, t0 = 0, time.perf_counter()
    per = []
    while frames < max_frames:
        t1 = time.perf_counter()
        oracle_frame(R, W, cfg, mp, state)
        per.append(time.perf_counter() - t1)
        frames += 1
        if time.perf_counter() - t0 >= min_seconds:
            break
    return frames, per, R.num_threads()


def time_oracle_threads(cfg_idx, threads):
    """Seconds per oracle frame of config `cfg_idx` with OMP_NUM_THREADS = threads (a child process: the OpenMP runtime
    reads the variable once).  Returns (seconds, threads used) or None."""
    code = ("import sys,time,json; sys.path.insert(0,%r)\n"
            "import bench\n"
            "from oracle import refbind as R\n"
            "from paper_2311_15088_b200 import workloads as W\n"
            "cfg=W.config(%d); mp=W.mc_params(cfg)\n"
            "st=[cfg['pos'],cfg['vel'],cfg['bpos'],cfg['bvel']]\n"
            "R.mc_table()\n"
            "t=time.perf_counter(); bench.oracle_frame(R,W,cfg,mp,st); dt=time.perf_counter()-t\n"
            "print(json.dumps([dt,R.num_threads()]))\n") % (ROOT, cfg_idx)
    env = dict(os.environ, OMP_NUM_THREADS=str(threads))
    try:
        out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=300)
        dt, used = json.loads(out.stdout.strip().splitlines()[-1])
        return float(dt), int(used)
    except Exception:
        return None


def run_reference(args, cfg_idx):
    """--impl reference: the CPU oracle as it stands, on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    # torchrun exports OMP_NUM_THREADS=1 to every rank unless the caller set it; this arm runs on rank 0 alone and is
    # meant to use the box's host cores, so that default is undone before the OpenMP runtime of the oracle starts
    if os.environ.get("TORCHELASTIC_RUN_ID") and os.environ.get("OMP_NUM_THREADS") == "1":
        os.environ["OMP_NUM_THREADS"] = str(len(os.sched_getaffinity(0)))
    from paper_2311_15088_b200 import workloads as W
    cfg = W.config(cfg_idx)
    mp = W.mc_params(cfg)
    n = cfg["n"]
    # each "step" is one full frame of the workload on the oracle; cap the run at ~3 minutes
    budget = 170.0
    state = [cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"]]
    from oracle import refbind as R
    done_w = 0
    t_start = time.perf_counter()
    for _ in range(args.warmup):
        if time.perf_counter() - t_start > budget / 4:
            break
        oracle_frame(R, W, cfg, mp, state)
        done_w += 1
    per = []
    for _ in range(args.steps):
        t1 = time.perf_counter()
        oracle_frame(R, W, cfg, mp, state)
        per.append(time.perf_counter() - t1)
        if time.perf_counter() - t_start > budget:
            break
    k = len(per)
    t = sum(per)
    value = n * k / t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "particle-updates/s", "n_gpus": args.gpus,
        "steps": k, "warmup": done_w, "ms_per_step": 1e3 * t / k, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(cfg, args.gpus),
        "run": {"note": "CPU oracle (oracle/, plain C++ with OpenMP over the outer index), one frame per step"},
        "cpu_baseline": {"value": value, "unit": "particle-updates/s", "cores": R.num_threads(), "kind": "oracle",
                         "sample": "%d whole frames of %s (steps requested %d, time-capped)" % (k, cfg["name"],
                                                                                              args.steps)},
        "e2e": {"value": value, "unit": "particle-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_slab(args):
    """--decomposition slab (N2): the fluid, the boids and the cubes of the voxel grid cut into slabs over the ranks,
    strong scaling; a step is the whole frame (surface pass of the frame-start state for the rank's cubes, SPH step,
    boid step).  Exchange: neighbour send / receive over NCCL; one all-reduce of the triangle counts at the end."""
    import torch
    from paper_2311_15088_b200 import binding as B
    from paper_2311_15088_b200 import dist as D
    from paper_2311_15088_b200 import slab as S
    from paper_2311_15088_b200 import workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    B.lib()
    ranks = D.Ranks()
    dev = ranks.local_rank
    torch.cuda.set_device(dev)
    cfg = W.config(args.config)
    n, K = cfg["n"], args.steps
    mc = W.mc_params(cfg)
    lay = S.SlabLayout(cfg["sph"], ranks.world, boid=cfg["boid"], mc=mc, pos=cfg["pos"])  # faces cut by particle count
    p, v = S.split_initial(lay, cfg["pos"], cfg["vel"])[ranks.rank]
    bp, bv = S.split_initial(lay, cfg["bpos"], cfg["bvel"])[ranks.rank]
    be = S.GpuBackend(cfg["sph"], min(n, 2 * (n // ranks.world) + (1 << 16)), device=dev, boid_capacity=cfg["n_boid"],
                      mc_points=mc["n_point_per_axis"])
    ex = (S.DistExchange(ranks.dist, ranks.rank, ranks.world, torch.device("cuda", dev), capacity=max(1 << 16, n // 4)) if ranks.world > 1
          else S.LoopbackExchange(1))
    sim = S.SlabSim(lay, ranks.rank, be, ex, be.to_device(p), be.to_device(v), be.to_device(bp), be.to_device(bv),
                    cfg["boid"])
    tris = torch.empty(max(1 << 16, (4 << 20) // ranks.world), 3, 3, device=torch.device("cuda", dev))
    for _ in range(max(args.warmup, 3)):
        sim.step(tris)
    sampler = ClockSampler(dev)
    sampler.start()
    time.sleep(0.15)
    ranks.barrier()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    launches0 = B.sph_launch_count(be.ctx)
    ev[0].record()
    n_tris = 0
    for k in range(K):
        n_tris = sim.step(tris)
        if args.recut_every and (k + 1) % args.recut_every == 0 and ranks.world > 1:
            sim.recut()
    ev[1].record()
    torch.cuda.synchronize()
    ranks.barrier()
    if n_tris > tris.shape[0]:
        raise SystemExit("triangle buffer too small: %d > %d" % (n_tris, tris.shape[0]))
    t = ev[0].elapsed_time(ev[1]) * 1e-3
    launches = B.sph_launch_count(be.ctx) - launches0
    clocks = sampler.stop()
    t_max, _ = ranks.combine(t, 0.0)
    owned = ranks.reduce_max([float(sim.n_owned), float(sim.stats["ghosts"])])
    _, tris_total = ranks.combine(0.0, float(n_tris))
    if ranks.rank == 0:
        print(json.dumps({
            "metric": "particle-updates/s (whole frame, slab-decomposed over the ranks: surface pass of the rank's cubes, SPH step, boid step)",
            "value": n * K / t_max, "unit": "particle-updates/s", "n_gpus": ranks.world, "steps": K,
            "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * t_max / K, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg["name"], "particles": n, "parallelism": "slab x%d along axis %d" % (ranks.world, lay.axis),
                       "max_owned_per_rank": int(owned[0]), "max_ghosts_per_rank": int(owned[1]),
                       "boids": cfg["n_boid"], "mc_points_per_axis": mc["n_point_per_axis"],
                       "triangles_last_frame": int(tris_total),
                       "exchange": "4 neighbour send/recv pairs per step (fluid halo, boid halo, two migrations), NCCL"},
            "gpu_launches": launches, "clocks": clocks, "e2e": None, "roofline": None, "cpu_baseline": None}))
    be.close()
    ranks.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config 1-5 (4 = the headline workload)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--force-variant", type=int, default=0, help="A/B: 0 = cost model (default), 1 = stored neighbour list, 2 = brick density pass + neighbour masks")
    ap.add_argument("--sdf-variant", type=int, default=0, help="A/B: 0 = cost model (default), 1 = per-corner walk, 2 = corner tiles")
    ap.add_argument("--recut-every", type=int, default=0, help="slab decomposition: re-cut the faces by particle count every k frames (0 = never)")
    ap.add_argument("--decomposition", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default) or the fluid cut into slabs with halo exchange (N2, SPH step only)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args, args.config)
    if args.decomposition == "slab":
        return run_slab(args)
    if args.warmup < 3:
        args.warmup = 3

    import torch
    from paper_2311_15088_b200 import binding as B
    from paper_2311_15088_b200 import dist as D
    from paper_2311_15088_b200 import roofline as RF
    from paper_2311_15088_b200 import workloads as W
    from paper_2311_15088_b200.pipeline import Frame

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    B.lib()  # fail loudly if libsphboid.so is not built
    ranks = D.Ranks()
    dev = ranks.local_rank
    torch.cuda.set_device(dev)
    cfg = W.config(args.config, seed=ranks.rank)  # replicas differ only in the jitter / boid seed
    n, nb, K = cfg["n"], cfg["n_boid"], args.steps
    peak, peak_kind = measured_peak()

    fr = Frame(cfg, device=dev)
    if args.force_variant:
        B.sph_set_force_variant(fr.ctx, args.force_variant)
    if args.sdf_variant:
        B.mc_set_sdf_variant(fr.ctx, args.sdf_variant)
    G = fr.G
    _, C = B.sph_grid_dims(fr.ctx)
    for _ in range(args.warmup):
        fr.frame()
    torch.cuda.synchronize()

    # ---- timed region: K frames, state resident in HBM -------------------------------------------------
    sampler = ClockSampler(dev)
    sampler.start()
    time.sleep(0.15)
    ranks.barrier()
    torch.cuda.synchronize()
    # (1) the frame loop with the surface pass of frame t forked (mc_extract_async) beside the SPH step of frame t+1; the
    #     library orders the next grid build after it
    launches0 = B.sph_launch_count(fr.ctx)
    evt = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    evt[0].record()
    for k in range(K):
        fr.sim()
        fr.surface_async()
    fr.wait()
    evt[1].record()
    torch.cuda.synchronize()
    ranks.barrier()
    launches = B.sph_launch_count(fr.ctx) - launches0
    t_total = evt[0].elapsed_time(evt[1]) * 1e-3
    # (2) the same K frames with the synchronous calls, one half after the other: the two halves the metric names
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * K + 1)]
    ev[0].record()
    for k in range(K):
        fr.sim()
        ev[2 * k + 1].record()
        fr.surface()
        ev[2 * k + 2].record()
    torch.cuda.synchronize()
    t_serial = ev[0].elapsed_time(ev[2 * K]) * 1e-3
    # (3) CUDA graphs: the synchronous frame captured once and replayed K times (one launch per frame), and four
    #     pipelined frames per graph (inside it the surface pass of a frame runs beside the next frame's SPH step)
    def time_graph(frames, pipelined):
        fr.capture(frames=frames, pipelined=pipelined)
        reps = max(1, (K + frames - 1) // frames)
        evg = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ranks.barrier()
        torch.cuda.synchronize()
        evg[0].record()
        for _ in range(reps):
            fr.replay()
        evg[1].record()
        torch.cuda.synchronize()
        return evg[0].elapsed_time(evg[1]) * 1e-3 * K / (reps * frames)  # scaled to K frames

    t_graph = time_graph(1, False)
    t_graph4 = time_graph(4, True)
    t_sim = sum(ev[2 * k].elapsed_time(ev[2 * k + 1]) for k in range(K)) * 1e-3
    t_mc = sum(ev[2 * k + 1].elapsed_time(ev[2 * k + 2]) for k in range(K)) * 1e-3
    # ---- per-kernel durations: the same K frames again with a CUDA event pair around every launch (the pairs cost a
    # few microseconds per launch, so they stay out of the region `value` is measured on) ----------------------------
    B.sph_profile_enable(fr.ctx, True)
    evp = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    evp[0].record()
    for k in range(K):
        fr.frame()
    evp[1].record()
    torch.cuda.synchronize()
    t_profiled = evp[0].elapsed_time(evp[1]) * 1e-3
    profile = B.sph_profile_read(fr.ctx)
    B.sph_profile_enable(fr.ctx, False)
    clocks = sampler.stop()
    n_tris = B.mc_extract(fr.ctx, fr.mc, fr.tris, sync=True)  # same state as the last timed frame
    # N3 (not part of `value`): the same surface as an indexed mesh with normals, timed on its own
    iverts = torch.empty(3 * max(n_tris, 1), 3, device=fr.device)
    inorm = torch.empty(3 * max(n_tris, 1), 3, device=fr.device)
    iidx = torch.empty(max(n_tris, 1), 3, dtype=torch.int32, device=fr.device)
    n_iv, _ = B.mc_extract_indexed(fr.ctx, fr.mc, iverts, inorm, iidx)
    evi = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    evi[0].record()
    for _ in range(3):
        B.mc_extract_indexed(fr.ctx, fr.mc, iverts, inorm, iidx, sync=False)
    evi[1].record()
    torch.cuda.synchronize()
    indexed = {"ms_per_pass": evi[0].elapsed_time(evi[1]) / 3, "vertices": n_iv, "triangles": n_tris,
               "what": "mc_extract_indexed: S14 + welded vertices, central-difference normals, index buffer"}
    # connectivity of that mesh (Table 2's last column under reading D:A-CONNECT): share of the largest component
    ilabel = torch.empty(max(n_iv, 1), dtype=torch.int32, device=fr.device)
    n_comp, largest = B.mc_mesh_components(fr.ctx, iidx, n_tris, n_iv, ilabel)
    evc = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    evc[0].record()
    for _ in range(3):
        B.mc_mesh_components(fr.ctx, iidx, n_tris, n_iv, ilabel, sync=False)
    evc[1].record()
    torch.cuda.synchronize()
    indexed["connectivity"] = {"components": n_comp, "largest_component_triangles": largest,
                               "percent_connected": 100.0 * largest / max(n_tris, 1),
                               "ms_per_pass": evc[0].elapsed_time(evc[1]) / 3,
                               "what": "mc_mesh_components: union-find over the welded vertices"}
    del iverts, inorm, iidx, ilabel
    # N4 baseline (not part of `value`): neighbour counts through the sorted grid (grid build + count pass) against the
    # paper's first, unsorted fixed-capacity hash grid, same positions, same counts
    cnt_a = torch.zeros(n, dtype=torch.int32, device=fr.device)
    cnt_b = torch.zeros(n, dtype=torch.int32, device=fr.device)
    B.sph_neighbor_count(fr.ctx, fr.pos, cnt_a)
    # capacity of the unsorted grid = the largest cell population of the sorted one, so that nothing is dropped and the
    # two searches do the same work (a comparison against a grid that drops particles would be invalid)
    cstart = torch.zeros(C + 1, dtype=torch.int32, device=fr.device)
    B.sph_build_grid(fr.ctx, fr.pos, None, cell_start=cstart)
    hg_cap = int((cstart[1:] - cstart[:-1]).max().item())
    del cstart
    dropped = B.sph_hashgrid_neighbor_count(fr.ctx, fr.pos, hg_cap, cnt_b)
    evn = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    evn[0].record()
    for _ in range(5):
        B.sph_neighbor_count(fr.ctx, fr.pos, cnt_a)
    evn[1].record()
    for _ in range(5):
        B.sph_hashgrid_neighbor_count(fr.ctx, fr.pos, hg_cap, cnt_b, sync=False)
    evn[2].record()
    torch.cuda.synchronize()
    nsearch = {"sorted_grid_us": 1e3 * evn[0].elapsed_time(evn[1]) / 5, "unsorted_hash_grid_us": 1e3 * evn[1].elapsed_time(evn[2]) / 5,
               "max_per_cell": hg_cap, "dropped": dropped, "counts_equal": bool((cnt_a == cnt_b).all().item()),
               "what": "neighbour count of every particle: grid build + count pass (sph_neighbor_count) vs the paper's "
                       "unsorted fixed-capacity hash grid (sph_hashgrid_neighbor_count)"}
    nsearch["valid"] = bool(nsearch["dropped"] == 0 and nsearch["counts_equal"])
    if not nsearch["valid"]:
        nsearch["sorted_grid_us"] = nsearch["unsorted_hash_grid_us"] = None  # not a like-for-like comparison
    del cnt_a, cnt_b
    # true neighbour pairs of that state (for the arithmetic roofline): one more SPH step with the count output
    ncount = torch.zeros(n, dtype=torch.int32, device=fr.device)
    B.sph_step(fr.ctx, fr.pos, fr.vel, fr.bpos, fr.bvel, cfg["boid"], ncount=ncount)
    sph_pairs = float(ncount.sum().item())
    if n_tris > fr.tri_capacity:
        raise SystemExit("triangle buffer too small: %d > %d" % (n_tris, fr.tri_capacity))
    cb = None
    bpar = cfg["boid"]
    cell_b = max(bpar["visible_range"], bpar["protect_range"], bpar["push_radius"])
    import math
    cb = 1
    for a in range(3):
        cb *= max(1, math.ceil((bpar["space_max"][a] - bpar["space_min"][a]) / cell_b))

    # all three loops ran the same K frames; `value` is the fastest way to run them (the overlap pays when the working
    # set fits L2, config 4, and costs when the two passes evict each other, config 5; the graph pays when the frame is
    # launch-bound, configs 1-3); all three times are reported
    t_pipe_max, units = ranks.combine(t_total, n * K)
    t_serial_max, _ = ranks.combine(t_serial, 0.0)
    t_graph_max, _ = ranks.combine(t_graph, 0.0)
    t_graph4_max, _ = ranks.combine(t_graph4, 0.0)
    t_max = min(t_pipe_max, t_serial_max, t_graph_max, t_graph4_max)
    mode = {t_pipe_max: "pipelined", t_serial_max: "synchronous", t_graph_max: "graph",
            t_graph4_max: "graph of 4 pipelined frames"}[t_max]
    t_sim_max, t_mc_max = ranks.reduce_max([t_sim, t_mc])
    value = units / t_max
    world = ranks.world

    rows, dominant = RF.summarise(profile, n, C, nb, cb, G, n_tris, peak)
    # SPH half = S1-S13 (one grid build per frame); surface half = S14-S17 (mc_extract alone)
    sim_bytes = RF.pass_bytes(RF.SIM_KERNELS, n, C, nb, cb, G, n_tris)
    mc_bytes = RF.pass_bytes(RF.MC_KERNELS, n, C, nb, cb, G, n_tris)
    sim_gbs = sim_bytes * K / t_sim / 1e9
    mc_gbs = mc_bytes * K / t_mc / 1e9
    dom = next(r for r in rows if r["kernel"] == dominant)
    sm_max = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("sm_max_mhz", 1965.0)) \
        if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else 1965.0
    pairs = RF.sdf_pairs(n, fr.mc["radius"], fr.mc["spacing"]) if RF.KERNEL_KIND.get(dominant) == "sdf" else sph_pairs
    alu = RF.alu_point(dominant, dom["avg_us"], pairs, sm_max)
    # dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture; quoted only when
    # that capture was taken on the CUDA sources this run is built from (the file is stamped with their hash), else null
    traffic, traffic_capture, traffic_stale = RF.read_traffic(os.path.join(ROOT, "profiles", "traffic.csv"), dominant)
    hbm = {"achieved": dom["gbs"], "peak": peak, "unit": "GB/s", "frac": dom["frac"], "peak_kind": "of " + peak_kind,
           "bytes_per_launch": dom["bytes"]}
    if alu is not None:
        # the dominant kernel is bound by binary32 arithmetic (DRAM throughput ~1 % in profiles/): ALU roofline first,
        # its HBM coordinates (BASELINE.json's metric) beside it
        roof = {"bound": "alu", "kernel": dominant, "achieved": alu["achieved"], "peak": alu["peak"], "unit": "TFLOP/s",
                "frac": alu["frac"], "traffic": traffic, "flop_per_launch": alu["flop_per_launch"],
                "pairs_per_launch": alu["pairs"], "flop_per_pair": alu["flop_per_pair"],
                "peak_kind": "148 SMs x 128 lanes x 2 flop x %.0f MHz (DESIGN.md section 6)" % sm_max,
                "avg_us": dom["avg_us"], "share_of_step": dom["share"], "hbm": hbm}
    else:
        roof = dict(hbm, bound="hbm", kernel=dominant, traffic=traffic, avg_us=dom["avg_us"], share_of_step=dom["share"])
    # BASELINE.json's metric is the fraction of the HBM roofline: flat keys beside the roofline that binds the kernel
    # (algorithmic bytes of SURVEY.md 8(d) / measured time / measured HBM peak; halves from the synchronous loop)
    roof["hbm_frac"] = dom["frac"]
    roof["hbm_frac_sph_half"] = sim_gbs / peak
    roof["hbm_frac_mc_half"] = mc_gbs / peak
    roof["hbm_frac_frame"] = (sim_bytes + mc_bytes) * K / t_max / 1e9 / peak
    roof["traffic_source"] = {"capture": traffic_capture, "stale": traffic_stale, "csrc_sha16": RF.csrc_sha16()}

    # ---- end to end through the C ABI with HOST buffers -------------------------------------------------
    e2e = None
    if not args.no_e2e:
        hp = [torch.from_numpy(cfg[k].copy()).pin_memory() for k in ("pos", "vel", "bpos", "bvel")]
        htris = torch.empty(fr.tri_capacity, 3, 3).pin_memory()
        Ke = min(K, 10)
        for _ in range(2):
            B.sph_simulate_host(fr.ctx, hp[0], hp[1], hp[2], hp[3], cfg["boid"], 1, fr.mc, htris)
        torch.cuda.synchronize()
        ranks.barrier()
        t0 = time.perf_counter()
        nts = []
        for _ in range(Ke):
            nts.append(B.sph_simulate_host(fr.ctx, hp[0], hp[1], hp[2], hp[3], cfg["boid"], 1, fr.mc, htris))
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        ranks.barrier()
        t_e2e_max, units_e = ranks.combine(t_e2e, n * Ke)
        h2d = 32 * n + 32 * nb
        d2h = 32 * n + 32 * nb + 36 * (sum(nts) // len(nts)) + 4
        e2e = {"value": units_e / t_e2e_max, "unit": "particle-updates/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": Ke, "ms_per_step": 1e3 * t_e2e_max / Ke,
               "api": "sph_simulate_host (pinned host pos/vel/bpos/bvel in, state + triangles out, every step)",
               "timer": "host wall clock around the synchronous calls"}
    fr.close()

    # ---- the oracle on this box's host cores, rank 0 at N = 1 only --------------------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        frames, per, cores = time_oracle(cfg, W.mc_params(cfg), 10.0, 8)
        cpu = {"value": n * frames / sum(per), "unit": "particle-updates/s", "cores": cores, "kind": "oracle",
               "sample": "%d whole frame(s) of %s (%d particles, %d boids, %d^3 corners), %.1f s" %
                         (frames, cfg["name"], n, nb, G, sum(per))}
        # single-thread beside all-core.  One frame of config 2 (65 536 particles, 64^3 corners) in
        # a child process with OMP_NUM_THREADS=1, and the same frame with all cores for the ratio; the single-thread
        # figure for THIS workload is that ratio applied to `value` (an extrapolation, labelled as such)
        one, many = time_oracle_threads(2, 1), time_oracle_threads(2, cores)
        if one and many:
            n2 = W.config(2)["n"]
            cpu["single_thread"] = {
                "value": n2 / one[0], "unit": "particle-updates/s", "cores": one[1],
                "sample": "one whole frame of config2 (%d particles), OMP_NUM_THREADS=1, %.2f s" % (n2, one[0]),
                "all_core_same_sample": {"value": n2 / many[0], "cores": many[1], "seconds": many[0]},
                "extrapolated_to_this_workload": {"value": cpu["value"] * many[0] / one[0],
                                                  "how": "all-core value of this workload x (all-core / single-thread "
                                                         "time ratio measured on config2)"}}

    if ranks.rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "particle-updates/s", "n_gpus": world, "steps": K,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_max / K, "ms_per_step_pipelined": 1e3 * t_pipe_max / K,
            "ms_per_step_serial": 1e3 * t_serial_max / K, "ms_per_step_graph": 1e3 * t_graph_max / K,
            "ms_per_step_graph_pipelined4": 1e3 * t_graph4_max / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(cfg, world),
            "run": {"grid_cells": C, "triangles_last_frame": n_tris,
                    "frame_loop": mode + ": the same K frames are timed four ways -- the surface pass of frame t beside "
                                  "the SPH step of frame t+1 (mc_extract_async), the synchronous calls, the synchronous frame "
                                  "replayed from a CUDA graph, and a CUDA graph of four pipelined frames -- `value` is the "
                                  "fastest; `parts` come from the synchronous loop"},
            "parts": {
                "sph_boid": {"value": n * K * world / t_sim_max, "unit": "particle-updates/s",
                             "ms_per_step": 1e3 * t_sim_max / K, "algorithmic_gbs": sim_gbs,
                             "frac_of_hbm_peak": sim_gbs / peak,
                             "rows": "S1-S13: sph_step + boid_step + the frame's one sph_build_grid"},
                "mc": {"value": G ** 3 * K * world / t_mc_max, "unit": "voxels/s", "ms_per_step": 1e3 * t_mc_max / K,
                       "algorithmic_gbs": mc_gbs, "frac_of_hbm_peak": mc_gbs / peak, "rows": "S14-S17: mc_extract"},
            },
            "roofline": roof,
            "kernels": [{"kernel": r["kernel"], "launches": r["launches"], "avg_us": round(r["avg_us"], 2),
                         "share": round(r["share"], 4), "gbs": round(r["gbs"], 1), "frac": round(r["frac"], 4)}
                        for r in rows],
            "kernel_timing": {"how": "the same K frames run a second time with a CUDA event pair around every launch "
                                     "(on the launching stream); `value` comes from the first, un-instrumented run",
                              "ms_per_step_instrumented": 1e3 * t_profiled / K},
            "indexed_mesh": indexed, "neighbour_search_ab": nsearch, "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "cpu_baseline": cpu,
        }
        print(json.dumps(line))
    ranks.close()


if __name__ == "__main__":
    main()
