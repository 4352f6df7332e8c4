"""N2 host logic on the CPU: slab layout, and the decomposed step end to end under gloo with world_size 2 (one process
per rank, neighbour exchange through torch.distributed) against the undecomposed oracle step."""
import os
import subprocess
import sys

import numpy as np

from paper_2311_15088_b200 import slab as S
from paper_2311_15088_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_layout_owns_every_coordinate_once():
    sph = W.config(3, scale=4)["sph"]  # box [0,2] x [0,1] x [0,1], h = 1/32: 64 cells along x
    for world in (1, 2, 3, 5):
        lay = S.SlabLayout(sph, world)
        assert lay.axis == 0 and lay.dim == 64 and len(lay.faces) == world - 1
        b = [lay.bounds(r) for r in range(world)]
        assert b[0][0] == -np.inf and b[-1][1] == np.inf
        for r in range(world - 1):
            assert b[r][1] == b[r + 1][0]  # faces shared, slabs contiguous
            assert abs(b[r][1] / sph["h"] - round(b[r][1] / sph["h"])) < 1e-6  # on a cell boundary
        x = np.float32(np.linspace(-0.5, 2.5, 1001))
        own = lay.owner(x)
        for r in range(world):
            lo, hi = b[r]
            assert np.array_equal(own == r, (x >= np.float32(lo)) & (x < np.float32(hi)))


def test_loopback_decomposition_equals_undecomposed_oracle():
    # 3 emulated ranks in one process, oracle as the stepper: four steps with migration; every particle ends where the
    # undecomposed oracle puts it (the neighbour sets are identical; only the order of the binary64 sums can differ)
    from oracle import refbind as R
    from tests.slabutil import OracleBackend, gather_by_id, tagged_state
    cfg = W.config(1)
    pos, vel = tagged_state(cfg)
    lay = S.SlabLayout(cfg["sph"], 3)
    ex = S.LoopbackExchange(3)
    be = OracleBackend(cfg["sph"])
    sims = [S.SlabSim(lay, r, be, ex, be.to_device(p), be.to_device(v)) for r, (p, v) in enumerate(S.split_initial(lay, pos, vel))]
    rp, rv = pos, vel
    moved = 0
    for _ in range(4):
        S.run_loopback(sims, 1)
        out = R.step(cfg["sph"], rp, rv)
        rp, rv = out["pos"], out["vel"]
        moved += sum(s.stats["migrated_out"] for s in sims)
        for s in sims:  # every rank owns exactly the particles of its slab
            x = s.pos[:, lay.axis].numpy()
            assert ((x >= np.float32(s.lo)) & (x < np.float32(s.hi))).all()
    assert moved > 0 and sims[0].stats["ghosts"] > 0 and sims[1].stats["ghosts"] > 0  # (rank 2's slab is empty)
    gp, gv = gather_by_id([(s.pos.numpy(), s.vel.numpy()) for s in sims], cfg["n"])
    assert np.abs(gp[:, :3] - rp[:, :3]).max() <= 1e-6 and np.abs(gv[:, :3] - rv[:, :3]).max() <= 1e-5



def test_loopback_decomposition_with_boids_equals_undecomposed_oracle():
    # fluid AND boids cut into slabs (ghost boids, wider fluid halo: push radius + h), oracle as the stepper: every
    # particle and every boid ends where the undecomposed oracle frames put it; boids migrate too
    from tests.slabutil import OracleBackend, gather_by_id, reference_frames, tagged_boids, tagged_state
    cfg = W.config(1)
    pos, vel = tagged_state(cfg)
    bpos, bvel, boid = tagged_boids(cfg)
    world = 3
    lay = S.SlabLayout(cfg["sph"], world, boid=boid)
    assert lay.halo_width() >= boid["push_radius"] + cfg["sph"]["h"] - 1e-6 and lay.boid_halo_width() >= boid["visible_range"]
    ex = S.LoopbackExchange(world)
    be = OracleBackend(cfg["sph"])
    fluid = S.split_initial(lay, pos, vel)
    boids = S.split_initial(lay, bpos, bvel)
    sims = [S.SlabSim(lay, r, be, ex, be.to_device(fluid[r][0]), be.to_device(fluid[r][1]), be.to_device(boids[r][0]),
                      be.to_device(boids[r][1]), boid) for r in range(world)]
    steps, moved = 4, 0
    for _ in range(steps):
        S.run_loopback(sims, 1)
        moved += sum(s.stats["boids_migrated_out"] for s in sims)
        for s in sims:
            x = s.bpos[:, lay.axis].numpy()
            assert ((x >= np.float32(s.lo)) & (x < np.float32(s.hi))).all()
    assert moved > 0 and sum(s.stats["boid_ghosts"] for s in sims) > 0
    rp, rv, rbp, rbv = reference_frames(cfg, pos, vel, bpos, bvel, boid, steps)
    gp, gv = gather_by_id([(s.pos.numpy(), s.vel.numpy()) for s in sims], cfg["n"])
    gbp, gbv = gather_by_id([(s.bpos.numpy(), s.bvel.numpy()) for s in sims], cfg["n_boid"])
    assert np.abs(gp[:, :3] - rp[:, :3]).max() <= 1e-6 and np.abs(gv[:, :3] - rv[:, :3]).max() <= 1e-5
    assert np.abs(gbp[:, :3] - rbp[:, :3]).max() <= 1e-6 and np.abs(gbv[:, :3] - rbv[:, :3]).max() <= 2e-5


def test_slab_layout_rejects_slabs_narrower_than_a_halo():
    import pytest
    cfg = W.config(1)  # 16 cells of h along x; visible range 0.1 = 1.6 h, push radius h: fluid halo 2 h, boid halo 1.6 h
    S.SlabLayout(cfg["sph"], 8, boid=cfg["boid"])  # 2 cells per rank: just wide enough
    with pytest.raises(ValueError):
        S.SlabLayout(cfg["sph"], 16, boid=cfg["boid"])
    with pytest.raises(ValueError):
        S.SlabLayout(cfg["sph"], 8, boid=dict(cfg["boid"], push_radius=2.0 * cfg["sph"]["h"]))  # fluid halo 3 h


def test_loopback_decomposed_surface_adds_up_to_the_undecomposed_mesh():
    # three emulated ranks, oracle as the stepper and as the mesher: every rank polygonises the cubes of its slab from
    # [owned | ghost] particles; each list is the undecomposed mesh's ordered subset for those cubes
    import torch
    from oracle import refbind as R
    from tests.slabutil import OracleBackend, gather_by_id, tagged_state, triangles_in_cube_range
    cfg = W.config(1)
    mc = W.mc_params(cfg)
    pos, vel = tagged_state(cfg)
    world = 3
    lay = S.SlabLayout(cfg["sph"], world, mc=mc)
    assert lay.halo_width() >= mc["radius"] + mc["spacing"] - 1e-7
    q = mc["n_point_per_axis"] - 1
    rng = [lay.cube_range(r) for r in range(world)]
    assert rng[0][0] == 0 and rng[-1][1] == q and all(rng[r][1] == rng[r + 1][0] for r in range(world - 1))
    ex = S.LoopbackExchange(world)
    be = OracleBackend(cfg["sph"])
    sims = [S.SlabSim(lay, r, be, ex, be.to_device(p), be.to_device(v)) for r, (p, v) in enumerate(S.split_initial(lay, pos, vel))]
    bufs = [torch.zeros(20000, 3, 3) for _ in range(world)]
    S.run_loopback(sims, 2)  # two frames without the surface pass (particles migrate), then one with it
    state = gather_by_id([(s.pos.numpy(), s.vel.numpy()) for s in sims], cfg["n"])[0]
    counts = S.run_loopback(sims, 1, tris=bufs)
    phi = R.voxel_sdf(cfg["sph"], mc, state)
    t_ref, nt_ref, cases = R.mc_polygonise(mc, phi, want_cases=True)
    assert sum(counts) == nt_ref and nt_ref > 0 and min(counts[:2]) > 0
    for r in range(world):
        keep = triangles_in_cube_range(mc, cases, lay.axis, *rng[r])
        assert counts[r] == int(keep.sum())
        if counts[r]:
            assert np.abs(bufs[r].numpy()[:counts[r]] - t_ref[keep]).max() <= 1e-6

_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch
import torch.distributed as dist
from paper_2311_15088_b200 import slab as S, workloads as W
from tests.slabutil import OracleBackend, tagged_state
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
cfg = W.config(1)
pos, vel = tagged_state(cfg)
be = OracleBackend(cfg["sph"])
ex = S.DistExchange(dist, rank, world, torch.device("cpu"))
if os.environ.get("SLAB_BOIDS") == "1":
    from tests.slabutil import tagged_boids
    bpos, bvel, boid = tagged_boids(cfg)
    lay = S.SlabLayout(cfg["sph"], world, boid=boid, mc=W.mc_params(cfg))
    p, v = S.split_initial(lay, pos, vel)[rank]
    bp, bv = S.split_initial(lay, bpos, bvel)[rank]
    sim = S.SlabSim(lay, rank, be, ex, be.to_device(p), be.to_device(v), be.to_device(bp), be.to_device(bv), boid)
else:
    lay = S.SlabLayout(cfg["sph"], world)
    p, v = S.split_initial(lay, pos, vel)[rank]
    sim = S.SlabSim(lay, rank, be, ex, be.to_device(p), be.to_device(v))
for _ in range(3):
    sim.step()
np.save({out!r} % rank, np.concatenate([sim.pos.numpy(), sim.vel.numpy()], 1))
if sim.boid is not None:
    np.save({bout!r} % rank, np.concatenate([sim.bpos.numpy(), sim.bvel.numpy()], 1))
    # a fourth frame with the surface pass of its start state (the state saved above) for this rank's cubes
    tris = torch.zeros(20000, 3, 3)
    nt = sim.step(tris)
    np.save({tout!r} % rank, tris.numpy()[:nt])
dist.barrier()
dist.destroy_process_group()
print("rank", rank, "ok", sim.n_owned, sim.stats)
"""


def _run_world2(tmp_path, boids):
    script = tmp_path / "worker.py"
    out_pat, bout_pat = str(tmp_path / "rank%d.npy"), str(tmp_path / "boids%d.npy")
    script.write_text(_WORKER.format(root=ROOT, out=out_pat, bout=bout_pat, tout=str(tmp_path / "tris%d.npy")))
    port = 29900 + (os.getpid() + (45 if boids else 0)) % 90
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2", SLAB_BOIDS="1" if boids else "0")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for rank, p in enumerate(procs):
        out, _ = p.communicate(timeout=300)
        assert p.returncode == 0, out
        assert "rank %d ok" % rank in out
    return out_pat, bout_pat


def test_decomposed_frames_with_boids_under_gloo_world_size_2(tmp_path):
    from tests.slabutil import gather_by_id, reference_frames, tagged_boids, tagged_state
    out_pat, bout_pat = _run_world2(tmp_path, True)
    cfg = W.config(1)
    pos, vel = tagged_state(cfg)
    bpos, bvel, boid = tagged_boids(cfg)
    rp, rv, rbp, rbv = reference_frames(cfg, pos, vel, bpos, bvel, boid, 3)
    parts, bparts = [], []
    for rank in range(2):
        a, b = np.load(out_pat % rank), np.load(bout_pat % rank)
        parts.append((a[:, :4], a[:, 4:]))
        bparts.append((b[:, :4], b[:, 4:]))
    gp, gv = gather_by_id(parts, cfg["n"])
    gbp, gbv = gather_by_id(bparts, cfg["n_boid"])
    assert np.abs(gp[:, :3] - rp[:, :3]).max() <= 1e-6 and np.abs(gv[:, :3] - rv[:, :3]).max() <= 1e-5
    assert np.abs(gbp[:, :3] - rbp[:, :3]).max() <= 1e-6 and np.abs(gbv[:, :3] - rbv[:, :3]).max() <= 2e-5
    # the surface pass of the two ranks: each the ordered subset of the mesh of the gathered state for its cubes
    from oracle import refbind as R
    from tests.slabutil import triangles_in_cube_range
    mc = W.mc_params(cfg)
    lay = S.SlabLayout(cfg["sph"], 2, boid=boid, mc=mc)
    t_ref, nt_ref, cases = R.mc_polygonise(mc, R.voxel_sdf(cfg["sph"], mc, gp), want_cases=True)
    total = 0
    for rank in range(2):
        t = np.load(str(tmp_path / "tris%d.npy") % rank)
        keep = triangles_in_cube_range(mc, cases, lay.axis, *lay.cube_range(rank))
        assert t.shape[0] == int(keep.sum()) and t.shape[0] > 0
        assert np.abs(t - t_ref[keep]).max() <= 1e-6
        total += t.shape[0]
    assert total == nt_ref


def test_decomposed_step_under_gloo_world_size_2(tmp_path):
    from oracle import refbind as R
    from tests.slabutil import gather_by_id, tagged_state
    out_pat, _ = _run_world2(tmp_path, False)
    cfg = W.config(1)
    rp, rv = tagged_state(cfg)
    for _ in range(3):
        o = R.step(cfg["sph"], rp, rv)
        rp, rv = o["pos"], o["vel"]
    parts = []
    for rank in range(2):
        a = np.load(out_pat % rank)
        parts.append((a[:, :4], a[:, 4:]))
    gp, gv = gather_by_id(parts, cfg["n"])
    assert np.abs(gp[:, :3] - rp[:, :3]).max() <= 1e-6 and np.abs(gv[:, :3] - rv[:, :3]).max() <= 1e-5


def test_faces_cut_by_particle_count_balance_config4_over_8_ranks():
    """N2: config 4's fluid fills half of the box along the slab axis, so uniform cell slabs leave half of the ranks
    empty at t = 0 (max owned / mean = 2.0); faces cut from the cell-column histogram balance it within 10 %, stay on
    cell boundaries, keep every slab at least a halo wide, and every coordinate still has exactly one owner."""
    cfg = W.config(4)
    mc = W.mc_params(cfg)
    for world in (2, 4, 8):
        uni = S.SlabLayout(cfg["sph"], world, boid=cfg["boid"], mc=mc)
        bal = S.SlabLayout(cfg["sph"], world, boid=cfg["boid"], mc=mc, pos=cfg["pos"])
        x = cfg["pos"][:, bal.axis]
        own_u = np.bincount(uni.owner(x), minlength=world)
        own_b = np.bincount(bal.owner(x), minlength=world)
        assert own_u.sum() == own_b.sum() == cfg["n"]
        assert own_u.max() / (cfg["n"] / world) > 1.9
        assert own_b.max() / (cfg["n"] / world) <= 1.10
        widths = np.diff([0] + bal.cuts + [bal.dim])
        assert (widths * bal.h >= max(bal.fluid_halo, bal.boid_halo) - 1e-9).all()
        for r in range(world):
            lo, hi = bal.bounds(r)
            sel = bal.owner(x) == r
            assert ((x[sel] >= np.float32(lo)) & (x[sel] < np.float32(hi))).all()
    # a histogram with everything in one column cannot be balanced: the cuts fall back to the narrowest legal slabs
    cuts = S.SlabLayout.balanced_cuts(np.array([0, 0, 1000, 0, 0, 0, 0, 0, 0, 0, 0, 0]), 3, 3)
    assert cuts == [3, 6] or (np.diff([0] + cuts + [12]) >= 3).all()


def test_recut_moves_the_faces_and_the_particles_two_hops_if_needed():
    """N2 re-cut (SlabSim.recut / run_recut): three emulated ranks start from uniform cell slabs of config 1 (the fluid
    fills half of the box: ranks own 3/4, 1/4 and nothing), the faces are re-cut from the global column histogram, the
    particles move to their new owners -- some from rank 0 to rank 2, two hops -- and the decomposed frames that follow
    still match the undecomposed oracle."""
    from oracle import refbind as R
    from tests.slabutil import OracleBackend, gather_by_id, tagged_state
    cfg = W.config(1)
    pos, vel = tagged_state(cfg, speed=2.0)
    world, n = 3, cfg["n"]
    lay = S.SlabLayout(cfg["sph"], world)
    assert lay.cuts == [6, 12]
    ex = S.LoopbackExchange(world)
    be = OracleBackend(cfg["sph"])
    sims = [S.SlabSim(lay, r, be, ex, be.to_device(p), be.to_device(v)) for r, (p, v) in enumerate(S.split_initial(lay, pos, vel))]
    assert [s.n_owned for s in sims] == [3 * n // 4, n // 4, 0]
    S.run_loopback(sims, 1)
    ref = R.step(cfg["sph"], pos, vel)
    cuts = S.run_recut(sims)
    assert cuts != [6, 12] and cuts == lay.cuts
    owned = np.array([s.n_owned for s in sims])
    assert owned.sum() == n and owned.max() / owned.mean() < 1.35 and owned.min() > 0
    for s in sims:
        x = s.pos[:, lay.axis].numpy()
        lo, hi = lay.bounds(s.rank)
        assert ((x >= np.float32(lo)) & (x < np.float32(hi))).all()
    gp, gv = gather_by_id([(s.pos.numpy(), s.vel.numpy()) for s in sims], n)
    assert np.array_equal(gp, ref["pos"]) or np.abs(gp - ref["pos"]).max() <= 1e-6   # the re-cut moves owners, not particles
    rp, rv = ref["pos"], ref["vel"]
    for _ in range(2):
        S.run_loopback(sims, 1)
        o = R.step(cfg["sph"], rp, rv)
        rp, rv = o["pos"], o["vel"]
    gp, gv = gather_by_id([(s.pos.numpy(), s.vel.numpy()) for s in sims], n)
    assert np.abs(gp[:, :3] - rp[:, :3]).max() <= 1e-6 and np.abs(gv[:, :3] - rv[:, :3]).max() <= 1e-5
