"""Parity of S7, S11-S13 (boid grid, probe density, boid rules, fluid->boid force, move) against the oracle."""
import numpy as np
import pytest
import torch

from oracle import refbind as R
from paper_2311_15088_b200 import binding as B
from paper_2311_15088_b200 import workloads as W
from tests.gpuutil import Sim, dev, vec_err

pytestmark = pytest.mark.gpu


def _frame(cfg, pos, vel, bpos, bvel):
    ref = R.step(cfg["sph"], pos, vel, bpos, bvel, cfg["boid"])
    refb = R.boid_step(cfg["sph"], cfg["boid"], pos, vel, ref["density"], bpos, bvel)
    with Sim(cfg) as sim:
        dbp, dbv = dev(bpos), dev(bvel)
        sim.step(dev(pos), dev(vel), dbp, dbv, cfg["boid"])
        out = sim.boid_step(cfg["boid"], dbp, dbv)
    return refb, out


def _compare(refb, out):
    bad, worst = vec_err(out["bvel"][:, :3], refb["bvel"][:, :3])
    assert bad == 0, ("bvel", bad, worst)
    bad, worst = vec_err(out["bpos"][:, :3], refb["bpos"][:, :3])
    assert bad == 0, ("bpos", bad, worst)
    # the four velocity increments (sep, ali, coh, fluid) per boid and per rule, each as a vector with the per-step
    # tolerance of DESIGN.md section 5 (1e-5 |ref| + floor); the floor is 1e-7: the increments are ~1e-3 .. 1e-1
    for k, rule in enumerate(("sep", "ali", "coh", "fluid")):
        bad, worst = vec_err(out["dv_parts"][:, k, :3], refb["dv_parts"][:, k, :3], abs_=1e-7)
        assert bad == 0, ("dv_" + rule, bad, worst)


@pytest.mark.parametrize("idx,scale", [(1, None), (2, None), (3, 2), (4, 4), (5, 4)])
def test_boid_step_matches_oracle(idx, scale):
    cfg = W.config(idx, scale=scale)
    vel0 = W.uniform_box(cfg["n"], (-0.2,) * 3, (0.2,) * 3, 1, 30)
    refb, out = _frame(cfg, cfg["pos"], vel0, cfg["bpos"], cfg["bvel"])
    _compare(refb, out)
    if idx in (3, 4, 5):
        assert np.abs(refb["dv_parts"][:, 3]).max() > 0  # fluid -> boid force is live


def test_boids_outside_space_fast_and_slow():
    cfg = W.config(1)
    bp = dict(cfg["boid"], min_speed=0.05)
    cfg = dict(cfg, boid=bp)
    bpos = W.uniform_box(200, (-0.2, -0.2, -0.2), (1.2, 1.2, 1.2), 3, 10)  # some outside the Boid Space: edge rule
    bvel = W.uniform_box(200, (-1.0,) * 3, (1.0,) * 3, 3, 20)              # many above max_speed
    bvel[:20, :3] *= 0.01                                                  # some below min_speed
    bvel[20] = 0.0
    cfg["n_boid"] = 200
    refb, out = _frame(cfg, cfg["pos"], cfg["vel"], bpos, bvel)
    _compare(refb, out)


def test_single_boid_and_clustered_boids():
    cfg = W.config(3, scale=4)
    one_p, one_v = cfg["bpos"][:1].copy(), cfg["bvel"][:1].copy()
    refb, out = _frame(dict(cfg, n_boid=1), cfg["pos"], cfg["vel"], one_p, one_v)
    _compare(refb, out)
    h = cfg["sph"]["h"]
    bpos = W.uniform_ball(900, (0.12, 0.12, 0.12), 2.0 * h, 5, 10)  # hundreds of boid neighbours each
    bvel = W.uniform_box(900, (-0.1,) * 3, (0.1,) * 3, 5, 20)
    refb, out = _frame(dict(cfg, n_boid=900), cfg["pos"], cfg["vel"], bpos, bvel)
    _compare(refb, out)


def test_boid_step_requires_matching_sph_step():
    cfg = W.config(1)
    with Sim(cfg) as sim:
        bpos, bvel = dev(cfg["bpos"]), dev(cfg["bvel"])
        with pytest.raises(B.SphError) as e:
            B.boid_step(sim.ctx, cfg["boid"], bpos, bvel)
        assert e.value.code == B.SPH_E_STALE_GRID
        sim.step(dev(cfg["pos"]), dev(cfg["vel"]), bpos, bvel, cfg["boid"])
        B.boid_step(sim.ctx, cfg["boid"], bpos, bvel)
        with pytest.raises(B.SphError):  # the boids moved: a second boid_step in the same frame is stale
            B.boid_step(sim.ctx, cfg["boid"], bpos, bvel)
        torch.cuda.synchronize()


def test_two_frames_free_running():
    cfg = W.config(3, scale=4)
    pos, vel, bpos, bvel = cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"]
    with Sim(cfg) as sim:
        dp, dv, dbp, dbv = dev(pos), dev(vel), dev(bpos), dev(bvel)
        for _ in range(2):
            ref = R.step(cfg["sph"], pos, vel, bpos, bvel, cfg["boid"])
            refb = R.boid_step(cfg["sph"], cfg["boid"], pos, vel, ref["density"], bpos, bvel)
            pos, vel, bpos, bvel = ref["pos"], ref["vel"], refb["bpos"], refb["bvel"]
            sim.step(dp, dv, dbp, dbv, cfg["boid"])
            out = sim.boid_step(cfg["boid"], dbp, dbv)
        bad, worst = vec_err(out["bvel"][:, :3], bvel[:, :3], rel=2e-5, abs_=2e-6)
        assert bad == 0, (bad, worst)


# ---- N4: obstacle avoidance (P:261, P:336 step 7; D:C-OBST) ----------------------------------------------------------
@pytest.mark.parametrize("idx,scale", [(1, None), (3, 2)])
def test_boid_step_with_obstacle_grid_matches_oracle(idx, scale):
    import torch
    from paper_2311_15088_b200 import binding as B
    cfg = W.config(idx, scale=scale)
    bp = cfg["boid"]
    lo, hi = np.array(bp["space_min"]), np.array(bp["space_max"])
    centre = cfg["bpos"][:, :3].mean(axis=0).astype(np.float64)  # an obstacle in the middle of the swarm
    op, normals = W.sphere_obstacle(lo, hi, 0.6 * bp["visible_range"], centre, 0.8 * bp["visible_range"],
                                    w_obs=0.07, heavy=2.5)
    ref = R.step(cfg["sph"], cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"], bp)
    refb = R.boid_step(cfg["sph"], bp, cfg["pos"], cfg["vel"], ref["density"], cfg["bpos"], cfg["bvel"])
    want = R.boid_obstacles(op, normals, bp["protect_range"], bp["visible_range"], refb["bpos"], refb["bvel"])
    assert (want != refb["bvel"]).any()  # the obstacle really acts on some boids
    with Sim(cfg) as sim:
        nrm = dev(normals)
        B.boid_set_obstacles(sim.ctx, op, nrm)
        pos, vel, bpos, bvel = dev(cfg["pos"]), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"])
        sim.step(pos, vel, bpos, bvel, bp)
        out = sim.boid_step(bp, bpos, bvel)
        bad, worst = vec_err(out["bpos"][:, :3], refb["bpos"][:, :3])
        assert bad == 0, ("bpos", bad, worst)
        bad, worst = vec_err(out["bvel"][:, :3], want[:, :3])
        assert bad == 0, ("bvel", bad, worst)
        # untouched boids are bitwise the plain step's; cleared grid -> plain step again
        same = (want == refb["bvel"]).all(axis=1)
        B.boid_set_obstacles(sim.ctx, None, None)
        pos, vel, bpos, bvel = dev(cfg["pos"]), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"])
        sim.step(pos, vel, bpos, bvel, bp)
        plain = sim.boid_step(bp, bpos, bvel)
        assert np.array_equal(plain["bvel"][same], out["bvel"][same])
        bad, worst = vec_err(plain["bvel"][:, :3], refb["bvel"][:, :3])
        assert bad == 0


def test_dv_parts_written_on_the_stream_just_before_the_call_is_ordered():
    # include/sphboid.h, boid_step stream contract: the library runs the step on a stream of its own beside the force
    # pass; a fill of dv_parts enqueued on the caller's stream right before the call (here behind a long matmul, so it
    # really is late) must still land BEFORE the kernel's writes
    cfg = W.config(2)
    ref = R.step(cfg["sph"], cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"], cfg["boid"])
    refb = R.boid_step(cfg["sph"], cfg["boid"], cfg["pos"], cfg["vel"], ref["density"], cfg["bpos"], cfg["bvel"])
    with Sim(cfg) as sim:
        pos, vel, bpos, bvel = dev(cfg["pos"]), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"])
        big = torch.randn(4096, 4096, device="cuda")
        parts = torch.empty(cfg["n_boid"], 4, 4, device="cuda")
        for _ in range(3):
            bp, bv = bpos.clone(), bvel.clone()
            B.sph_step(sim.ctx, pos.clone(), vel.clone(), bp, bv, cfg["boid"])
            _ = big @ big                      # keeps the stream busy ...
            parts.fill_(float("nan"))          # ... so this fill is still queued when boid_step is called
            B.boid_step(sim.ctx, cfg["boid"], bp, bv, dv_parts=parts)
            torch.cuda.synchronize()
            got = parts.cpu().numpy()
            assert np.isfinite(got[:, :, :3]).all()
            for k in range(4):
                bad, worst = vec_err(got[:, k, :3], refb["dv_parts"][:, k, :3], abs_=1e-7)
                assert bad == 0, (k, bad, worst)
