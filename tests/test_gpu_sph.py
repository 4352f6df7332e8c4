"""Parity of S6-S10 (density, neighbour count, forces, boid push, integration) against the oracle.

Integers (ncount, touched) bit-exact.  Floats per particle, vector norm:
  rho, v, x : |d| <= 1e-5 |ref| + 1e-6            a : |d| <= 1e-5 |a_ref| + 1e-6
  step displacement x' - x : |d| <= 1e-5 |ref| + 2 ulp(box extent)   (x itself is stored in binary32)
"""
import numpy as np
import pytest
import torch

from oracle import refbind as R
from paper_2311_15088_b200 import binding as B
from paper_2311_15088_b200 import workloads as W
from tests import gpuutil
from tests.gpuutil import Sim, dev, vec_err

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True, params=[1, 2], ids=["nbrlist", "masks"])
def force_variant(request):
    """Every test runs on both S6 / S8 paths: the stored 16-bit neighbour list (default) and the brick density pass with
    neighbour masks (sph_set_force_variant)."""
    gpuutil.FORCE_VARIANT = request.param
    yield request.param
    gpuutil.FORCE_VARIANT = None


def _compare_step(cfg, out, ref, pos0):
    assert np.array_equal(out["ncount"], ref["ncount"])
    assert np.array_equal(out["touched"], ref["touched"])
    bad, worst = vec_err(out["density"], ref["density"])
    assert bad == 0, ("density", bad, worst)
    bad, worst = vec_err(out["accel"][:, :3], ref["accel"][:, :3])
    assert bad == 0, ("accel", bad, worst)
    bad, worst = vec_err(out["vel"][:, :3], ref["vel"][:, :3])
    assert bad == 0, ("vel", bad, worst)
    bad, worst = vec_err(out["pos"][:, :3], ref["pos"][:, :3])
    assert bad == 0, ("pos", bad, worst)
    ulp = 2.0 * np.spacing(np.float32(max(cfg["sph"]["box_max"])))
    bad, worst = vec_err(out["pos"][:, :3] - pos0[:, :3], ref["pos"][:, :3] - pos0[:, :3], abs_=float(ulp) * np.sqrt(3))
    assert bad == 0, ("displacement", bad, worst)
    # the 4th lanes are carried through
    assert np.array_equal(out["pos"][:, 3], pos0[:, 3])


@pytest.mark.parametrize("idx,scale", [(1, None), (2, None), (3, 2), (4, 4), (5, 4)])
def test_single_step_matches_oracle(idx, scale):
    cfg = W.config(idx, scale=scale)
    vel0 = W.uniform_box(cfg["n"], (-0.2,) * 3, (0.2,) * 3, 1, 30)
    pos0 = cfg["pos"].copy()
    pos0[:, 3] = np.arange(cfg["n"], dtype=np.float32)  # payload lane must survive
    ref = R.step(cfg["sph"], pos0, vel0, cfg["bpos"], cfg["bvel"], cfg["boid"])
    with Sim(cfg) as sim:
        out = sim.step(dev(pos0), dev(vel0), dev(cfg["bpos"]), dev(cfg["bvel"]), cfg["boid"])
    _compare_step(cfg, out, ref, pos0)
    if idx in (3, 4, 5):
        assert ref["touched"].max() > 0  # the coupling path really ran


def test_step_without_boids_and_explicit_grid():
    cfg = W.config(1)
    ref = R.step(cfg["sph"], cfg["pos"], cfg["vel"])
    with Sim(cfg) as sim:
        pos, vel = dev(cfg["pos"]), dev(cfg["vel"])
        sim.build_grid(pos, vel)  # sph_step must reuse this grid (same pointers), result identical either way
        out = sim.step(pos, vel)
    _compare_step(cfg, out, ref, cfg["pos"])
    assert not out["touched"].any()


def test_teacher_forced_ten_steps_config1():
    # D:A-MULTI (i): feed the oracle's state to the GPU at every step, single-step tolerances each time
    cfg = W.config(1)
    pos, vel = cfg["pos"], cfg["vel"]
    with Sim(cfg) as sim:
        for _ in range(10):
            ref = R.step(cfg["sph"], pos, vel, cfg["bpos"], cfg["bvel"], cfg["boid"])
            out = sim.step(dev(pos), dev(vel), dev(cfg["bpos"]), dev(cfg["bvel"]), cfg["boid"])
            _compare_step(cfg, out, ref, pos)
            pos, vel = ref["pos"], ref["vel"]


def test_free_running_ten_steps_config1_bounded_divergence():
    # D:A-MULTI (ii): free-running states stay within a stated growing bound: eps(s) = s * (1e-5 |x| + 2e-6)
    cfg = W.config(1)
    rp, rv = cfg["pos"], cfg["vel"]
    with Sim(cfg) as sim:
        gp, gv = dev(cfg["pos"]), dev(cfg["vel"])
        for s in range(1, 11):
            ref = R.step(cfg["sph"], rp, rv)
            rp, rv = ref["pos"], ref["vel"]
            out = sim.step(gp, gv)
            bad, worst = vec_err(out["pos"][:, :3], rp[:, :3], rel=1e-5 * s, abs_=2e-6 * s)
            assert bad <= cfg["n"] // 10000, (s, bad, worst)
            bad, worst = vec_err(out["vel"][:, :3], rv[:, :3], rel=1e-5 * s, abs_=2e-5 * s)
            assert bad <= cfg["n"] // 10000, (s, bad, worst)


def test_walls_and_out_of_box_particles():
    cfg = W.config(1, scale=2)
    sp = cfg["sph"]
    pos = W.random_cloud(3000, (-0.02, -0.02, -0.02), (0.3, 0.3, 0.3), seed=7)  # some start outside the box
    vel = W.uniform_box(3000, (-30.0,) * 3, (30.0,) * 3, 8, 30)                  # many hit a wall in one step
    ref = R.step(sp, pos, vel)
    with Sim(dict(sph=sp, n=3000)) as sim:
        out = sim.step(dev(pos), dev(vel))
    assert (ref["pos"][:, :3] == 0.0).sum() > 100
    _compare_step(dict(sph=sp), out, ref, pos)
    assert np.array_equal(out["pos"][:, :3] == 0.0, ref["pos"][:, :3] == 0.0)


def test_dense_cluster_many_neighbours():
    # degenerate: hundreds of neighbours per particle (one cell holds them all), plus coincident particles
    sp = dict(W.config(1)["sph"])
    pos = W.random_cloud(700, (0.40, 0.40, 0.40), (0.43, 0.43, 0.43), seed=11)
    pos[10] = pos[11]  # coincident pair: counted as neighbours, no force between them
    vel = W.uniform_box(700, (-0.1,) * 3, (0.1,) * 3, 12, 30)
    ref = R.step(sp, pos, vel)
    with Sim(dict(sph=sp, n=700)) as sim:
        out = sim.step(dev(pos), dev(vel))
    assert ref["ncount"].min() > 300
    _compare_step(dict(sph=sp), out, ref, pos)


@pytest.mark.parametrize("idx", [4, 5])
def test_full_size_step_matches_oracle(idx):
    # BASELINE.json's full sizes in the launch configuration bench.py times (one whole step, every particle compared)
    cfg = W.config(idx)
    ref = R.step(cfg["sph"], cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"], cfg["boid"])
    with Sim(cfg) as sim:
        out = sim.step(dev(cfg["pos"]), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"]), cfg["boid"])
    _compare_step(cfg, out, ref, cfg["pos"])


@pytest.mark.parametrize("idx,frames", [(2, 100), (3, 100), (4, 100), (5, 20)])
def test_free_running_frames_as_baseline_states_them(idx, frames, force_variant):
    """BASELINE.json configs[1..4] with the particle, boid and step counts they state (65 536 / 256 / 100, 262 144 / 1 024 /
    100 with the boids pushing the fluid, 1 048 576 / 4 096 / 100, 4 194 304 / 16 384 / 20).  The GPU frames (sph_step +
    boid_step) run free beside the oracle's; D:A-MULTI (ii) bounds the divergence by eps(s) = s * (1e-5 |x| + 2e-6) (2e-5
    for velocities).  Measured on B200 after 100 frames of config 2: max |dpos| 2.7e-7, max |dvel| 8.7e-7, two neighbour
    counts off by one, so a fixed bound of ten single-step floors is asserted at the end as well; the neighbour counts
    (integers decided on r^2 < h^2) may differ only where a pair sits within rounding of h."""
    if force_variant == 2 and idx not in (2, 5):
        pytest.skip("the default path runs every config, the mask path configs 2 and 5 (the dense one)")
    cfg = W.config(idx)
    rp, rv, rbp, rbv = cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"]
    with Sim(cfg) as sim:
        gp, gv, gbp, gbv = dev(rp), dev(rv), dev(rbp), dev(rbv)
        for s in range(1, frames + 1):
            ref = R.step(cfg["sph"], rp, rv, rbp, rbv, cfg["boid"])
            refb = R.boid_step(cfg["sph"], cfg["boid"], rp, rv, ref["density"], rbp, rbv)
            rp, rv, rbp, rbv = ref["pos"], ref["vel"], refb["bpos"], refb["bvel"]
            out = sim.step(gp, gv, gbp, gbv, cfg["boid"])
            ob = sim.boid_step(cfg["boid"], gbp, gbv)
            if s % 10 == 0:
                for got, want, a in ((out["pos"], rp, 2e-6), (out["vel"], rv, 2e-5), (ob["bpos"], rbp, 2e-6), (ob["bvel"], rbv, 2e-5)):
                    bad, worst = vec_err(got[:, :3], want[:, :3], rel=1e-5 * s, abs_=a * s)
                    assert bad == 0, (s, bad, worst)
    assert float(np.abs(out["pos"][:, :3] - rp[:, :3]).max()) < 1e-5
    assert float(np.abs(out["vel"][:, :3] - rv[:, :3]).max()) < 1e-4
    assert float(np.abs(ob["bpos"][:, :3] - rbp[:, :3]).max()) < 1e-5
    assert int((out["ncount"] != ref["ncount"]).sum()) <= cfg["n"] // 1000
    print("free run, config %d, %d frames: max|dpos| %.3g max|dvel| %.3g ncount mismatches %d" % (
        idx, frames,
        float(np.abs(out["pos"][:, :3] - rp[:, :3]).max()), float(np.abs(out["vel"][:, :3] - rv[:, :3]).max()),
        int((out["ncount"] != ref["ncount"]).sum())))


@pytest.mark.parametrize("idx,frames", [(2, 1000), (3, 400)])
def test_single_step_parity_from_a_late_state(idx, frames, force_variant):
    """Single-step parity not from the initial lattice but from a state deep into the run (config 2 after 1 s of simulated
    time: the dam has broken, run up the far wall and fallen back -- wall clamps, compressed clusters, boids inside the
    fluid): the GPU runs `frames` frames on its own, then one more step is compared with the oracle's step from that same
    state with the single-step tolerances."""
    cfg = W.config(idx)
    with Sim(cfg) as sim:
        pos, vel, bpos, bvel = dev(cfg["pos"]), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"])
        for _ in range(frames):
            B.sph_step(sim.ctx, pos, vel, bpos, bvel, cfg["boid"])
            B.boid_step(sim.ctx, cfg["boid"], bpos, bvel)
        torch.cuda.synchronize()
        p0, v0, bp0, bv0 = (t.cpu().numpy() for t in (pos, vel, bpos, bvel))
        assert np.isfinite(p0).all() and np.isfinite(v0).all() and np.isfinite(bp0).all() and np.isfinite(bv0).all()
        lo, hi = np.array(cfg["sph"]["box_min"], np.float32), np.array(cfg["sph"]["box_max"], np.float32)
        assert (p0[:, :3] >= lo).all() and (p0[:, :3] <= hi).all()
        assert ((p0[:, :3] == lo) | (p0[:, :3] == hi)).any()  # some particles sit on a wall: the clamp is exercised
        ref = R.step(cfg["sph"], p0, v0, bp0, bv0, cfg["boid"])
        out = sim.step(pos, vel, bpos, bvel, cfg["boid"])
        _compare_step(cfg, out, ref, p0)
        assert ref["ncount"].max() > 40  # compressed regions: well above the lattice's ~30 neighbours
        refb = R.boid_step(cfg["sph"], cfg["boid"], p0, v0, ref["density"], bp0, bv0)
        ob = sim.boid_step(cfg["boid"], bpos, bvel)
        bad, worst = vec_err(ob["bvel"][:, :3], refb["bvel"][:, :3])
        assert bad == 0, ("bvel", bad, worst)
        bad, worst = vec_err(ob["bpos"][:, :3], refb["bpos"][:, :3])
        assert bad == 0, ("bpos", bad, worst)
