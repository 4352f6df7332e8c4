"""N2 on the GPU: the ordered range selection (sph_pack_range) bit-exact against a numpy mask, and the slab-decomposed
SPH step -- several ranks emulated one after the other in ONE process on one GPU (LoopbackExchange) -- against the
undecomposed oracle, particle by particle (ids ride in pos.w)."""
import numpy as np
import pytest
import torch

from oracle import refbind as R
from paper_2311_15088_b200 import binding as B
from paper_2311_15088_b200 import slab as S
from paper_2311_15088_b200 import workloads as W
from tests.gpuutil import Sim, dev, vec_err
from tests.slabutil import gather_by_id, tagged_state

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n", [1, 255, 256, 257, 70001])
def test_pack_range_is_the_ordered_mask(n):
    rng = np.random.default_rng(n)
    pos = rng.uniform(-1, 2, (n, 4)).astype(np.float32)
    vel = rng.uniform(-1, 1, (n, 4)).astype(np.float32)
    with Sim(dict(sph=W.config(1)["sph"], n=n)) as sim:
        dp, dv = dev(pos), dev(vel)
        for axis, lo, hi in ((0, 0.25, 1.5), (1, -np.inf, 0.5), (2, 0.5, np.inf), (0, 5.0, 6.0)):
            want = (pos[:, axis] >= np.float32(lo)) & (pos[:, axis] < np.float32(hi))
            op, ov = torch.full((n + 3, 4), -7.0, device="cuda"), torch.full((n + 3, 4), -7.0, device="cuda")
            k = B.sph_pack_range(sim.ctx, dp, dv, n, axis, lo, hi, op, ov)
            assert k == int(want.sum())
            assert np.array_equal(op.cpu().numpy()[:k], pos[want]) and np.array_equal(ov.cpu().numpy()[:k], vel[want])
            assert bool((op[k:] == -7.0).all())
        # only the first m particles; too small a buffer
        m = max(n // 2, 1)
        want = pos[:m, 0] >= np.float32(0.0)
        op, ov = torch.zeros(n, 4, device="cuda"), torch.zeros(n, 4, device="cuda")
        assert B.sph_pack_range(sim.ctx, dp, dv, m, 0, 0.0, np.inf, op, ov) == int(want.sum())
        if want.sum() > 1:
            with pytest.raises(B.SphError) as e:
                B.sph_pack_range(sim.ctx, dp, dv, m, 0, 0.0, np.inf, op[:1], ov[:1])
            assert e.value.code == B.SPH_E_CAPACITY


@pytest.mark.parametrize("idx,scale,world", [(1, None, 2), (2, None, 3), (3, 2, 4)])
def test_slab_decomposed_steps_match_undecomposed_oracle(idx, scale, world):
    cfg = W.config(idx, scale=scale)
    pos, vel = tagged_state(cfg, speed=8.0)
    n, steps = cfg["n"], 3
    lay = S.SlabLayout(cfg["sph"], world)
    ex = S.LoopbackExchange(world)
    backends = [S.GpuBackend(cfg["sph"], n) for _ in range(world)]
    try:
        sims = [S.SlabSim(lay, r, backends[r], ex, backends[r].to_device(p), backends[r].to_device(v))
                for r, (p, v) in enumerate(S.split_initial(lay, pos, vel))]
        rp, rv = pos, vel
        moved = 0
        for s in range(1, steps + 1):
            S.run_loopback(sims, 1)
            o = R.step(cfg["sph"], rp, rv)
            rp, rv = o["pos"], o["vel"]
            moved += sum(x.stats["migrated_out"] for x in sims)
            gp, gv = gather_by_id([(x.pos.cpu().numpy(), x.vel.cpu().numpy()) for x in sims], n)
            # free-running comparison, the bound of test_free_running_ten_steps (D:A-MULTI (ii))
            bad, worst = vec_err(gp[:, :3], rp[:, :3], rel=1e-5 * s, abs_=2e-6 * s)
            assert bad <= n // 10000, ("pos", s, bad, worst)
            bad, worst = vec_err(gv[:, :3], rv[:, :3], rel=1e-5 * s, abs_=2e-5 * s)
            assert bad <= n // 10000, ("vel", s, bad, worst)
            for x in sims:
                xs = x.pos[:, lay.axis]
                assert bool(((xs >= x.lo) & (xs < x.hi)).all())
        assert moved > 0 and sum(x.stats["ghosts"] for x in sims) > 0
        # against the undecomposed GPU run as well: same kernels, same neighbour sets -> same tolerance, tighter in practice
        with Sim(cfg) as one:
            dp, dv = dev(pos), dev(vel)
            for _ in range(steps):
                B.sph_step(one.ctx, dp, dv)
            bad, worst = vec_err(gp[:, :3], dp.cpu().numpy()[:, :3], rel=1e-5 * steps, abs_=2e-6 * steps)
            assert bad <= n // 10000, ("pos vs one GPU", bad, worst)
    finally:
        for b in backends:
            b.close()


@pytest.mark.parametrize("idx,scale,world", [(1, None, 3), (2, None, 3), (2, None, 4)])
def test_slab_decomposed_frames_with_boids_match_undecomposed_oracle(idx, scale, world):
    # fluid and boids both cut into slabs (ghost boids; fluid halo push radius + h): sph_step + boid_step per emulated
    # rank, against the undecomposed oracle frames, particle by particle and boid by boid
    from tests.slabutil import reference_frames, tagged_boids
    cfg = W.config(idx, scale=scale)
    pos, vel = tagged_state(cfg, speed=8.0)
    bpos, bvel, boid = tagged_boids(cfg)
    n, nb, steps = cfg["n"], cfg["n_boid"], 3
    lay = S.SlabLayout(cfg["sph"], world, boid=boid)
    ex = S.LoopbackExchange(world)
    backends = [S.GpuBackend(cfg["sph"], n, boid_capacity=nb) for _ in range(world)]
    try:
        fluid, boids = S.split_initial(lay, pos, vel), S.split_initial(lay, bpos, bvel)
        sims = [S.SlabSim(lay, r, backends[r], ex, backends[r].to_device(fluid[r][0]), backends[r].to_device(fluid[r][1]),
                          backends[r].to_device(boids[r][0]), backends[r].to_device(boids[r][1]), boid)
                for r in range(world)]
        moved = ghosts = 0
        for s in range(steps):
            S.run_loopback(sims, 1)
            moved += sum(x.stats["boids_migrated_out"] for x in sims)
            ghosts += sum(x.stats["boid_ghosts"] for x in sims)
            for x in sims:
                xs = x.bpos[:, lay.axis]
                assert bool(((xs >= x.lo) & (xs < x.hi)).all())
        assert moved > 0 and ghosts > 0
        rp, rv, rbp, rbv = reference_frames(cfg, pos, vel, bpos, bvel, boid, steps)
        gp, gv = gather_by_id([(x.pos.cpu().numpy(), x.vel.cpu().numpy()) for x in sims], n)
        gbp, gbv = gather_by_id([(x.bpos.cpu().numpy(), x.bvel.cpu().numpy()) for x in sims], nb)
        for got, want, what, abs_ in ((gp, rp, "pos", 2e-6), (gv, rv, "vel", 2e-5), (gbp, rbp, "bpos", 2e-6),
                                      (gbv, rbv, "bvel", 1e-4)):
            bad, worst = vec_err(got[:, :3], want[:, :3], rel=1e-5 * steps, abs_=abs_ * steps)
            assert bad <= got.shape[0] // 10000, (what, bad, worst)
    finally:
        for b in backends:
            b.close()


@pytest.mark.parametrize("idx,scale,world", [(1, None, 3), (2, None, 2), (3, 2, 4)])
def test_slab_decomposed_surface_matches_the_undecomposed_pass(idx, scale, world):
    # every emulated rank polygonises the cubes of its slab (mc_set_cube_range) from [owned | ghost] particles; against
    # (a) the same cube range polygonised by ONE context that holds all particles (same kernels; phi differs only by
    # the order of the binary32 sums) and (b) the oracle's mesh of the gathered state, restricted to the rank's cubes
    from tests.slabutil import triangles_in_cube_range
    cfg = W.config(idx, scale=scale)
    mc = W.mc_params(cfg)
    G, h = mc["n_point_per_axis"], cfg["sph"]["h"]
    pos, vel = tagged_state(cfg, speed=8.0)
    n = cfg["n"]
    lay = S.SlabLayout(cfg["sph"], world, mc=mc)
    ex = S.LoopbackExchange(world)
    backends = [S.GpuBackend(cfg["sph"], n, mc_points=G) for _ in range(world)]
    try:
        sims = [S.SlabSim(lay, r, backends[r], ex, backends[r].to_device(p), backends[r].to_device(v))
                for r, (p, v) in enumerate(S.split_initial(lay, pos, vel))]
        bufs = [torch.zeros(300000, 3, 3, device="cuda") for _ in range(world)]
        S.run_loopback(sims, 2)
        state, svel = gather_by_id([(x.pos.cpu().numpy(), x.vel.cpu().numpy()) for x in sims], n)
        counts = S.run_loopback(sims, 1, tris=bufs)
        phi_ref = R.voxel_sdf(cfg["sph"], mc, state)
        t_ref, nt_ref, cases = R.mc_polygonise(mc, phi_ref, want_cases=True)
        risky = int((np.abs(phi_ref - mc["iso"]) <= 1e-5 * h).sum())
        assert abs(sum(counts) - nt_ref) <= 5 * 8 * risky and sum(counts) > 0
        with Sim(cfg, G=G) as one:
            B.sph_build_grid(one.ctx, dev(state))
            whole = torch.zeros(300000, 3, 3, device="cuda")
            for r in range(world):
                i0, i1 = lay.cube_range(r)
                B.mc_set_cube_range(one.ctx, lay.axis, i0, i1)
                nt = B.mc_extract(one.ctx, mc, whole)
                assert abs(nt - counts[r]) <= 5 * 8 * risky
                keep = triangles_in_cube_range(mc, cases, lay.axis, i0, i1)
                assert abs(int(keep.sum()) - counts[r]) <= 5 * 8 * risky
                if nt == counts[r] and nt > 0:
                    d = (whole[:nt] - bufs[r][:nt]).abs().flatten().cpu().numpy()
                    assert np.quantile(d, 0.999) <= 1e-3 * mc["spacing"], (r, float(d.max()))
                if int(keep.sum()) == counts[r] and counts[r] > 0:
                    d = np.abs(bufs[r][:counts[r]].cpu().numpy() - t_ref[keep]).ravel()
                    assert np.quantile(d, 0.999) <= 1e-3 * mc["spacing"], (r, float(d.max()))
        assert sum(c > 0 for c in counts) >= 2
    finally:
        for b in backends:
            b.close()


def test_balanced_slabs_config4_over_8_emulated_ranks():
    """N2 with faces cut by particle count (SlabLayout(pos=...)): config 4 over 8 ranks emulated one after the other on
    one GPU; the owned-particle imbalance (max / mean) is printed and stays within 10 % over the frames, and the
    decomposed frames match the undecomposed GPU run particle by particle."""
    cfg = W.config(4)
    world, steps, n = 8, 3, cfg["n"]
    pos = cfg["pos"].copy()
    pos[:, 3] = np.arange(n, dtype=np.float32)
    lay = S.SlabLayout(cfg["sph"], world, boid=cfg["boid"], pos=pos)
    ex = S.LoopbackExchange(world)
    cap = n // world + n // 16
    backends = [S.GpuBackend(cfg["sph"], cap, boid_capacity=cfg["n_boid"]) for _ in range(world)]
    try:
        parts, bparts = S.split_initial(lay, pos, cfg["vel"]), S.split_initial(lay, cfg["bpos"], cfg["bvel"])
        sims = [S.SlabSim(lay, r, backends[r], ex, backends[r].to_device(parts[r][0]), backends[r].to_device(parts[r][1]),
                          backends[r].to_device(bparts[r][0]), backends[r].to_device(bparts[r][1]), cfg["boid"])
                for r in range(world)]
        for s in range(steps):
            S.run_loopback(sims, 1)
            owned = np.array([x.n_owned for x in sims])
            print("frame %d: owned per rank %s, imbalance max/mean %.3f, ghosts max %d" % (
                s + 1, owned.tolist(), owned.max() / owned.mean(), max(x.stats["ghosts"] for x in sims)))
            assert owned.sum() == n and owned.max() / owned.mean() <= 1.10
        got = np.concatenate([np.concatenate([x.pos.cpu().numpy(), x.vel.cpu().numpy()], 1) for x in sims], 0)
    finally:
        for b in backends:
            b.close()
    with Sim(cfg) as one:
        dp, dv, dbp, dbv = dev(pos), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"])
        for _ in range(steps):
            B.sph_step(one.ctx, dp, dv, dbp, dbv, cfg["boid"])
            B.boid_step(one.ctx, cfg["boid"], dbp, dbv)
        ref_p, ref_v = dp.cpu().numpy(), dv.cpu().numpy()
    ids = got[:, 3].astype(np.int64)
    assert np.array_equal(np.sort(ids), np.arange(n))
    gp, gv = np.zeros_like(ref_p), np.zeros_like(ref_v)
    gp[ids], gv[ids] = got[:, :4], got[:, 4:]
    bad, worst = vec_err(gp[:, :3], ref_p[:, :3], rel=1e-5 * steps, abs_=2e-6 * steps)
    assert bad <= n // 10000, ("pos", bad, worst)
    bad, worst = vec_err(gv[:, :3], ref_v[:, :3], rel=1e-5 * steps, abs_=2e-5 * steps)
    assert bad <= n // 10000, ("vel", bad, worst)


def test_recut_on_the_gpu_backend_balances_and_keeps_parity():
    """N2 re-cut with the library as the stepper: config 2 over 4 emulated ranks from UNIFORM slabs (the fluid fills half
    of the box: two ranks own nothing), one frame, a re-cut from the global column histogram (multi-hop migration), two
    more frames; owned counts balance and the result matches the undecomposed GPU run."""
    cfg = W.config(2)
    world, n = 4, cfg["n"]
    pos = cfg["pos"].copy()
    pos[:, 3] = np.arange(n, dtype=np.float32)
    lay = S.SlabLayout(cfg["sph"], world, boid=cfg["boid"])
    ex = S.LoopbackExchange(world)
    backends = [S.GpuBackend(cfg["sph"], n, boid_capacity=cfg["n_boid"]) for _ in range(world)]
    try:
        parts, bparts = S.split_initial(lay, pos, cfg["vel"]), S.split_initial(lay, cfg["bpos"], cfg["bvel"])
        sims = [S.SlabSim(lay, r, backends[r], ex, backends[r].to_device(parts[r][0]), backends[r].to_device(parts[r][1]),
                          backends[r].to_device(bparts[r][0]), backends[r].to_device(bparts[r][1]), cfg["boid"])
                for r in range(world)]
        before = np.array([s.n_owned for s in sims])
        assert before.max() / before.mean() > 1.9
        S.run_loopback(sims, 1)
        S.run_recut(sims)
        after = np.array([s.n_owned for s in sims])
        print("owned before", before.tolist(), "after", after.tolist(), "cuts", lay.cuts)
        assert after.sum() == n and after.max() / after.mean() <= 1.10
        assert sum(s.nb_owned for s in sims) == cfg["n_boid"]
        S.run_loopback(sims, 2)
        got = np.concatenate([np.concatenate([x.pos.cpu().numpy(), x.vel.cpu().numpy()], 1) for x in sims], 0)
    finally:
        for b in backends:
            b.close()
    with Sim(cfg) as one:
        dp, dv, dbp, dbv = dev(pos), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"])
        for _ in range(3):
            B.sph_step(one.ctx, dp, dv, dbp, dbv, cfg["boid"])
            B.boid_step(one.ctx, cfg["boid"], dbp, dbv)
        ref_p, ref_v = dp.cpu().numpy(), dv.cpu().numpy()
    ids = got[:, 3].astype(np.int64)
    assert np.array_equal(np.sort(ids), np.arange(n))
    gp, gv = np.zeros_like(ref_p), np.zeros_like(ref_v)
    gp[ids], gv[ids] = got[:, :4], got[:, 4:]
    bad, worst = vec_err(gp[:, :3], ref_p[:, :3], rel=3e-5, abs_=6e-6)
    assert bad <= n // 10000, ("pos", bad, worst)
    bad, worst = vec_err(gv[:, :3], ref_v[:, :3], rel=3e-5, abs_=6e-5)
    assert bad <= n // 10000, ("vel", bad, worst)
