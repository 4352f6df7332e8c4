"""The end-to-end entry point with HOST buffers (sph_simulate_host, what bench.py's `e2e` times) against the oracle."""
import numpy as np
import pytest
import torch

from oracle import refbind as R
from paper_2311_15088_b200 import binding as B
from paper_2311_15088_b200 import workloads as W
from tests.gpuutil import Sim, vec_err

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("pinned", [True, False])
def test_simulate_host_one_frame_matches_oracle(pinned):
    cfg = W.config(1)
    mp = W.mc_params(cfg)
    G, h = mp["n_point_per_axis"], cfg["sph"]["h"]
    ref = R.step(cfg["sph"], cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"], cfg["boid"])
    refb = R.boid_step(cfg["sph"], cfg["boid"], cfg["pos"], cfg["vel"], ref["density"], cfg["bpos"], cfg["bvel"])
    phi_ref = R.voxel_sdf(cfg["sph"], mp, ref["pos"])
    _, nt_ref, _ = R.mc_polygonise(mp, phi_ref)

    def host(a):
        t = torch.from_numpy(np.ascontiguousarray(a).copy())
        return t.pin_memory() if pinned else t

    pos, vel, bpos, bvel = host(cfg["pos"]), host(cfg["vel"]), host(cfg["bpos"]), host(cfg["bvel"])
    tris = torch.zeros(nt_ref + 64, 3, 3)
    if pinned:
        tris = tris.pin_memory()
    with Sim(cfg, G=G) as sim:
        nt = B.sph_simulate_host(sim.ctx, pos, vel, bpos, bvel, cfg["boid"], 1, mp, tris)
        for got, want, what in ((pos, ref["pos"], "pos"), (vel, ref["vel"], "vel"), (bpos, refb["bpos"], "bpos"),
                                (bvel, refb["bvel"], "bvel")):
            bad, worst = vec_err(got.numpy()[:, :3], want[:, :3])
            assert bad == 0, (what, bad, worst)
        # the mesh is that of the GPU's own phi on the new positions: same count as the device path, and as the oracle's
        # unless a corner sits within the phi tolerance of iso
        risky = int((np.abs(phi_ref - mp["iso"]) <= 1e-5 * h).sum())
        assert abs(nt - nt_ref) <= 5 * 8 * risky and nt > 0
        buf = torch.zeros(nt + 64, 3, 3, device="cuda")
        B.sph_build_grid(sim.ctx, pos.cuda())
        assert B.mc_extract(sim.ctx, mp, buf) == nt
        assert np.array_equal(buf.cpu().numpy()[:nt], tris.numpy()[:nt])
        # capacity too small: the required count still comes back
        small = torch.zeros(max(nt // 4, 1), 3, 3)
        pos2, vel2 = host(cfg["pos"]), host(cfg["vel"])
        nt2 = B.sph_simulate_host(sim.ctx, pos2, vel2, host(cfg["bpos"]), host(cfg["bvel"]), cfg["boid"], 1, mp, small)
        assert nt2 == nt and np.array_equal(pos2.numpy(), pos.numpy())


def test_async_surface_pass_is_bitwise_the_synchronous_one():
    # three frames: (a) sph_step, boid_step, build_grid, mc_extract in stream order; (b) the same with the surface pass
    # forked by mc_extract_async and running beside the NEXT frame's SPH step.  State and meshes must be identical bit
    # for bit, frame by frame (the library orders the next grid build after the pending pass)
    from paper_2311_15088_b200.pipeline import Frame
    cfg = W.config(2, scale=2)
    meshes = []
    with Frame(cfg) as fa:
        for _ in range(3):
            fa.sim()
            nt = fa.surface(sync=True)
            meshes.append((nt, fa.tris[:nt].cpu().numpy().copy(), fa.pos.cpu().numpy().copy()))
    with Frame(cfg) as fb:
        bufs = [torch.zeros_like(fb.tris) for _ in range(3)]
        counts, states = [], []
        for t in range(3):
            fb.sim()
            if t > 0:
                counts.append(fb.wait(sync=True))  # frame t-1's mesh: its pass overlapped this frame's sph_step
            fb.tris = bufs[t]
            fb.surface_async()
            states.append(fb.pos.clone())
        counts.append(fb.wait(sync=True))
        torch.cuda.synchronize()
        for t in range(3):
            nt, tris, pos = meshes[t]
            assert counts[t] == nt and nt > 0
            assert np.array_equal(bufs[t][:nt].cpu().numpy(), tris)
            assert np.array_equal(states[t].cpu().numpy(), pos)
        with pytest.raises(B.SphError):
            B.mc_wait(fb.ctx)  # nothing pending any more


def test_cuda_graph_replay_is_bitwise_the_eager_frame():
    # a frame captured once into a CUDA graph and replayed: state and mesh identical, bit for bit, to eager frames
    # (the library keeps no per-launch host state: scan epochs, work counters and the bounding box live on the device)
    from paper_2311_15088_b200.pipeline import Frame
    cfg = W.config(2, scale=2)
    eager = []
    with Frame(cfg) as fa:
        for _ in range(5):
            fa.sim()
            nt = fa.surface(sync=True)
            eager.append((nt, fa.tris[:nt].cpu().numpy().copy(), fa.pos.cpu().numpy().copy(), fa.bpos.cpu().numpy().copy()))
    with Frame(cfg) as fb:
        fb.capture()  # runs frame 1 eagerly, then captures (the capture itself does not execute)
        for t in range(1, 5):
            fb.replay()
            torch.cuda.synchronize()
            nt = int(B.mc_extract(fb.ctx, fb.mc, torch.zeros_like(fb.tris)))  # count of the same state, eagerly
            want_nt, want_tris, want_pos, want_bpos = eager[t]
            assert nt == want_nt
            assert np.array_equal(fb.tris[:nt].cpu().numpy(), want_tris)
            assert np.array_equal(fb.pos.cpu().numpy(), want_pos) and np.array_equal(fb.bpos.cpu().numpy(), want_bpos)


def test_cuda_graph_of_pipelined_frames_matches_eager():
    # three frames per graph, inside it every surface pass forked beside the next frame's SPH step: after each replay
    # the state and the mesh are those of the eager frames 3, 6, ... (frame 1 runs eagerly before the capture... so 4, 7)
    from paper_2311_15088_b200.pipeline import Frame
    cfg = W.config(2, scale=2)
    eager = []
    with Frame(cfg) as fa:
        for _ in range(7):
            fa.sim()
            nt = fa.surface(sync=True)
            eager.append((nt, fa.tris[:nt].cpu().numpy().copy(), fa.pos.cpu().numpy().copy()))
    with Frame(cfg) as fb:
        fb.capture(frames=3, pipelined=True)  # eager frame 1, then frames 2-4 per replay
        for rep in range(2):
            fb.replay()
            torch.cuda.synchronize()
            want_nt, want_tris, want_pos = eager[3 * (rep + 1)]
            assert np.array_equal(fb.pos.cpu().numpy(), want_pos)
            assert np.array_equal(fb.tris[:want_nt].cpu().numpy(), want_tris)


@pytest.mark.parametrize("pinned", [True, False])
def test_simulate_host_three_steps_is_bitwise_the_device_path(pinned):
    # sph_simulate_host uploads the velocities beside the first step's grid build and density pass (k_gather_vel
    # completes the sorted copy afterwards): the state after three steps must be bit for bit what the device-resident
    # calls give, with pinned and with pageable host buffers
    from paper_2311_15088_b200.pipeline import Frame
    cfg = W.config(2, scale=2)
    with Frame(cfg) as fr:
        for _ in range(3):
            fr.sim()
        want = [t.cpu().numpy().copy() for t in (fr.pos, fr.vel, fr.bpos, fr.bvel)]

    def host(a):
        t = torch.from_numpy(np.ascontiguousarray(a).copy())
        return t.pin_memory() if pinned else t

    got = [host(cfg[k]) for k in ("pos", "vel", "bpos", "bvel")]
    with Sim(cfg, G=0) as sim:
        B.sph_simulate_host(sim.ctx, got[0], got[1], got[2], got[3], cfg["boid"], 3, None, None)
        for g, w, what in zip(got, want, ("pos", "vel", "bpos", "bvel")):
            assert np.array_equal(g.numpy(), w), what
        # zero steps: the state makes the round trip unchanged
        again = [host(cfg[k]) for k in ("pos", "vel", "bpos", "bvel")]
        B.sph_simulate_host(sim.ctx, again[0], again[1], again[2], again[3], cfg["boid"], 0, None, None)
        for g, k in zip(again, ("pos", "vel", "bpos", "bvel")):
            assert np.array_equal(g.numpy(), np.ascontiguousarray(cfg[k]))


def test_particle_aabb_is_exact_and_frame_can_follow_it():
    """sph_particle_aabb returns the exact binary32 bounding box of the particles the grid was built on, and
    Frame(track_aabb=True) lays config 4's voxel grid over the fluid box at extraction time (workloads.mc_params on the
    current positions), not over the initial one."""
    import numpy as np
    import torch
    from paper_2311_15088_b200 import binding as B
    from paper_2311_15088_b200 import workloads as W
    from paper_2311_15088_b200.pipeline import Frame
    cfg = W.config(4, scale=4)
    with Frame(cfg, track_aabb=True) as fr:
        with pytest.raises(B.SphError) as e:
            B.sph_particle_aabb(fr.ctx)
        assert e.value.code == B.SPH_E_STALE_GRID
        for _ in range(30):
            fr.frame()
        torch.cuda.synchronize()
        p = fr.pos.cpu().numpy()
        lo, hi = B.sph_particle_aabb(fr.ctx)
        assert np.array_equal(np.float32(lo), p[:, :3].min(axis=0)) and np.array_equal(np.float32(hi), p[:, :3].max(axis=0))
        want = W.mc_params(cfg, p)
        assert fr.mc["origin"] == want["origin"] and fr.mc["spacing"] == want["spacing"]
        assert fr.mc["origin"] != W.mc_params(cfg)["origin"] or fr.mc["spacing"] != W.mc_params(cfg)["spacing"]
