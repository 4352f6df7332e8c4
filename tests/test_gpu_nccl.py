"""N2 over NCCL: two ranks, one GPU each, exchanging halos and migrants through DistExchange.  Skipped below two
devices (this pool's boxes have one); it exists so that the first multi-GPU run is not the first time the exchange
meets NCCL.  The decomposed frames are compared with the undecomposed GPU run particle by particle."""
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu

_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch
import torch.distributed as dist
from paper_2311_15088_b200 import slab as S, workloads as W
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(rank)
dist.init_process_group("nccl", rank=rank, world_size=world)
cfg = W.config(2)
pos = cfg["pos"].copy(); pos[:, 3] = np.arange(cfg["n"], dtype=np.float32)   # id rides in the payload lane
lay = S.SlabLayout(cfg["sph"], world, boid=cfg["boid"], pos=pos)
p, v = S.split_initial(lay, pos, cfg["vel"])[rank]
bp, bv = S.split_initial(lay, cfg["bpos"], cfg["bvel"])[rank]
be = S.GpuBackend(cfg["sph"], cfg["n"], device=rank, boid_capacity=cfg["n_boid"])
ex = S.DistExchange(dist, rank, world, torch.device("cuda", rank), capacity=cfg["n"])
sim = S.SlabSim(lay, rank, be, ex, be.to_device(p), be.to_device(v), be.to_device(bp), be.to_device(bv), cfg["boid"])
for _ in range(5):
    sim.step()
torch.cuda.synchronize()
np.save({out!r} % rank, np.concatenate([sim.pos.cpu().numpy(), sim.vel.cpu().numpy()], 1))
dist.barrier()
dist.destroy_process_group()
be.close()
print("rank", rank, "ok", sim.n_owned)
"""


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices")
def test_decomposed_frames_over_nccl_world_size_2(tmp_path):
    from paper_2311_15088_b200 import binding as B
    from paper_2311_15088_b200 import workloads as W
    from tests.gpuutil import Sim, dev, vec_err
    script = tmp_path / "worker.py"
    out_pat = str(tmp_path / "rank%d.npy")
    script.write_text(_WORKER.format(root=ROOT, out=out_pat))
    port = 29700 + os.getpid() % 200
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for rank, p in enumerate(procs):
        out, _ = p.communicate(timeout=600)
        assert p.returncode == 0, out
    cfg = W.config(2)
    with Sim(cfg) as sim:
        pos, vel, bpos, bvel = dev(cfg["pos"]), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"])
        for _ in range(5):
            B.sph_step(sim.ctx, pos, vel, bpos, bvel, cfg["boid"])
            B.boid_step(sim.ctx, cfg["boid"], bpos, bvel)
        torch.cuda.synchronize()
        ref_p, ref_v = pos.cpu().numpy(), vel.cpu().numpy()
    got = np.concatenate([np.load(out_pat % r) for r in range(2)], 0)
    ids = got[:, 3].astype(np.int64)
    assert np.array_equal(np.sort(ids), np.arange(cfg["n"]))
    gp, gv = np.zeros_like(ref_p), np.zeros_like(ref_v)
    gp[ids], gv[ids] = got[:, :4], got[:, 4:]
    bad, worst = vec_err(gp[:, :3], ref_p[:, :3], rel=5e-5, abs_=1e-5)
    assert bad == 0, ("pos", bad, worst)
    bad, worst = vec_err(gv[:, :3], ref_v[:, :3], rel=5e-5, abs_=1e-4)
    assert bad == 0, ("vel", bad, worst)
