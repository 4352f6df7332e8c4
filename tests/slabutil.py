"""Test-only backend for paper_2311_15088_b200.slab: selection in numpy, the step on the CPU oracle (CPU tensors).

It lets the decomposition logic (who owns what, what travels as a ghost, who migrates) be exercised end to end on the
CPU -- under torch.distributed / gloo with one process per rank -- against the undecomposed oracle step."""
import numpy as np
import torch

from oracle import refbind as R


class OracleBackend:
    def __init__(self, sph):
        self.sph = sph

    def to_device(self, a):
        return torch.from_numpy(np.ascontiguousarray(a, np.float32).copy())

    def empty(self):
        return torch.empty(0, 4)

    def pack(self, pos, vel, n, axis, lo, hi):
        if n == 0:
            return self.empty(), self.empty()
        x = pos[:n, axis].numpy()
        sel = torch.from_numpy((x >= np.float32(lo)) & (x < np.float32(hi)))
        return pos[:n][sel].clone(), vel[:n][sel].clone()

    def column_hist(self, pos, n, axis, origin, h, dim):
        x = pos[:n, axis].numpy()
        col = np.clip(np.floor((x - np.float32(origin)) / np.float32(h)).astype(np.int64), 0, dim - 1)
        return np.bincount(col, minlength=dim)

    def step(self, pos, vel, bpos=None, bvel=None, boid=None):
        if bpos is None or bpos.shape[0] == 0:
            out = R.step(self.sph, pos.numpy(), vel.numpy())
        else:
            p0, v0 = pos.numpy().copy(), vel.numpy().copy()
            out = R.step(self.sph, p0, v0, bpos.numpy(), bvel.numpy(), boid)
            ob = R.boid_step(self.sph, boid, p0, v0, out["density"], bpos.numpy(), bvel.numpy())
            bpos.copy_(torch.from_numpy(ob["bpos"]))
            bvel.copy_(torch.from_numpy(ob["bvel"]))
        pos.copy_(torch.from_numpy(out["pos"]))
        vel.copy_(torch.from_numpy(out["vel"]))

    def surface(self, pos, vel, mc, axis, lo, hi, tris):
        phi = R.voxel_sdf(self.sph, mc, pos.numpy())
        t, nt, cases = R.mc_polygonise(mc, phi, want_cases=True)
        keep = triangles_in_cube_range(mc, cases, axis, lo, hi)
        k = int(keep.sum())
        tris[:k] = torch.from_numpy(t[keep])
        return k

    def cat(self, parts):
        return torch.cat(parts, 0) if len(parts) > 1 else parts[0].clone()

    def close(self):
        pass


def tagged_state(cfg, seed=5, speed=6.0):
    """Config state with the particle id in pos.w (carried through by the step) and velocities that make particles
    cross slab faces within a few steps."""
    from paper_2311_15088_b200 import workloads as W
    pos = cfg["pos"].copy()
    pos[:, 3] = np.arange(cfg["n"], dtype=np.float32)
    vel = W.uniform_box(cfg["n"], (-speed,) * 3, (speed,) * 3, seed, 30)
    return pos, vel


def gather_by_id(parts, n):
    """parts: list of (pos, vel) numpy arrays of the ranks -> (pos, vel) in id order; checks ids are a permutation."""
    pos = np.concatenate([p for p, _ in parts], 0)
    vel = np.concatenate([v for _, v in parts], 0)
    ids = pos[:, 3].astype(np.int64)
    assert ids.shape[0] == n and np.array_equal(np.sort(ids), np.arange(n)), "particles lost or duplicated"
    order = np.argsort(ids)
    return pos[order], vel[order]


def tagged_boids(cfg, seed=9, speed=25.0):
    """Boids of the config with the boid id in bpos.w (carried through by boid_step), velocities and a speed cap that
    carry boids across slab faces within a few steps.  Returns (bpos, bvel, boid params)."""
    from paper_2311_15088_b200 import workloads as W
    nb = cfg["n_boid"]
    bpos = cfg["bpos"].copy()
    bpos[:, 3] = np.arange(nb, dtype=np.float32)
    bvel = W.uniform_box(nb, (-speed,) * 3, (speed,) * 3, seed, 31)
    return bpos, bvel, dict(cfg["boid"], max_speed=2.0 * speed)


def reference_frames(cfg, pos, vel, bpos, bvel, boid, steps):
    """The undecomposed oracle: `steps` frames of step + boid_step.  Returns (pos, vel, bpos, bvel)."""
    for _ in range(steps):
        o = R.step(cfg["sph"], pos, vel, bpos, bvel, boid)
        ob = R.boid_step(cfg["sph"], boid, pos, vel, o["density"], bpos, bvel)
        pos, vel, bpos, bvel = o["pos"], o["vel"], ob["bpos"], ob["bvel"]
    return pos, vel, bpos, bvel


def triangles_in_cube_range(mc, cases, axis, lo, hi):
    """Mask over the oracle's triangle list (cube-major, ntri[case] triangles per cube): cubes with lo <= index < hi."""
    q = int(mc["n_point_per_axis"]) - 1
    _, ntri, _ = R.mc_table()
    cube = np.repeat(np.arange(q ** 3), ntri[cases].astype(np.int64))
    c = (cube % q, (cube // q) % q, cube // (q * q))[axis]
    return (c >= lo) & (c < hi)
