"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI binding on torch tensors."""
import numpy as np
import torch

from paper_2311_15088_b200 import binding as B


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def u32(n):
    return torch.zeros(n, dtype=torch.int32, device="cuda")


def host_u32(t):
    return t.cpu().numpy().view(np.uint32)


FORCE_VARIANT = None  # set by a test fixture: 1 = stored neighbour list, 2 = brick density + neighbour masks; None = the library's cost model


class Sim:
    """One libsphboid context sized for a workload dict (workloads.config)."""

    def __init__(self, cfg, max_particles=None, G=None):
        self.cfg = cfg
        self.G = G if G is not None else cfg.get("G", 0)
        self.ctx = B.sph_create(cfg["sph"], max_particles or max(cfg["n"], 1), max(cfg.get("n_boid", 0), 1), self.G)
        self.dims, self.C = B.sph_grid_dims(self.ctx)
        if FORCE_VARIANT is not None:
            B.sph_set_force_variant(self.ctx, FORCE_VARIANT)

    def close(self):
        if self.ctx is not None:
            B.sph_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def build_grid(self, pos, vel=None):
        n = pos.shape[0]
        cell, perm, start = u32(max(n, 1)), u32(max(n, 1)), u32(self.C + 1)
        B.sph_build_grid(self.ctx, pos, vel, cell_of_particle=cell, perm=perm, cell_start=start)
        torch.cuda.synchronize()
        return host_u32(cell)[:n], host_u32(perm)[:n], host_u32(start)

    def step(self, pos, vel, bpos=None, bvel=None, boid=None):
        """pos/vel CUDA tensors updated in place.  Returns dict of numpy outputs."""
        n = pos.shape[0]
        rho = torch.zeros(n, device="cuda")
        acc = torch.zeros(n, 4, device="cuda")
        cnt, tch = u32(n), u32(n)
        B.sph_step(self.ctx, pos, vel, bpos, bvel, boid, density=rho, accel=acc, ncount=cnt, touched=tch)
        torch.cuda.synchronize()
        return dict(pos=pos.cpu().numpy(), vel=vel.cpu().numpy(), density=rho.cpu().numpy(), accel=acc.cpu().numpy(),
                    ncount=host_u32(cnt), touched=host_u32(tch))

    def boid_step(self, boid, bpos, bvel):
        nb = bpos.shape[0]
        parts = torch.zeros(nb, 4, 4, device="cuda")
        B.boid_step(self.ctx, boid, bpos, bvel, dv_parts=parts)
        torch.cuda.synchronize()
        return dict(bpos=bpos.cpu().numpy(), bvel=bvel.cpu().numpy(), dv_parts=parts.cpu().numpy())


def vec_err(got, ref, rel=1e-5, abs_=1e-6, scale=None):
    """Per-row vector-norm error: returns (n_bad, worst ratio err/allowed).  allowed = rel*|ref| + abs (or rel*scale+abs)."""
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    if got.ndim == 1:
        got, ref = got[:, None], ref[:, None]
    err = np.linalg.norm(got - ref, axis=1)
    base = np.linalg.norm(ref, axis=1) if scale is None else np.asarray(scale, np.float64)
    allowed = rel * base + abs_
    ratio = err / allowed
    return int((ratio > 1.0).sum()), float(ratio.max()) if ratio.size else 0.0
