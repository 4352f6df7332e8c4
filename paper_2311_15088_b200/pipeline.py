"""One frame of the particle pipeline through the C ABI (include/sphboid.h) -- argument marshalling only.

A frame is the paper's per-frame loop: neighbour structure, SPH density and forces,
integration, boid update with two-way coupling, then the surface pass on the new positions:

    sph_step -> boid_step -> sph_build_grid(pos, vel) -> mc_extract

The grid built on the new positions at the end of frame t serves the surface pass of frame t AND is the
neighbour structure of frame t+1 (same positions): sph_step finds it current and does not rebuild it, so there
is exactly one grid build per frame (the very first sph_step builds its own).

Everything runs in libsphboid's CUDA kernels on the caller's stream; this class only owns the torch tensors
(device memory) and the context.  There is no CPU fallback: without the library or a CUDA device it raises.
"""
import numpy as np

from . import binding as B
from . import workloads as W


class Frame:
    def __init__(self, cfg, device=0, tri_capacity=None, with_mc=True, track_aabb=False):
        """track_aabb: lay the voxel grid over the fluid's bounding box AT EXTRACTION TIME (BASELINE config 4 / 5: 'MC
        256^3 over the fluid bounding box'): after every grid build the box is read back from the device
        (sph_particle_aabb, one small synchronising copy per frame) and origin / spacing follow it.  Off by default:
        the grid then stays where the initial state put it, and a frame enqueues without any host synchronisation."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2311_15088_b200 needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.cfg = cfg
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.n, self.nb = cfg["n"], cfg["n_boid"]
        self.with_mc = with_mc
        self.track_aabb = bool(track_aabb) and with_mc and cfg.get("idx") in (4, 5)
        self.mc = W.mc_params(cfg) if with_mc else None
        self.G = self.mc["n_point_per_axis"] if with_mc else 0
        self.ctx = B.sph_create(cfg["sph"], max(self.n, 1), max(self.nb, 1), self.G, device=device)
        self.pos = self._dev(cfg["pos"])
        self.vel = self._dev(cfg["vel"])
        self.bpos = self._dev(cfg["bpos"]) if self.nb else None
        self.bvel = self._dev(cfg["bvel"]) if self.nb else None
        if with_mc:
            # a closed surface around N particles of radius 0.5 h has O(N^(2/3)) cubes; 4 triangles per particle
            # is far above anything the dam-break configs emit and is checked after every run (SPH_E_CAPACITY)
            self.tri_capacity = tri_capacity or max(4 * self.n, 1024)
            self.tris = torch.empty(self.tri_capacity, 3, 3, device=self.device)
        self.n_tris = 0

    def _dev(self, a):
        return self.torch.from_numpy(np.ascontiguousarray(a)).to(self.device)

    def sim(self):
        """S6-S13 then S1-S5 on the new state: SPH step, boid step (in place), grid for what follows."""
        B.sph_step(self.ctx, self.pos, self.vel, self.bpos, self.bvel, self.cfg["boid"])
        if self.nb:
            B.boid_step(self.ctx, self.cfg["boid"], self.bpos, self.bvel)
        B.sph_build_grid(self.ctx, self.pos, self.vel)
        if self.track_aabb:
            lo, hi = B.sph_particle_aabb(self.ctx)
            extent = max(np.float32(hi[a]) - np.float32(lo[a]) for a in range(3))
            self.mc = dict(self.mc, origin=tuple(float(x) for x in lo), spacing=float(np.float32(extent / (self.G - 1))))

    def surface(self, sync=False):
        """S14-S17 on the current grid.  Returns the triangle count when sync."""
        nt = B.mc_extract(self.ctx, self.mc, self.tris, sync=sync)
        if sync:
            self.n_tris = nt
        return nt

    def surface_async(self):
        """S14-S17 of this frame beside the next frame's SPH step (mc_extract_async); pair with wait()."""
        B.mc_extract_async(self.ctx, self.mc, self.tris)

    def wait(self, sync=False):
        nt = B.mc_wait(self.ctx, sync=sync)
        if sync:
            self.n_tris = nt
        return nt

    def capture(self, frames=1, pipelined=False):
        """Capture `frames` whole frames into a CUDA graph; replay() then runs them with one launch.  The library keeps
        no per-launch state on the host (scan epochs, work counters and the bounding box live in device memory), and
        the state of the context after a frame equals the state before it, so the captured sequence is valid for
        every later frame.  pipelined: inside the graph the surface pass of a frame is forked (mc_extract_async) and
        runs beside the next frame's SPH step; the last one is joined before the graph ends.  The frame just before
        the capture runs eagerly."""
        torch = self.torch
        self.frame()
        torch.cuda.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        self.graph_frames = frames
        with torch.cuda.graph(self.graph):
            for _ in range(frames):
                self.sim()
                if pipelined:
                    self.surface_async()
                else:
                    self.surface()
            if pipelined:
                self.wait()
        return self.graph

    def replay(self):
        self.graph.replay()

    def frame(self, sync=False):
        self.sim()
        if self.with_mc:
            return self.surface(sync=sync)
        return None

    def close(self):
        if self.ctx is not None:
            B.sph_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
