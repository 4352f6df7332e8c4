"""N2 (SURVEY.md sections 8(e), 8(f)): slab decomposition of the SPH step over ranks, one process per GPU.

The paper runs on one GPU and only names a multi-node decomposition as future work; the
scheme here is the standard one for a short-range particle method:

* the box is cut into slabs along its longest axis, at cell boundaries (multiples of h from box_min); rank r owns the
  particles with lo_r <= x < hi_r, the outermost slabs being open towards -inf / +inf (particles clamped onto a wall
  or started outside the box still have an owner);
* every step each rank receives, from its two neighbours, copies of their particles within 2 h of the shared face
  ("ghosts": the force on an owned particle needs rho of its neighbours within h, and the rho of those needs THEIR
  neighbours within another h), runs the unmodified single-GPU step (sph_step through the C ABI) on
  [owned | ghosts], and keeps the first n_owned results -- an owned particle sees exactly the neighbour set of the
  undecomposed run, so its new state is that run's up to the order of the binary64 sums;
* owned particles that crossed a face migrate to the neighbour.

Exchange steps: two neighbour send / receive pairs per step (halo, migration), variable-size; no global collective.
This module is orchestration only: selection and packing run in libsphboid (sph_pack_range), the step is sph_step,
torch.distributed (NCCL on GPUs, gloo in the CPU tests) moves the packed buffers.

Boids are decomposed the same way (optional: pass bpos / bvel / boid): a rank owns the boids inside its slab, receives
ghost boids within max(visible, protect, push radius) of its faces, runs the unmodified sph_step + boid_step on
[owned | ghost] fluid and [owned | ghost] boids, keeps the owned results and lets boids that crossed a face migrate.
With boids the fluid halo is max(2 h, push radius + h): a ghost boid up to the push radius beyond the face pushes owned
fluid and needs its own probe density (fluid within h of it), and a ghost particle up to the push radius beyond the
face pushes an owned boid and needs its own density.  Every owned particle and boid then sees exactly the neighbours
of the undecomposed run; no collective is needed.

The surface pass is decomposed by cubes (optional: pass mc to the layout): the voxel grid is the global one on every
rank; a rank polygonises the cubes whose lower corner lies in its slab (mc_set_cube_range) from [owned | ghost]
particles, which requires a fluid halo of R + one voxel spacing (the upper corners of its last cubes lie up to one
spacing beyond the face, and phi there needs the particles within R).  The ranks' triangle lists add up to the mesh of
the undecomposed run (each is that mesh's ordered subset for the rank's cubes); an all-gather of the counts would give
output offsets where one buffer is wanted.

The exchange is pluggable (`Exchange`): `DistExchange` uses torch.distributed; `LoopbackExchange` connects several
domains inside ONE process (the single-GPU emulation the GPU test uses: ranks run one after the other, never
concurrently waiting on each other).
"""
import math

import numpy as np


class SlabLayout:
    """Which rank owns which x-range (pure host logic, no device)."""

    def __init__(self, sph, world, axis=None, boid=None, mc=None, pos=None):
        """pos (optional, (n, >=3) host array): cut the faces by PARTICLE count instead of uniformly in cells -- the
        cell-column histogram along the slab axis (what the grid build's start[] prefix gives on the device) is cut
        into `world` pieces of near-equal population, still at cell boundaries and never narrower than a halo."""
        lo, hi = np.asarray(sph["box_min"], np.float64), np.asarray(sph["box_max"], np.float64)
        self.h = float(sph["h"])
        self.axis = int(np.argmax(hi - lo)) if axis is None else int(axis)
        self.world = int(world)
        self.dim = max(1, int(math.ceil((hi[self.axis] - lo[self.axis]) / self.h)))
        self.cells_per_rank = int(math.ceil(self.dim / self.world))
        self.fluid_halo = 2.0 * self.h
        self.boid_halo = 0.0
        if boid is not None:
            self.fluid_halo = max(2.0 * self.h, float(boid["push_radius"]) + self.h)
            self.boid_halo = max(float(boid["visible_range"]), float(boid["protect_range"]), float(boid["push_radius"]))
        self.mc = mc
        if mc is not None:
            self.fluid_halo = max(self.fluid_halo, float(mc["radius"]) + float(mc["spacing"]))
        self.origin = float(np.float32(lo[self.axis]))
        min_cells = int(math.ceil(max(self.fluid_halo, self.boid_halo) / self.h - 1e-9))
        if pos is None:
            cuts = [self.cells_per_rank * r for r in range(1, self.world)]
        else:
            col = self.column_of(np.asarray(pos)[:, self.axis])
            cuts = self.balanced_cuts(np.bincount(col, minlength=self.dim), self.world, min_cells)
        self.min_cells = min_cells
        self.set_cuts(cuts)

    def set_cuts(self, cuts):
        """Move the faces to these cell indices (a re-cut during a run: SlabSim.recut / run_recut)."""
        widths = np.diff([0] + list(cuts) + [self.dim])
        if self.world > 1 and (len(cuts) != self.world - 1 or (widths < self.min_cells).any()):
            raise ValueError("slabs must be at least one halo wide")
        self.cuts = [int(c) for c in cuts]
        # faces in binary32, the precision positions are compared in
        self.faces = [float(np.float32(self.origin + np.float32(c) * np.float32(self.h))) for c in self.cuts]

    def column_of(self, x):
        """Cell column along the slab axis of coordinate(s) x (numpy), clamped like the grid's cells."""
        x = np.asarray(x, np.float32)
        return np.clip(np.floor((x - np.float32(self.origin)) / np.float32(self.h)).astype(np.int64), 0, self.dim - 1)

    @staticmethod
    def balanced_cuts(hist, world, min_cells):
        """Cell indices of the world - 1 faces: face r goes where the running particle count reaches r / world of the
        total, moved as little as needed so that every slab (the outermost ones too) is >= min_cells cells wide."""
        hist = np.asarray(hist, np.int64)
        dim = hist.shape[0]
        cum = np.concatenate([[0], np.cumsum(hist)])
        total = int(cum[-1])
        cuts = []
        for r in range(1, world):
            c = int(np.searchsorted(cum, total * r / world, side="left"))
            # the nearer of the two cell boundaries around the target count
            if c > 0 and abs(cum[c - 1] - total * r / world) <= abs(cum[min(c, dim)] - total * r / world):
                c -= 1
            lo = (cuts[-1] if cuts else 0) + min_cells
            hi = dim - (world - r) * min_cells
            cuts.append(min(max(c, lo), hi))
        return cuts

    def bounds(self, rank):
        """[lo, hi) of rank's slab; the outermost slabs are open."""
        lo = -math.inf if rank == 0 else self.faces[rank - 1]
        hi = math.inf if rank == self.world - 1 else self.faces[rank]
        return lo, hi

    def owner(self, x):
        """Rank that owns coordinate(s) x (numpy, binary32 comparison)."""
        x = np.asarray(x, np.float32)
        return np.searchsorted(np.asarray(self.faces, np.float32), x, side="right").astype(np.int64)

    def cube_range(self, rank):
        """[i0, i1): the cubes (by index along the slab axis) whose lower corner lies in rank's slab; corner
        coordinates in binary32 as the kernels form them (origin + i * spacing)."""
        mc = self.mc
        q = int(mc["n_point_per_axis"]) - 1
        x = np.float32(mc["origin"][self.axis]) + np.arange(q, dtype=np.float32) * np.float32(mc["spacing"])
        lo, hi = self.bounds(rank)
        return (int(np.searchsorted(x, np.float32(lo), side="left")) if rank > 0 else 0,
                int(np.searchsorted(x, np.float32(hi), side="left")) if rank < self.world - 1 else q)

    def halo_width(self):
        return float(np.float32(self.fluid_halo))

    def boid_halo_width(self):
        return float(np.float32(self.boid_halo))


class LoopbackExchange:
    """Connects the domains of ONE process: a two-phase exchange (everybody posts, then everybody collects), so the
    emulated ranks run one after the other and never wait on each other."""

    def __init__(self, world):
        self.world = world
        self.box = {}

    def post(self, rank, tag, to_left, to_right):
        """to_left / to_right: (pos, vel) tensors or None."""
        if rank > 0 and to_left is not None:
            self.box[(rank - 1, tag, "from_right")] = to_left
        if rank < self.world - 1 and to_right is not None:
            self.box[(rank + 1, tag, "from_left")] = to_right

    def collect(self, rank, tag):
        return self.box.pop((rank, tag, "from_left"), None), self.box.pop((rank, tag, "from_right"), None)

    def post_reduce(self, rank, tag, arr):
        """Sum of int64 arrays over the ranks (the re-cut's column histogram, its 'anybody still moving' count)."""
        self.box.setdefault(("sum", tag), []).append(np.asarray(arr, np.int64))

    def collect_reduce(self, rank, tag):
        parts = self.box[("sum", tag)]
        assert len(parts) >= self.world, "every rank posts before anybody collects"
        total = np.sum(parts[:self.world], axis=0)
        parts.append(None)  # one marker per collector; the entry goes when everybody has collected
        if len(parts) == 2 * self.world:
            del self.box[("sum", tag)]
        return total


class DistExchange:
    """torch.distributed neighbour exchange (NCCL on GPUs, gloo on CPU tensors).  Count and payload travel in ONE
    message per neighbour and direction: a preallocated buffer of capacity + 1 rows of 8 floats, row 0 carrying the
    row count (as a binary32 integer, exact below 2^24), rows 1.. the (pos | vel) records.  The message size is fixed,
    so nothing has to be known before the receive is posted: one batch of sends / receives per exchange and one host
    read of the two received counts, no count round trip and no allocation per step.  The tensors `collect` returns are
    views of the receive buffers: valid until the next collect (SlabSim copies them into [owned | ghosts] at once)."""

    def __init__(self, dist, rank, world, device, capacity=1 << 18):
        import torch
        self.dist, self.rank, self.world, self.device = dist, rank, world, device
        self.capacity = int(capacity)
        self.pending = {}
        mk = lambda: torch.zeros(self.capacity + 1, 8, dtype=torch.float32, device=device)  # noqa: E731
        self.send = {"l": mk(), "r": mk()}
        self.recv = {"l": mk(), "r": mk()}
        self.counts = torch.zeros(2, dtype=torch.float32, device=device)

    def post(self, rank, tag, to_left, to_right):
        self.pending[tag] = (to_left, to_right)

    def _fill(self, side, t):
        buf = self.send[side]
        k = 0 if t is None else int(t[0].shape[0])
        if k > self.capacity:
            raise RuntimeError("exchange buffer too small: %d rows > capacity %d" % (k, self.capacity))
        buf[0, 0] = float(k)
        if k:
            buf[1:1 + k, 0:4] = t[0]
            buf[1:1 + k, 4:8] = t[1]
        return buf

    def collect(self, rank, tag):
        to_left, to_right = self.pending.pop(tag)
        dist = self.dist
        left, right = rank - 1, rank + 1
        has_l, has_r = rank > 0, rank < self.world - 1
        ops = []
        if has_l:
            ops += [dist.P2POp(dist.isend, self._fill("l", to_left), left), dist.P2POp(dist.irecv, self.recv["l"], left)]
        if has_r:
            ops += [dist.P2POp(dist.isend, self._fill("r", to_right), right), dist.P2POp(dist.irecv, self.recv["r"], right)]
        for w in (dist.batch_isend_irecv(ops) if ops else []):
            w.wait()
        self.counts[0] = self.recv["l"][0, 0] if has_l else 0.0
        self.counts[1] = self.recv["r"][0, 0] if has_r else 0.0
        nl, nr = (int(v) for v in self.counts.tolist())  # the one host read of this exchange
        out = []
        for side, k in (("l", nl), ("r", nr)):
            out.append((self.recv[side][1:1 + k, 0:4], self.recv[side][1:1 + k, 4:8]) if k else None)
        return out[0], out[1]

    def post_reduce(self, rank, tag, arr):
        self.pending[("sum", tag)] = np.asarray(arr, np.int64)

    def collect_reduce(self, rank, tag):
        import torch
        t = torch.from_numpy(self.pending.pop(("sum", tag)).copy()).to(self.device)
        self.dist.all_reduce(t)
        return t.cpu().numpy()


class GpuBackend:
    """Selection and stepping through libsphboid on one GPU (device memory from torch)."""

    def __init__(self, sph, capacity, device=0, boid_capacity=1, mc_points=0):
        import torch
        from . import binding as B
        self.B, self.torch = B, torch
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.capacity = int(capacity)
        self.ctx = B.sph_create(sph, self.capacity, max(int(boid_capacity), 1), int(mc_points), device=device)
        self.scratch = [torch.empty(self.capacity, 4, device=self.device) for _ in range(2)]

    def to_device(self, a):
        return self.torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(self.device)

    def pack(self, pos, vel, n, axis, lo, hi):
        """Ordered copy of the particles of the first n with lo <= x < hi -> (pos, vel) tensors (fresh storage)."""
        if n == 0:
            return self.empty(), self.empty()
        k = self.B.sph_pack_range(self.ctx, pos, vel, n, axis, lo, hi, self.scratch[0], self.scratch[1])
        return self.scratch[0][:k].clone(), self.scratch[1][:k].clone()

    def column_hist(self, pos, n, axis, origin, h, dim):
        """Particles per cell column along `axis` (decomposition bookkeeping, not part of the frame: torch on the device,
        one small copy to the host)."""
        t = self.torch
        if n == 0:
            return np.zeros(dim, np.int64)
        col = t.clamp(t.floor((pos[:n, axis] - np.float32(origin)) / np.float32(h)).to(t.int64), 0, dim - 1)
        return t.bincount(col, minlength=dim).cpu().numpy()

    def step(self, pos, vel, bpos=None, bvel=None, boid=None):
        if bpos is None or bpos.shape[0] == 0:
            self.B.sph_step(self.ctx, pos, vel)
        else:
            self.B.sph_step(self.ctx, pos, vel, bpos, bvel, boid)
            self.B.boid_step(self.ctx, boid, bpos, bvel)

    def surface(self, pos, vel, mc, axis, lo, hi, tris):
        """S14-S17 on these particles for the cubes lo <= index < hi along axis; returns the triangle count.  The grid
        it builds is the one the following step on the same (pos, vel) reuses."""
        B = self.B
        B.mc_set_cube_range(self.ctx, -1)
        B.mc_set_cube_range(self.ctx, axis, lo, hi)
        B.sph_build_grid(self.ctx, pos, vel)
        return B.mc_extract(self.ctx, mc, tris)

    def cat(self, parts):
        return self.torch.cat(parts, 0) if len(parts) > 1 else parts[0]

    def empty(self):
        return self.torch.empty(0, 4, device=self.device)

    def close(self):
        if self.ctx is not None:
            self.B.sph_destroy(self.ctx)
            self.ctx = None


class SlabSim:
    """One rank of the decomposed run.  pos / vel: this rank's OWNED particles ((n, 4) tensors of the backend);
    bpos / bvel / boid (optional): its OWNED boids and the boid parameters."""

    def __init__(self, layout, rank, backend, exchange, pos, vel, bpos=None, bvel=None, boid=None):
        self.layout, self.rank, self.backend, self.exchange = layout, rank, backend, exchange
        self.lo, self.hi = layout.bounds(rank)
        self.pos, self.vel = pos, vel
        self.n_owned = pos.shape[0]
        self.boid = boid
        self.bpos, self.bvel = bpos, bvel
        self.nb_owned = 0 if bpos is None else bpos.shape[0]
        if boid is not None and layout.boid_halo <= 0.0:
            raise ValueError("the layout was made without the boid parameters")
        # a little over the nominal widths: the pair predicates are evaluated in binary32
        self.halo = layout.halo_width() * 1.001
        self.bhalo = layout.boid_halo_width() * 1.001
        self.step_no = 0
        self.stats = dict(ghosts=0, migrated_out=0, boid_ghosts=0, boids_migrated_out=0)

    def _faces(self, pos, vel, n, width):
        """(to_left, to_right): the first n rows within `width` of the lower / upper face."""
        ax, be = self.layout.axis, self.backend
        to_left = be.pack(pos, vel, n, ax, self.lo, self.lo + width) if self.rank > 0 else None
        to_right = be.pack(pos, vel, n, ax, self.hi - width, self.hi) if self.rank < self.layout.world - 1 else None
        return to_left, to_right

    def _leavers(self, pos, vel, n):
        """(go_left, go_right, stay) of the first n rows."""
        ax, be, inf = self.layout.axis, self.backend, math.inf
        go_left = be.pack(pos, vel, n, ax, -inf, self.lo) if self.rank > 0 else None
        go_right = be.pack(pos, vel, n, ax, self.hi, inf) if self.rank < self.layout.world - 1 else None
        return go_left, go_right, be.pack(pos, vel, n, ax, self.lo, self.hi)

    @staticmethod
    def _nonempty(parts):
        return [g for g in parts if g is not None and g[0].shape[0] > 0]

    # -- phase 1: halo ---------------------------------------------------------------------------------------------
    def post_halo(self):
        self.exchange.post(self.rank, ("halo", self.step_no), *self._faces(self.pos, self.vel, self.n_owned, self.halo))
        if self.boid is not None:
            self.exchange.post(self.rank, ("bhalo", self.step_no),
                               *self._faces(self.bpos, self.bvel, self.nb_owned, self.bhalo))

    def collect_halo(self):
        """[owned | ghosts] of this frame (fluid, and boids when present)."""
        be = self.backend
        ghosts = self._nonempty(self.exchange.collect(self.rank, ("halo", self.step_no)))
        self._all = [be.cat([self.pos] + [g[0] for g in ghosts]), be.cat([self.vel] + [g[1] for g in ghosts])]
        self.stats["ghosts"] = self._all[0].shape[0] - self.n_owned
        if self.boid is not None:
            bghosts = self._nonempty(self.exchange.collect(self.rank, ("bhalo", self.step_no)))
            self._all += [be.cat([self.bpos] + [g[0] for g in bghosts]), be.cat([self.bvel] + [g[1] for g in bghosts])]
            self.stats["boid_ghosts"] = self._all[2].shape[0] - self.nb_owned

    def surface(self, tris):
        """The surface of the CURRENT state for this rank's cubes (between collect_halo and step_collected).  Returns
        the triangle count; tris holds them in the order of the undecomposed mesh."""
        lay = self.layout
        i0, i1 = lay.cube_range(self.rank)
        return self.backend.surface(self._all[0], self._all[1], lay.mc, lay.axis, i0, i1, tris)

    def step_collected(self):
        be = self.backend
        if self.boid is None:
            be.step(self._all[0], self._all[1])  # in place; the ghosts' results are not used
        else:
            be.step(self._all[0], self._all[1], self._all[2], self._all[3], self.boid)
            self.bpos, self.bvel = self._all[2][:self.nb_owned], self._all[3][:self.nb_owned]
        self.pos, self.vel = self._all[0][:self.n_owned], self._all[1][:self.n_owned]
        self._all = None

    def step_with_halo(self):
        self.collect_halo()
        self.step_collected()

    # -- phase 2: migration ----------------------------------------------------------------------------------------
    def post_migration(self):
        go_left, go_right, self._stay = self._leavers(self.pos, self.vel, self.n_owned)
        self.stats["migrated_out"] = self.n_owned - self._stay[0].shape[0]
        self.exchange.post(self.rank, ("move", self.step_no), go_left, go_right)
        if self.boid is not None:
            go_left, go_right, self._bstay = self._leavers(self.bpos, self.bvel, self.nb_owned)
            self.stats["boids_migrated_out"] = self.nb_owned - self._bstay[0].shape[0]
            self.exchange.post(self.rank, ("bmove", self.step_no), go_left, go_right)

    def finish_migration(self):
        be = self.backend
        parts = [self._stay] + self._nonempty(self.exchange.collect(self.rank, ("move", self.step_no)))
        self.pos = be.cat([p[0] for p in parts])
        self.vel = be.cat([p[1] for p in parts])
        self.n_owned = self.pos.shape[0]
        if self.boid is not None:
            parts = [self._bstay] + self._nonempty(self.exchange.collect(self.rank, ("bmove", self.step_no)))
            self.bpos = be.cat([p[0] for p in parts])
            self.bvel = be.cat([p[1] for p in parts])
            self.nb_owned = self.bpos.shape[0]
        self.step_no += 1

    # -- re-cut: move the faces to where the particles are now --------------------------------------------------------
    def post_recut(self):
        lay = self.layout
        self._recut_tag = ("recut", self.step_no)
        self.exchange.post_reduce(self.rank, self._recut_tag,
                                  self.backend.column_hist(self.pos, self.n_owned, lay.axis, lay.origin, lay.h, lay.dim))

    def apply_recut(self):
        """New faces from the global column histogram (the same on every rank); returns the new cuts.  The particles and
        boids that now lie outside the rank's slab are moved by migration rounds (migrate_round) until none is left:
        a face that moved further than one slab needs more than one."""
        lay = self.layout
        hist = self.exchange.collect_reduce(self.rank, self._recut_tag)
        lay.set_cuts(SlabLayout.balanced_cuts(hist, lay.world, lay.min_cells))
        self.lo, self.hi = lay.bounds(self.rank)
        self._round = 0
        return lay.cuts

    def migrate_round_post(self):
        self.post_migration()

    def migrate_round_finish(self):
        """Finishes one migration round and posts how many of this rank's particles / boids are still foreign."""
        self.finish_migration()
        self.step_no -= 1  # finish_migration counts a frame; a re-cut round is not one
        self._round += 1
        ax, be, inf = self.layout.axis, self.backend, math.inf
        foreign = self.n_owned - be.pack(self.pos, self.vel, self.n_owned, ax, self.lo, self.hi)[0].shape[0]
        if self.boid is not None:
            foreign += self.nb_owned - be.pack(self.bpos, self.bvel, self.nb_owned, ax, self.lo, self.hi)[0].shape[0]
        self._round_tag = ("recut-left", self.step_no, self._round)
        self.exchange.post_reduce(self.rank, self._round_tag, [foreign])

    def migrate_round_left(self):
        return int(self.exchange.collect_reduce(self.rank, self._round_tag)[0])

    def recut(self):
        """The whole re-cut on one rank (DistExchange: every rank calls it at the same frame)."""
        self.post_recut()
        cuts = self.apply_recut()
        for _ in range(self.layout.world):
            self.migrate_round_post()
            self.migrate_round_finish()
            if self.migrate_round_left() == 0:
                break
        return cuts

    def step(self, tris=None):
        """One decomposed frame (with DistExchange every rank calls this; with LoopbackExchange drive the phases).
        With tris: the surface of the frame-start state for this rank's cubes first; returns its triangle count."""
        self.post_halo()
        self.collect_halo()
        nt = self.surface(tris) if tris is not None else None
        self.step_collected()
        self.post_migration()
        self.finish_migration()
        return nt


def split_initial(layout, pos, vel):
    """Host-side initial distribution: per rank, the (pos, vel) rows it owns, in ascending index order."""
    own = layout.owner(np.asarray(pos)[:, layout.axis])
    return [(np.ascontiguousarray(pos[own == r]), np.ascontiguousarray(vel[own == r])) for r in range(layout.world)]


def run_loopback(sims, steps, tris=None):
    """Single-process emulation: all ranks post, then all ranks collect, phase by phase.  tris: one triangle buffer
    per rank -> the surface pass of every frame-start state runs too; returns the counts of the last frame."""
    counts = None
    for _ in range(steps):
        for s in sims:
            s.post_halo()
        for s in sims:
            s.collect_halo()
        if tris is not None:
            counts = [s.surface(t) for s, t in zip(sims, tris)]
        for s in sims:
            s.step_collected()
        for s in sims:
            s.post_migration()
        for s in sims:
            s.finish_migration()
    return counts


def run_recut(sims):
    """Single-process emulation of SlabSim.recut: all ranks post, then all ranks collect, phase by phase."""
    for s in sims:
        s.post_recut()
    cuts = [s.apply_recut() for s in sims][0]
    for _ in range(len(sims)):
        for s in sims:
            s.migrate_round_post()
        for s in sims:
            s.migrate_round_finish()
        if [s.migrate_round_left() for s in sims][0] == 0:
            break
    return cuts
