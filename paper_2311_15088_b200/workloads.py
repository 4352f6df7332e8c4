"""Seeded synthetic workloads (the five BASELINE.json configs) -- inputs only, no method arithmetic.

This module serves BOTH the CPU oracle's tests and the CUDA path (it imports neither): it builds
dam-break particle lattices, boid swarms and parameter dictionaries whose keys are the field names of
the parameter structs.  The paper's own workloads are Unity scenes that do not exist
here; these configs stand in for them with the paper's workload shape (N up to 1e6+, tens of
neighbours per particle, uniform grid; Tables 1-2).  Recipe: DESIGN.md section 4.

Random numbers come from a counter-based integer hash of (seed, stream, index, axis), so any element
can be regenerated independently and the result does not depend on numpy's generator version.
"""
import numpy as np

_M32 = np.uint64(0xFFFFFFFF)


def _mix32(x):
    """A 32-bit integer finaliser (xor-shift-multiply rounds) applied elementwise to uint64-held values."""
    x = x & _M32
    x ^= x >> np.uint64(16)
    x = (x * np.uint64(0x7FEB352D)) & _M32
    x ^= x >> np.uint64(15)
    x = (x * np.uint64(0x846CA68B)) & _M32
    x ^= x >> np.uint64(16)
    return x


def uniform01(seed, stream, index, axis):
    """U[0,1) float64 with 24 random bits from hash(seed, stream, index, axis)."""
    index = np.asarray(index, dtype=np.uint64)
    x = _mix32(index * np.uint64(3) + np.uint64(axis) + np.uint64(0x9E3779B9) * np.uint64(stream + 1))
    x = _mix32(x ^ (np.uint64(seed) * np.uint64(0x85EBCA6B) & _M32) ^ np.uint64(0x68E31DA4))
    return (x >> np.uint64(8)).astype(np.float64) / float(1 << 24)


def lattice(nx, ny, nz, spacing, jitter, seed, origin=(0.0, 0.0, 0.0)):
    """Cell-centred lattice x = origin + (i + 1/2) * spacing, id = i + nx*(j + ny*k), jittered by +-jitter."""
    n = nx * ny * nz
    idx = np.arange(n, dtype=np.uint64)
    i = (idx % np.uint64(nx)).astype(np.float64)
    j = ((idx // np.uint64(nx)) % np.uint64(ny)).astype(np.float64)
    k = (idx // np.uint64(nx * ny)).astype(np.float64)
    pos = np.zeros((n, 4), np.float32)
    for axis, c in enumerate((i, j, k)):
        u = uniform01(seed, 0, idx, axis) * 2.0 - 1.0
        pos[:, axis] = (origin[axis] + (c + 0.5) * spacing + u * jitter).astype(np.float32)
    return pos


def uniform_box(n, lo, hi, seed, stream):
    idx = np.arange(n, dtype=np.uint64)
    out = np.zeros((n, 4), np.float32)
    for axis in range(3):
        u = uniform01(seed, stream, idx, axis)
        out[:, axis] = (lo[axis] + u * (hi[axis] - lo[axis])).astype(np.float32)
    return out


def uniform_ball(n, centre, radius, seed, stream):
    """Uniform in a ball: direction from three hashed normals (Box-Muller), radius ~ U^(1/3)."""
    idx = np.arange(n, dtype=np.uint64)
    g = []
    for axis in range(3):
        u1 = np.maximum(uniform01(seed, stream, idx, axis), 1e-12)
        u2 = uniform01(seed, stream + 1, idx, axis)
        g.append(np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2))
    g = np.stack(g, 1)
    g /= np.maximum(np.linalg.norm(g, axis=1, keepdims=True), 1e-30)
    r = radius * uniform01(seed, stream + 2, idx, 0) ** (1.0 / 3.0)
    out = np.zeros((n, 4), np.float32)
    out[:, :3] = (np.asarray(centre)[None, :] + g * r[:, None]).astype(np.float32)
    return out


# name -> (nx, ny, nz, log2(1/a), spacing factor, box_max, n_boid, steps, G)
_CONFIGS = {
    1: dict(lat=(16, 16, 16), a=2.0 ** -5, sf=1.0, box=(1.0, 1.0, 1.0), n_boid=64, steps=10, G=32),
    2: dict(lat=(64, 64, 16), a=2.0 ** -7, sf=1.0, box=(1.0, 1.0, 1.0), n_boid=256, steps=100, G=64),
    3: dict(lat=(64, 64, 64), a=2.0 ** -6, sf=1.0, box=(2.0, 1.0, 1.0), n_boid=1024, steps=100, G=128),
    4: dict(lat=(128, 128, 64), a=2.0 ** -7, sf=1.0, box=(2.0, 1.0, 0.5), n_boid=4096, steps=100, G=256),
    5: dict(lat=(256, 128, 128), a=2.0 ** -7, sf=0.8, box=(2.0, 1.0, 1.0), n_boid=16384, steps=20, G=256),
}


def config(idx, seed=0, scale=None):
    """Return the workload dict for BASELINE.json config `idx` (1-5).

    Keys: name, n, n_boid, steps, sph (dict), boid (dict), pos, vel, bpos, bvel ((n,4) float32), G.
    `scale` (tests only) shrinks the lattice extents by an integer factor per axis, keeping h and spacing.
    """
    c = _CONFIGS[idx]
    nx, ny, nz = c["lat"]
    if scale:
        nx, ny, nz = max(nx // scale, 1), max(ny // scale, 1), max(nz // scale, 1)
    a = c["a"]
    h = 2.0 * a
    spacing = a * c["sf"]
    pos = lattice(nx, ny, nz, spacing, 0.096 * spacing, seed)
    vel = np.zeros_like(pos)
    fluid_hi = (nx * spacing, ny * spacing, nz * spacing)
    sph = dict(box_min=(0.0, 0.0, 0.0), box_max=c["box"], h=h, rest_density=1000.0, mass=1000.0 * a ** 3,
               stiffness=3.0, viscosity=0.1, gravity=(0.0, -9.81, 0.0), dt=1e-3, wall_damping=0.5)
    nb = c["n_boid"] if not scale else max(c["n_boid"] // scale ** 2, 8)
    rng_range = 0.1 if idx == 1 else 1.6 * h
    boid = dict(protect_range=rng_range, visible_range=rng_range, w_sep=1.5, w_ali=1.0, w_coh=1.0, min_speed=0.0,
                max_speed=0.5, edge_turn=0.05, sph_factor=1.0, push_radius=(2.0 * h if idx == 3 else h), w_push=1.0,
                space_min=(0.0, 0.0, 0.0), space_max=c["box"])
    if idx in (1, 2):
        bpos = uniform_box(nb, (0.6, 0.6, 0.6), (0.9, 0.9, 0.9), seed, 10)
        bvel = uniform_box(nb, (-0.1,) * 3, (0.1,) * 3, seed, 20)
    elif idx == 3:
        bpos = uniform_box(nb, tuple(0.2 * x for x in fluid_hi), tuple(0.8 * x for x in fluid_hi), seed, 10)
        bvel = uniform_box(nb, (0.25, -0.05, -0.05), (0.35, 0.05, 0.05), seed, 20)
    elif idx == 4:
        bpos = uniform_box(nb, (0.0, 0.0, 0.0), fluid_hi, seed, 10)
        bvel = uniform_box(nb, (-0.1,) * 3, (0.1,) * 3, seed, 20)
    else:
        bpos = uniform_ball(nb, (0.5 * fluid_hi[0], 0.5 * fluid_hi[1], 0.5 * fluid_hi[2]), 3.0 * h, seed, 10)
        bvel = uniform_box(nb, (-0.1,) * 3, (0.1,) * 3, seed, 20)
    return dict(name="config%d" % idx, idx=idx, n=pos.shape[0], n_boid=nb, steps=c["steps"], sph=sph, boid=boid,
                pos=pos, vel=vel, bpos=bpos, bvel=bvel, G=c["G"] if not scale else max(c["G"] // scale, 8),
                lattice=(nx, ny, nz), spacing=spacing)


def mc_params(cfg, pos=None):
    """MC grid for a workload: configs 1-3 span the box from the origin; 4-5 span the fluid AABB of `pos`."""
    h = cfg["sph"]["h"]
    G = cfg["G"]
    if cfg["idx"] in (1, 2, 3):
        origin = (0.0, 0.0, 0.0)
        extent = max(cfg["sph"]["box_max"])
    else:
        p = cfg["pos"] if pos is None else np.asarray(pos)
        lo = p[:, :3].min(axis=0)
        hi = p[:, :3].max(axis=0)
        origin = tuple(float(x) for x in lo)
        extent = float((hi - lo).max())
    return dict(origin=origin, spacing=float(np.float32(extent / (G - 1))), n_point_per_axis=G, radius=h,
                particle_radius=0.5 * h, iso=0.0)


def random_cloud(n, lo, hi, seed):
    """Uniform random points (tests: brute-force pins)."""
    return uniform_box(n, lo, hi, seed, 40)


def sphere_obstacle(space_min, space_max, cell, centre, radius, w_obs=0.05, heavy=2.0):
    """Synthetic Obstacle Grid (stands in for the paper's obstacle meshes): a grid of `cell`
    over the Boid Space whose cells within half a cell diagonal of the sphere's surface carry the outward unit normal of
    the sphere at the cell centre, all others zero.  Returns (obstacle params dict, normals (cells, 4) float32).
    Input construction only: no part of the avoidance rule is evaluated here."""
    lo = np.asarray(space_min, np.float64)
    hi = np.asarray(space_max, np.float64)
    dims = np.maximum(1, np.ceil((hi - lo) / cell)).astype(np.int64)
    cz, cy, cx = np.meshgrid(np.arange(dims[2]), np.arange(dims[1]), np.arange(dims[0]), indexing="ij")
    xc = np.stack([np.float32(lo[0]) + (cx.astype(np.float32) + np.float32(0.5)) * np.float32(cell),
                   np.float32(lo[1]) + (cy.astype(np.float32) + np.float32(0.5)) * np.float32(cell),
                   np.float32(lo[2]) + (cz.astype(np.float32) + np.float32(0.5)) * np.float32(cell)], -1).reshape(-1, 3)
    d = xc.astype(np.float64) - np.asarray(centre, np.float64)
    r = np.linalg.norm(d, axis=1)
    on = np.abs(r - radius) <= 0.5 * np.sqrt(3.0) * cell
    normals = np.zeros((xc.shape[0], 4), np.float32)
    normals[on, :3] = (d[on] / r[on, None]).astype(np.float32)
    op = dict(origin=tuple(float(np.float32(v)) for v in lo), cell=float(np.float32(cell)),
              dims=tuple(int(v) for v in dims), w_obs=float(w_obs), heavy=float(heavy))
    return op, normals
