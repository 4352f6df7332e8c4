"""ctypes binding of the CPU oracle (oracle/libsphref.so).  Test infrastructure only (see ref.h).

Argument marshalling only: numpy float32 (n,4) / uint32 arrays in, numpy arrays out.
"""
import ctypes as C

import numpy as np

from . import build as _build

_f = C.c_float
_u32 = C.c_uint32


class SphParams(C.Structure):
    _fields_ = [("box_min", _f * 3), ("box_max", _f * 3), ("h", _f), ("rest_density", _f), ("mass", _f),
                ("stiffness", _f), ("viscosity", _f), ("gravity", _f * 3), ("dt", _f), ("wall_damping", _f)]


class BoidParams(C.Structure):
    _fields_ = [("protect_range", _f), ("visible_range", _f), ("w_sep", _f), ("w_ali", _f), ("w_coh", _f),
                ("min_speed", _f), ("max_speed", _f), ("edge_turn", _f), ("sph_factor", _f), ("push_radius", _f),
                ("w_push", _f), ("space_min", _f * 3), ("space_max", _f * 3)]


class ObstacleParams(C.Structure):
    _fields_ = [("origin", _f * 3), ("cell", _f), ("dims", _u32 * 3), ("w_obs", _f), ("heavy", _f)]


class McParams(C.Structure):
    _fields_ = [("origin", _f * 3), ("spacing", _f), ("n_point_per_axis", _u32), ("radius", _f),
                ("particle_radius", _f), ("iso", _f)]


def _fill(struct, d):
    s = struct()
    for name, ctype in struct._fields_:
        if name not in d:
            continue
        v = d[name]
        if hasattr(ctype, "_length_"):
            conv = int if ctype._type_ is C.c_uint32 else float
            setattr(s, name, ctype(*[conv(x) for x in v]))
        else:
            setattr(s, name, v)
    return s


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp = C.c_void_p
        L.ref_grid_dims.restype = _u32
        L.ref_grid_dims.argtypes = [vp, vp]
        L.ref_build_grid.argtypes = [vp, vp, _u32, vp, vp, vp]
        L.ref_density.argtypes = [vp, vp, _u32, C.c_int, vp, vp]
        L.ref_boid_density.argtypes = [vp, vp, _u32, vp, _u32, C.c_int, vp]
        L.ref_step.argtypes = [vp, vp, vp, _u32, vp, vp, _u32, vp, C.c_int, vp, vp, vp, vp, vp]
        L.ref_boid_step.argtypes = [vp, vp, vp, vp, vp, _u32, vp, vp, _u32, C.c_int, vp]
        L.ref_boid_obstacles.argtypes = [vp, vp, _f, _f, vp, vp, _u32, C.c_int]
        L.ref_voxel_sdf.argtypes = [vp, vp, vp, _u32, C.c_int, vp]
        L.ref_mc_polygonise.argtypes = [vp, vp, vp, _u32, vp, vp]
        L.ref_mc_indexed.argtypes = [vp, vp, vp, vp, _u32, vp, _u32, vp, vp]
        L.ref_mesh_components.argtypes = [vp, _u32, _u32, vp, vp, vp]
        L.ref_mc_table.argtypes = [vp, vp, vp]
        L.ref_mc_table.restype = None
        L.ref_mc_numbering.argtypes = [vp, vp]
        L.ref_mc_numbering.restype = None
        L.ref_w_poly6.restype = C.c_double
        L.ref_w_poly6.argtypes = [C.c_double, C.c_double]
        L.ref_pair_term.argtypes = [_f, _f, _f, _f, _f, vp, vp, _f, vp, vp, _f, vp]
        L.ref_pair_term.restype = None
        L.ref_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f4(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] == 4
    return a


def num_threads():
    return int(lib().ref_num_threads())


def grid_dims(sp):
    s = _fill(SphParams, sp)
    dims = np.zeros(3, np.uint32)
    c = lib().ref_grid_dims(C.byref(s), _p(dims))
    return tuple(int(x) for x in dims), int(c)


def build_grid(sp, pos):
    pos = _f4(pos)
    n = pos.shape[0]
    _, ncell = grid_dims(sp)
    s = _fill(SphParams, sp)
    cell = np.zeros(n, np.uint32)
    perm = np.zeros(n, np.uint32)
    start = np.zeros(ncell + 1, np.uint32)
    rc = lib().ref_build_grid(C.byref(s), _p(pos), n, _p(cell), _p(perm), _p(start))
    assert rc == 0
    return cell, perm, start


def density(sp, pos, brute=False):
    pos = _f4(pos)
    n = pos.shape[0]
    s = _fill(SphParams, sp)
    rho = np.zeros(n, np.float32)
    cnt = np.zeros(n, np.uint32)
    rc = lib().ref_density(C.byref(s), _p(pos), n, int(brute), _p(rho), _p(cnt))
    assert rc == 0
    return rho, cnt


def boid_density(sp, pos, bpos, brute=False):
    pos, bpos = _f4(pos), _f4(bpos)
    s = _fill(SphParams, sp)
    rho_b = np.zeros(bpos.shape[0], np.float32)
    rc = lib().ref_boid_density(C.byref(s), _p(pos), pos.shape[0], _p(bpos), bpos.shape[0], int(brute), _p(rho_b))
    assert rc == 0
    return rho_b


def step(sp, pos, vel, bpos=None, bvel=None, bp=None, brute=False):
    """One SPH step.  Returns dict(pos, vel, density, accel, ncount, touched, amag); inputs untouched."""
    pos, vel = _f4(pos).copy(), _f4(vel).copy()
    n = pos.shape[0]
    s = _fill(SphParams, sp)
    nb = 0 if bpos is None else bpos.shape[0]
    b = _fill(BoidParams, bp) if nb > 0 else None
    if nb > 0:
        bpos, bvel = _f4(bpos), _f4(bvel)
    rho = np.zeros(n, np.float32)
    acc = np.zeros((n, 4), np.float32)
    cnt = np.zeros(n, np.uint32)
    tch = np.zeros(n, np.uint32)
    amag = np.zeros(n, np.float32)
    rc = lib().ref_step(C.byref(s), _p(pos), _p(vel), n, _p(bpos) if nb else None, _p(bvel) if nb else None, nb,
                        C.byref(b) if nb else None, int(brute), _p(rho), _p(acc), _p(cnt), _p(tch), _p(amag))
    assert rc == 0
    return dict(pos=pos, vel=vel, density=rho, accel=acc, ncount=cnt, touched=tch, amag=amag)


def boid_step(sp, bp, pos, vel, rho, bpos, bvel, brute=False):
    """One boid step from the step-start fluid state.  Returns dict(bpos, bvel, dv_parts)."""
    pos, vel = _f4(pos), _f4(vel)
    rho = np.ascontiguousarray(rho, np.float32)
    bpos, bvel = _f4(bpos).copy(), _f4(bvel).copy()
    nb = bpos.shape[0]
    s, b = _fill(SphParams, sp), _fill(BoidParams, bp)
    parts = np.zeros((nb, 4, 4), np.float32)
    rc = lib().ref_boid_step(C.byref(s), C.byref(b), _p(pos), _p(vel), _p(rho), pos.shape[0], _p(bpos), _p(bvel),
                             nb, int(brute), _p(parts))
    assert rc == 0
    return dict(bpos=bpos, bvel=bvel, dv_parts=parts)


def boid_obstacles(op, normals, protect_range, visible_range, bpos, bvel, brute=False):
    """N4: obstacle avoidance on the post-update boid state.  normals (cells, 4) float32.  Returns the new bvel."""
    o = _fill(ObstacleParams, op)
    normals = np.ascontiguousarray(normals, np.float32)
    assert normals.shape == (int(np.prod(op["dims"])), 4)
    bpos, bvel = _f4(bpos), _f4(bvel).copy()
    rc = lib().ref_boid_obstacles(C.byref(o), _p(normals), protect_range, visible_range, _p(bpos), _p(bvel),
                                  bpos.shape[0], int(brute))
    assert rc == 0
    return bvel


def voxel_sdf(sp, mp, pos, brute=False):
    pos = _f4(pos)
    s, m = _fill(SphParams, sp), _fill(McParams, mp)
    g = int(mp["n_point_per_axis"])
    phi = np.zeros(g * g * g, np.float32)
    rc = lib().ref_voxel_sdf(C.byref(s), C.byref(m), _p(pos), pos.shape[0], int(brute), _p(phi))
    assert rc == 0
    return phi


def mc_polygonise(mp, phi, capacity=None, want_cases=False):
    """Returns (tris (T,3,3) float32, n_tris required, cases or None)."""
    m = _fill(McParams, mp)
    g = int(mp["n_point_per_axis"])
    phi = np.ascontiguousarray(phi, np.float32)
    assert phi.size == g ** 3
    nt = _u32(0)
    cases = np.zeros(max(g - 1, 0) ** 3, np.uint8) if want_cases else None
    if capacity is None:
        lib().ref_mc_polygonise(C.byref(m), _p(phi), None, 0, C.byref(nt), None)
        capacity = nt.value
    tris = np.zeros((max(capacity, 1), 3, 3), np.float32)
    rc = lib().ref_mc_polygonise(C.byref(m), _p(phi), _p(tris), capacity, C.byref(nt), _p(cases))
    assert rc in (0, 1)
    return tris[:min(capacity, nt.value)], int(nt.value), cases


def mc_indexed(mp, phi):
    """N3: returns (verts (V,3), normals (V,3), indices (T,3) uint32) of the welded mesh."""
    m = _fill(McParams, mp)
    g = int(mp["n_point_per_axis"])
    phi = np.ascontiguousarray(phi, np.float32)
    assert phi.size == g ** 3
    nv, nt = _u32(0), _u32(0)
    lib().ref_mc_indexed(C.byref(m), _p(phi), None, None, 0, None, 0, C.byref(nv), C.byref(nt))
    verts = np.zeros((max(nv.value, 1), 3), np.float32)
    normals = np.zeros((max(nv.value, 1), 3), np.float32)
    idx = np.zeros((max(nt.value, 1), 3), np.uint32)
    rc = lib().ref_mc_indexed(C.byref(m), _p(phi), _p(verts), _p(normals), nv.value, _p(idx), nt.value, C.byref(nv),
                              C.byref(nt))
    assert rc == 0
    return verts[:nv.value], normals[:nv.value], idx[:nt.value]


def mesh_components(indices, n_verts):
    """N3 connectivity: returns (label (V,) uint32 = smallest vertex id of the component, n_components, largest_tris)."""
    idx = np.ascontiguousarray(indices, np.uint32).reshape(-1, 3)
    label = np.zeros(max(int(n_verts), 1), np.uint32)
    nc, big = _u32(0), _u32(0)
    rc = lib().ref_mesh_components(_p(idx) if idx.size else None, idx.shape[0], int(n_verts), _p(label), C.byref(nc),
                                   C.byref(big))
    assert rc == 0
    return label[:int(n_verts)], int(nc.value), int(big.value)


def mc_table():
    tri = np.zeros((256, 16), np.int8)
    ntri = np.zeros(256, np.uint8)
    edge = np.zeros(256, np.uint16)
    lib().ref_mc_table(_p(tri), _p(ntri), _p(edge))
    return tri, ntri, edge


def mc_numbering():
    corners = np.zeros((8, 3), np.int32)
    edges = np.zeros((12, 2), np.int32)
    lib().ref_mc_numbering(_p(corners), _p(edges))
    return corners, edges


def w_poly6(r, h):
    return float(lib().ref_w_poly6(float(r), float(h)))


def pair_term(mass, radius, stiffness, rest_density, viscosity, pa, va, rho_a, pb, vb, rho_b):
    out = np.zeros(3, np.float32)
    a = [np.ascontiguousarray(x, np.float32) for x in (pa, va, pb, vb)]
    lib().ref_pair_term(mass, radius, stiffness, rest_density, viscosity, _p(a[0]), _p(a[1]), rho_a, _p(a[2]),
                        _p(a[3]), rho_b, _p(out))
    return out
