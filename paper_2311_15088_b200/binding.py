"""ctypes binding of libsphboid.so -- same names as include/sphboid.h, argument marshalling only.

Device arrays are torch CUDA tensors (PyTorch supplies device memory and streams, nothing else): float32
(n,4) for pos / vel / bpos / bvel / accel, uint32-as-int32 for index outputs.  Every step of the path runs
in the library's CUDA kernels; there is NO CPU fallback -- a missing library or device raises.
"""
import ctypes as C
import os

_f = C.c_float
_u32 = C.c_uint32
_vp = C.c_void_p

SPH_OK, SPH_E_INVALID, SPH_E_CAPACITY, SPH_E_STALE_GRID, SPH_E_CUDA = 0, -1, -2, -3, -4


class SphParams(C.Structure):
    _fields_ = [("box_min", _f * 3), ("box_max", _f * 3), ("h", _f), ("rest_density", _f), ("mass", _f),
                ("stiffness", _f), ("viscosity", _f), ("gravity", _f * 3), ("dt", _f), ("wall_damping", _f),
                ("max_particles", _u32), ("max_boids", _u32), ("max_mc_points_per_axis", _u32)]


class BoidParams(C.Structure):
    _fields_ = [("protect_range", _f), ("visible_range", _f), ("w_sep", _f), ("w_ali", _f), ("w_coh", _f),
                ("min_speed", _f), ("max_speed", _f), ("edge_turn", _f), ("sph_factor", _f), ("push_radius", _f),
                ("w_push", _f), ("space_min", _f * 3), ("space_max", _f * 3)]


class ObstacleParams(C.Structure):
    _fields_ = [("origin", _f * 3), ("cell", _f), ("dims", _u32 * 3), ("w_obs", _f), ("heavy", _f)]


class McParams(C.Structure):
    _fields_ = [("origin", _f * 3), ("spacing", _f), ("n_point_per_axis", _u32), ("radius", _f),
                ("particle_radius", _f), ("iso", _f)]


class SphError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libsphboid error %d: %s" % (code, msg))
        self.code = code


def _fill(struct, d):
    if isinstance(d, struct):
        return d
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


LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libsphboid.so")
_lib = None


def lib():
    """Load libsphboid.so (built in-tree by paper_2311_15088_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libsphboid.so is not built: run `python -m paper_2311_15088_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.sph_create.argtypes = [C.POINTER(_vp), _vp, C.c_int]
        L.sph_destroy.argtypes = [_vp]
        L.sph_last_error.argtypes = [_vp]
        L.sph_last_error.restype = C.c_char_p
        L.sph_grid_dims.argtypes = [_vp, _vp]
        L.sph_grid_dims.restype = _u32
        L.sph_build_grid.argtypes = [_vp, _vp, _vp, _u32, _vp, _vp, _vp, _vp]
        L.sph_step.argtypes = [_vp, _vp, _vp, _u32, _vp, _vp, _u32, _vp, _vp, _vp, _vp, _vp, _vp]
        L.boid_step.argtypes = [_vp, _vp, _vp, _vp, _u32, _vp, _vp]
        L.mc_voxel_sdf.argtypes = [_vp, _vp, _vp, _vp]
        L.mc_set_sdf_variant.argtypes = [_vp, C.c_int]
        L.mc_set_cube_range.argtypes = [_vp, C.c_int, _u32, _u32]
        L.boid_set_obstacles.argtypes = [_vp, _vp, _vp]
        L.sph_neighbor_count.argtypes = [_vp, _vp, _u32, _vp, _vp]
        L.sph_pack_range.argtypes = [_vp, _vp, _vp, _u32, C.c_int, _f, _f, _vp, _vp, _vp, _u32, _vp]
        L.sph_hashgrid_neighbor_count.argtypes = [_vp, _vp, _u32, _u32, _vp, _vp, _vp]
        L.sph_set_force_variant.argtypes = [_vp, C.c_int]
        L.sph_particle_aabb.argtypes = [_vp, _vp, _vp]
        L.sph_invalidate_grid.argtypes = [_vp]
        L.mc_polygonise.argtypes = [_vp, _vp, _vp, _vp, _vp, _u32, _vp, _vp]
        L.mc_extract.argtypes = [_vp, _vp, _vp, _vp, _vp, _u32, _vp]
        L.mc_extract_async.argtypes = [_vp, _vp, _vp, _vp, _vp, _u32]
        L.mc_wait.argtypes = [_vp, _vp, _vp]
        L.mc_polygonise_indexed.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _u32, _vp, _u32, _vp, _vp]
        L.mc_extract_indexed.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _u32, _vp, _u32, _vp, _vp]
        L.mc_mesh_components.argtypes = [_vp, _vp, _u32, _u32, _vp, _vp, _vp, _vp]
        L.sph_simulate_host.argtypes = [_vp, _vp, _vp, _u32, _vp, _vp, _u32, _vp, _u32, _vp, _vp, _u32, _vp]
        L.sph_mc_table.argtypes = [_vp, _vp]
        L.sph_mc_table.restype = None
        L.sph_launch_count.argtypes = [_vp]
        L.sph_launch_count.restype = C.c_uint64
        L.sph_profile_enable.argtypes = [_vp, C.c_int]
        L.sph_profile_read.argtypes = [_vp, _u32, _vp, _vp]
        L.sph_kernel_name.argtypes = [_u32]
        L.sph_kernel_name.restype = C.c_char_p
        L.sph_build_grid_static.argtypes = [_vp, _vp, _f, _vp, _u32, _vp, _vp, _vp, _vp, _u32]
        L.sph_static_last_error.argtypes = []
        L.sph_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


EXPORTS = ["sph_create", "sph_destroy", "sph_last_error", "sph_grid_dims", "sph_build_grid", "sph_step", "boid_step",
           "sph_particle_aabb", "sph_invalidate_grid", "mc_voxel_sdf", "mc_set_sdf_variant", "mc_set_cube_range", "sph_set_force_variant", "boid_set_obstacles", "sph_neighbor_count", "sph_pack_range", "sph_hashgrid_neighbor_count", "mc_polygonise", "mc_extract", "mc_extract_async", "mc_wait", "mc_polygonise_indexed", "mc_extract_indexed", "mc_mesh_components", "sph_simulate_host", "sph_mc_table", "sph_launch_count", "sph_profile_enable",
           "sph_profile_read", "sph_kernel_name", "sph_build_grid_static", "sph_static_last_error"]


def _ptr(t):
    """Device pointer of a torch CUDA tensor (or None)."""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "expected a contiguous CUDA tensor"
    return _vp(t.data_ptr())


def _hptr(a):
    """Host pointer of a numpy array or CPU torch tensor (or None)."""
    if a is None:
        return None
    if hasattr(a, "data_ptr"):
        assert not a.is_cuda and a.is_contiguous()
        return _vp(a.data_ptr())
    assert a.flags["C_CONTIGUOUS"]
    return _vp(a.ctypes.data)


def _stream(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    elif hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    return _vp(stream)


def _check(ctx, rc, allow=()):
    if rc != SPH_OK and rc not in allow:
        raise SphError(rc, lib().sph_last_error(ctx).decode() if ctx else "no context")
    return rc


def sph_create(params, max_particles, max_boids=0, max_mc_points_per_axis=0, device=0):
    p = _fill(SphParams, dict(params, max_particles=max_particles, max_boids=max_boids,
                              max_mc_points_per_axis=max_mc_points_per_axis))
    h = _vp()
    rc = lib().sph_create(C.byref(h), C.byref(p), device)
    if rc != SPH_OK:
        raise SphError(rc, "sph_create failed (no CUDA device, bad parameters or out of memory)")
    return h


def sph_destroy(ctx):
    lib().sph_destroy(ctx)


def sph_grid_dims(ctx):
    dims = (_u32 * 3)()
    c = lib().sph_grid_dims(ctx, dims)
    return tuple(dims), int(c)


def sph_launch_count(ctx):
    return int(lib().sph_launch_count(ctx))


def sph_profile_enable(ctx, enable=True):
    return _check(ctx, lib().sph_profile_enable(ctx, 1 if enable else 0))


def sph_profile_read(ctx):
    """{kernel name: (launches, total ms)} for every kernel that launched since sph_profile_enable."""
    out = {}
    k = 0
    while True:
        name = lib().sph_kernel_name(k)
        if name is None:
            break
        n, ms = C.c_uint64(0), C.c_double(0.0)
        _check(ctx, lib().sph_profile_read(ctx, k, C.byref(n), C.byref(ms)))
        if n.value:
            out[name.decode()] = (int(n.value), float(ms.value))
        k += 1
    return out


def sph_mc_table():
    import numpy as np
    tri = np.zeros((256, 16), np.int8)
    ntri = np.zeros(256, np.uint8)
    lib().sph_mc_table(_hptr(tri), _hptr(ntri))
    return tri, ntri


def sph_build_grid(ctx, pos, vel=None, stream=None, cell_of_particle=None, perm=None, cell_start=None):
    n = 0 if pos is None else pos.shape[0]
    return _check(ctx, lib().sph_build_grid(ctx, _ptr(pos), _ptr(vel), n, _stream(stream), _ptr(cell_of_particle),
                                            _ptr(perm), _ptr(cell_start)))


SPH_STATIC_MAX_POINTS, SPH_STATIC_MAX_CELLS = 16384, 8192


def sph_build_grid_static(box_min, box_max, h, pos, cell_of_particle, perm, cell_start, stream=None):
    """S1-S5 without a context and without any allocation (include/sphboid.h): at most SPH_STATIC_MAX_POINTS points and
    SPH_STATIC_MAX_CELLS cells; the outputs are the caller's CUDA tensors (cell_start: at least C + 1 entries)."""
    lo = (_f * 3)(*[float(v) for v in box_min])
    hi = (_f * 3)(*[float(v) for v in box_max])
    n = 0 if pos is None else pos.shape[0]
    rc = lib().sph_build_grid_static(lo, hi, float(h), _ptr(pos), n, _stream(stream), _ptr(cell_of_particle), _ptr(perm),
                                     _ptr(cell_start), 0 if cell_start is None else cell_start.numel())
    if rc != SPH_OK:
        raise SphError(rc, lib().sph_static_last_error().decode())
    return rc


def sph_step(ctx, pos, vel, bpos=None, bvel=None, boid=None, stream=None, density=None, accel=None, ncount=None,
             touched=None):
    nb = 0 if bpos is None else bpos.shape[0]
    bp = _fill(BoidParams, boid) if nb else None
    return _check(ctx, lib().sph_step(ctx, _ptr(pos), _ptr(vel), pos.shape[0], _ptr(bpos) if nb else None,
                                      _ptr(bvel) if nb else None, nb, C.byref(bp) if nb else None, _stream(stream),
                                      _ptr(density), _ptr(accel), _ptr(ncount), _ptr(touched)))


def boid_step(ctx, boid, bpos, bvel, stream=None, dv_parts=None):
    bp = _fill(BoidParams, boid)
    return _check(ctx, lib().boid_step(ctx, C.byref(bp), _ptr(bpos), _ptr(bvel), bpos.shape[0], _stream(stream),
                                       _ptr(dv_parts)))


def mc_voxel_sdf(ctx, mc, phi, stream=None):
    m = _fill(McParams, mc)
    return _check(ctx, lib().mc_voxel_sdf(ctx, C.byref(m), _stream(stream), _ptr(phi)))


def boid_set_obstacles(ctx, op, normals):
    """N4: Obstacle Grid for the boids (op dict + (cells, 4) float32 CUDA tensor that must stay alive), or None to clear."""
    if op is None or normals is None:
        return _check(ctx, lib().boid_set_obstacles(ctx, None, None))
    o = _fill(ObstacleParams, op)
    return _check(ctx, lib().boid_set_obstacles(ctx, C.byref(o), _ptr(normals)))


def sph_pack_range(ctx, pos, vel, n, axis, lo, hi, out_pos, out_vel, stream=None):
    """N2: ordered copy of the particles with lo <= pos[axis] < hi among the first n; returns their number."""
    cnt = _u32(0)
    rc = lib().sph_pack_range(ctx, _ptr(pos), _ptr(vel), int(n), int(axis), float(lo), float(hi), _stream(stream),
                              _ptr(out_pos), _ptr(out_vel), 0 if out_pos is None else out_pos.shape[0], C.byref(cnt))
    _check(ctx, rc)
    return int(cnt.value)


def sph_neighbor_count(ctx, pos, ncount, stream=None):
    """Neighbour counts through the sorted grid (builds it on pos)."""
    return _check(ctx, lib().sph_neighbor_count(ctx, _ptr(pos), pos.shape[0], _stream(stream), _ptr(ncount)))


def sph_hashgrid_neighbor_count(ctx, pos, max_per_cell, ncount, stream=None, sync=True):
    """N4 baseline: the same counts through the paper's unsorted fixed-capacity hash grid.  Returns the number of
    particles dropped from full cells when sync."""
    dropped = _u32(0)
    _check(ctx, lib().sph_hashgrid_neighbor_count(ctx, _ptr(pos), pos.shape[0], int(max_per_cell), _stream(stream),
                                                  _ptr(ncount), C.byref(dropped) if sync else None))
    return int(dropped.value) if sync else None


def sph_invalidate_grid(ctx):
    return _check(ctx, lib().sph_invalidate_grid(ctx))


def sph_particle_aabb(ctx, stream=None):
    """(lo, hi): exact bounding box of the particles of the last sph_build_grid; synchronises the stream."""
    out = (C.c_float * 6)()
    _check(ctx, lib().sph_particle_aabb(ctx, _stream(stream), out))
    return tuple(out[0:3]), tuple(out[3:6])


def sph_set_force_variant(ctx, variant):
    return _check(ctx, lib().sph_set_force_variant(ctx, int(variant)))


def mc_set_cube_range(ctx, axis, lo=0, hi=0xffffffff):
    """Polygonise only the cubes with lo <= index < hi along axis (axis = -1: the whole grid again)."""
    return _check(ctx, lib().mc_set_cube_range(ctx, int(axis), int(lo), int(hi)))


def mc_set_sdf_variant(ctx, variant):
    return _check(ctx, lib().mc_set_sdf_variant(ctx, int(variant)))


def mc_polygonise(ctx, mc, phi, tris, stream=None, sync=True, n_tris_dev=None):
    """Returns the required triangle count (int) when sync, else None.  tris: (capacity, 3, 3) float32 CUDA."""
    m = _fill(McParams, mc)
    nt = _u32(0)
    cap = 0 if tris is None else tris.shape[0]
    rc = lib().mc_polygonise(ctx, C.byref(m), _ptr(phi), _stream(stream), _ptr(tris), cap,
                             C.byref(nt) if sync else None, _ptr(n_tris_dev))
    _check(ctx, rc, allow=(SPH_E_CAPACITY,))
    return int(nt.value) if sync else None


def mc_extract(ctx, mc, tris, phi=None, stream=None, sync=True):
    m = _fill(McParams, mc)
    nt = _u32(0)
    cap = 0 if tris is None else tris.shape[0]
    rc = lib().mc_extract(ctx, C.byref(m), _stream(stream), _ptr(phi), _ptr(tris), cap, C.byref(nt) if sync else None)
    _check(ctx, rc, allow=(SPH_E_CAPACITY,))
    return int(nt.value) if sync else None


def mc_extract_async(ctx, mc, tris, phi=None, stream=None):
    """S14-S17 on the context's surface stream, beside whatever is enqueued on `stream` afterwards; see mc_wait."""
    m = _fill(McParams, mc)
    cap = 0 if tris is None else tris.shape[0]
    return _check(ctx, lib().mc_extract_async(ctx, C.byref(m), _stream(stream), _ptr(phi), _ptr(tris), cap))


def mc_wait(ctx, stream=None, sync=True):
    """Orders `stream` after the pending surface pass; returns the required triangle count when sync."""
    nt = _u32(0)
    rc = lib().mc_wait(ctx, _stream(stream), C.byref(nt) if sync else None)
    _check(ctx, rc, allow=(SPH_E_CAPACITY,))
    return int(nt.value) if sync else None


def mc_polygonise_indexed(ctx, mc, phi, verts, normals, indices, stream=None, sync=True):
    """N3: indexed mesh of a given phi.  verts / normals (Vcap, 3) float32, indices (Tcap, 3) int32 CUDA tensors
    (normals may be None).  Returns (n_verts, n_tris) required when sync, else None."""
    m = _fill(McParams, mc)
    nv, nt = _u32(0), _u32(0)
    rc = lib().mc_polygonise_indexed(ctx, C.byref(m), _ptr(phi), _stream(stream), _ptr(verts), _ptr(normals),
                                     0 if verts is None else verts.shape[0], _ptr(indices),
                                     0 if indices is None else indices.shape[0], C.byref(nv) if sync else None,
                                     C.byref(nt) if sync else None)
    _check(ctx, rc, allow=(SPH_E_CAPACITY,))
    return (int(nv.value), int(nt.value)) if sync else None


def mc_extract_indexed(ctx, mc, verts, normals, indices, phi=None, stream=None, sync=True):
    """N3: S14 then the indexed mesh (see mc_polygonise_indexed)."""
    m = _fill(McParams, mc)
    nv, nt = _u32(0), _u32(0)
    rc = lib().mc_extract_indexed(ctx, C.byref(m), _stream(stream), _ptr(phi), _ptr(verts), _ptr(normals),
                                  0 if verts is None else verts.shape[0], _ptr(indices),
                                  0 if indices is None else indices.shape[0], C.byref(nv) if sync else None,
                                  C.byref(nt) if sync else None)
    _check(ctx, rc, allow=(SPH_E_CAPACITY,))
    return (int(nv.value), int(nt.value)) if sync else None


def mc_mesh_components(ctx, indices, n_tris, n_verts, label, stream=None, sync=True):
    """N3 connectivity: label[v] = smallest vertex id of v's component; returns (n_components, largest_tris)."""
    nc, big = _u32(0), _u32(0)
    rc = lib().mc_mesh_components(ctx, _ptr(indices), int(n_tris), int(n_verts), _stream(stream), _ptr(label),
                                  C.byref(nc) if sync else None, C.byref(big) if sync else None)
    _check(ctx, rc)
    return (int(nc.value), int(big.value)) if sync else None


def sph_simulate_host(ctx, pos, vel, bpos=None, bvel=None, boid=None, steps=1, mc=None, tris=None):
    """HOST arrays (numpy / pinned CPU tensors) in and out; returns the required triangle count."""
    nb = 0 if bpos is None else bpos.shape[0]
    bp = _fill(BoidParams, boid) if nb else None
    m = _fill(McParams, mc) if mc is not None else None
    nt = _u32(0)
    cap = 0 if tris is None else tris.shape[0]
    rc = lib().sph_simulate_host(ctx, _hptr(pos), _hptr(vel), pos.shape[0], _hptr(bpos) if nb else None,
                                 _hptr(bvel) if nb else None, nb, C.byref(bp) if nb else None, steps,
                                 C.byref(m) if m is not None else None, _hptr(tris), cap, C.byref(nt))
    _check(ctx, rc, allow=(SPH_E_CAPACITY,))
    return int(nt.value)
