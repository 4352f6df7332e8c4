"""Parity of S14-S17 (voxel SDF, marching cubes) against the oracle.

Stage-isolated (oracle phi fed to the CUDA polygoniser): triangle count, order and vertices bit-exact.
phi itself: |d| <= 1e-5 h; vertices of the end-to-end mesh: |d| <= 4e-5 h.  End to end: counts may differ only at cubes that touch a corner whose
|phi - iso| is below the phi tolerance; those are counted and must be few.
"""
import numpy as np
import pytest
import torch

from oracle import refbind as R
from paper_2311_15088_b200 import binding as B
from paper_2311_15088_b200 import workloads as W
from tests.gpuutil import Sim, dev, host_u32

pytestmark = pytest.mark.gpu


def _polygonise_gpu(sim, mp, phi_np, capacity):
    tris = torch.zeros(max(capacity, 1), 3, 3, device="cuda")
    nt = B.mc_polygonise(sim.ctx, mp, dev(phi_np), tris)
    return tris.cpu().numpy()[:min(nt, capacity)], nt


@pytest.mark.parametrize("idx,scale", [(1, None), (2, None), (3, 2), (4, 4), (5, 4)])
def test_sdf_and_polygonise_on_configs(idx, scale):
    cfg = W.config(idx, scale=scale)
    mp = W.mc_params(cfg)
    G, h = mp["n_point_per_axis"], cfg["sph"]["h"]
    phi_ref = R.voxel_sdf(cfg["sph"], mp, cfg["pos"])
    tris_ref, nt_ref, _ = R.mc_polygonise(mp, phi_ref)
    with Sim(cfg, G=G) as sim:
        B.sph_build_grid(sim.ctx, dev(cfg["pos"]))
        phi = torch.zeros(G ** 3, device="cuda")
        B.mc_voxel_sdf(sim.ctx, mp, phi)
        phi_gpu = phi.cpu().numpy()
        assert np.abs(phi_gpu - phi_ref).max() <= 1e-5 * h
        # stage-isolated: bit-exact
        tris, nt = _polygonise_gpu(sim, mp, phi_ref, nt_ref + 7)
        assert nt == nt_ref and nt > 0
        assert np.array_equal(tris, tris_ref)
        # end to end through mc_extract (library scratch phi)
        buf = torch.zeros(nt_ref + 1000, 3, 3, device="cuda")
        nt2 = B.mc_extract(sim.ctx, mp, buf)
        risky = np.abs(phi_ref - mp["iso"]) <= 1e-5 * h
        assert abs(nt2 - nt_ref) <= 5 * 8 * int(risky.sum())
        if not risky.any():
            # a vertex moves by d(phi) / |phi_b - phi_a| of an edge: with |grad phi| ~ 1 at the surface that is the phi
            # tolerance itself; 4x leaves room for crossing edges where phi is flatter
            assert nt2 == nt_ref and np.abs(buf.cpu().numpy()[:nt2] - tris_ref).max() <= 4e-5 * h


@pytest.mark.parametrize("rho,rfac,G", [(4.3, 1.0, 70), (3.0, 1.0, 61), (2.49, 1.0, 50), (2.0, 1.0, 40), (5.0, 1.7, 64),
                                         (1.0, 1.0, 24), (8.5, 0.6, 90)])
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_sdf_group_and_scalar_kernels_any_spacing(rho, rfac, G, variant):
    # voxel grids finer / coarser than the particle cells (rho = corners per cell and axis), search radius below and
    # above h (reach 1 and 2), a voxel grid that sticks out of the particle box on every side, and particles that
    # start outside the box (they sit in the clamped boundary cells): the walk must still find every neighbour
    sp = dict(W.config(1)["sph"], h=0.05, box_max=(0.6, 0.5, 0.4))
    h = sp["h"]
    pos = W.random_cloud(6000, (-0.04, -0.03, -0.02), (0.45, 0.42, 0.38), seed=int(rho * 10))
    spacing = h / rho
    ext = spacing * (G - 1)
    mp = dict(origin=(0.2 - 0.5 * ext, 0.2 - 0.5 * ext, 0.2 - 0.5 * ext), spacing=float(np.float32(spacing)),
              n_point_per_axis=G, radius=rfac * h, particle_radius=0.4 * h, iso=0.0)
    phi_ref = R.voxel_sdf(sp, mp, pos)
    with Sim(dict(sph=sp, n=pos.shape[0]), G=G) as sim:
        B.sph_build_grid(sim.ctx, dev(pos))
        phi = torch.full((G ** 3,), 123.0, device="cuda")
        B.mc_set_sdf_variant(sim.ctx, variant)  # 0 = cost model; 1 = per-corner walk, 2 = corner tiles
        B.mc_voxel_sdf(sim.ctx, mp, phi)
        err = np.abs(phi.cpu().numpy() - phi_ref)
        assert err.max() <= 1e-5 * h, (err.max() / h, int(err.argmax()))
        # corners with no neighbour carry exactly R - rbar (D:A-PHI0); the oracle agrees on which ones those are,
        # except where the only neighbours sit within rounding of r = R
        empty = np.float32(mp["radius"]) - np.float32(mp["particle_radius"])
        assert ((phi.cpu().numpy() == empty) != (phi_ref == empty)).sum() <= 5
        assert (phi_ref == empty).sum() > 0 and (phi_ref != empty).sum() > 0


def test_sdf_no_particles_and_far_grid():
    sp = W.config(1)["sph"]
    mp = dict(origin=(3.0, 3.0, 3.0), spacing=0.01, n_point_per_axis=40, radius=sp["h"], particle_radius=0.5 * sp["h"],
              iso=0.0)
    empty = np.float32(mp["radius"]) - np.float32(mp["particle_radius"])
    with Sim(dict(sph=sp, n=4096), G=40) as sim:
        phi = torch.zeros(40 ** 3, device="cuda")
        B.sph_build_grid(sim.ctx, None)  # n = 0
        B.mc_voxel_sdf(sim.ctx, mp, phi)
        assert bool((phi == float(empty)).all())
        phi.zero_()
        B.sph_build_grid(sim.ctx, dev(W.config(1)["pos"]))  # particles exist, but the voxel grid is far away
        B.mc_voxel_sdf(sim.ctx, mp, phi)
        assert bool((phi == float(empty)).all())
        phi.zero_()
        B.sph_build_grid(sim.ctx, None)  # back to n = 0: the bounding box must be empty again
        B.mc_voxel_sdf(sim.ctx, dict(mp, origin=(0.0, 0.0, 0.0)), phi)
        assert bool((phi == float(empty)).all())


def test_polygonise_random_noise_all_cases_ragged_tiles():
    # white noise: all 256 cases; G-1 = 22 -> 10648 cubes = 10 tiles + a ragged tail
    G = 23
    rng = np.random.default_rng(5)
    phi = rng.standard_normal(G ** 3).astype(np.float32)
    mp = dict(origin=(0.1, -0.2, 0.3), spacing=0.013, n_point_per_axis=G, radius=0.05, particle_radius=0.02, iso=0.1)
    tris_ref, nt_ref, cases = R.mc_polygonise(mp, phi, want_cases=True)
    assert len(np.unique(cases)) == 256
    cfg = dict(sph=W.config(1)["sph"], n=1)
    with Sim(cfg, G=G) as sim:
        tris, nt = _polygonise_gpu(sim, mp, phi, nt_ref)
        assert nt == nt_ref and np.array_equal(tris, tris_ref)
        # capacity smaller than needed: required count still reported, nothing past capacity written
        cap = nt_ref // 3
        buf = torch.full((cap + 50, 3, 3), -7.0, device="cuda")
        m = B._fill(B.McParams, mp)
        import ctypes as C
        got = C.c_uint32(0)
        rc = B.lib().mc_polygonise(sim.ctx, C.byref(m), C.c_void_p(dev(phi).data_ptr()), None,
                                   C.c_void_p(buf.data_ptr()), cap, C.byref(got), None)
        assert rc == B.SPH_E_CAPACITY and got.value == nt_ref
        out = buf.cpu().numpy()
        assert np.array_equal(out[:cap], tris_ref[:cap]) and np.all(out[cap:] == -7.0)


@pytest.mark.parametrize("G", [2, 3, 17, 33, 34, 130])
def test_polygonise_tiny_and_empty_grids(G):
    mp = dict(origin=(0.0, 0.0, 0.0), spacing=0.1, n_point_per_axis=G, radius=0.05, particle_radius=0.02, iso=0.0)
    cfg = dict(sph=W.config(1)["sph"], n=1)
    with Sim(cfg, G=G) as sim:
        phi = np.ones(G ** 3, np.float32)  # nothing below iso: zero triangles
        _, nt = _polygonise_gpu(sim, mp, phi, 4)
        assert nt == 0
        phi[0] = -1.0  # one corner below: exactly one triangle
        tris, nt = _polygonise_gpu(sim, mp, phi, 4)
        ref, nt_ref, _ = R.mc_polygonise(mp, phi)
        assert nt == nt_ref == 1 and np.array_equal(tris, ref)


def test_sdf_requires_fresh_grid_and_empty_space():
    cfg = W.config(1)
    mp = W.mc_params(cfg)
    G = mp["n_point_per_axis"]
    with Sim(cfg, G=G) as sim:
        phi = torch.zeros(G ** 3, device="cuda")
        with pytest.raises(B.SphError) as e:
            B.mc_voxel_sdf(sim.ctx, mp, phi)
        assert e.value.code == B.SPH_E_STALE_GRID
        pos, vel = dev(cfg["pos"]), dev(cfg["vel"])
        sim.step(pos, vel)
        with pytest.raises(B.SphError):  # positions moved since the grid was built
            B.mc_voxel_sdf(sim.ctx, mp, phi)
        B.sph_build_grid(sim.ctx, pos)
        B.mc_voxel_sdf(sim.ctx, mp, phi)
        far = phi.view(G, G, G)[G - 1, G - 1, G - 1].item()  # corner (1,1,1): no particle within R
        assert far == np.float32(mp["radius"]) - np.float32(mp["particle_radius"])


@pytest.mark.parametrize("idx", [4, 5])
def test_full_size_mc_config4_sampled(idx):
    # BASELINE.json's headline surface pass (1 048 576 particles, 256^3 corners) and the stress config (4 194 304
    # particles at 0.8 x spacing, 256^3 corners: the dense quadrant lists of the tile kernel): phi of the WHOLE field
    # against the oracle, the mesh of that phi bit for bit, and the fused mc_extract the same again
    cfg = W.config(idx)
    mp = W.mc_params(cfg)
    G, h = mp["n_point_per_axis"], cfg["sph"]["h"]
    with Sim(cfg, G=G) as sim:
        B.sph_build_grid(sim.ctx, dev(cfg["pos"]))
        phi = torch.zeros(G ** 3, device="cuda")
        B.mc_voxel_sdf(sim.ctx, mp, phi)
        phi_gpu = phi.cpu().numpy().reshape(G, G, G)
        # whole-field comparison is affordable on the oracle (16.7M corners): do it outright
        phi_ref = R.voxel_sdf(cfg["sph"], mp, cfg["pos"]).reshape(G, G, G)
        assert np.abs(phi_gpu - phi_ref).max() <= 1e-5 * h
        tris_ref, nt_ref, _ = R.mc_polygonise(mp, phi_gpu.reshape(-1))
        buf = torch.zeros(nt_ref + 10, 3, 3, device="cuda")
        nt = B.mc_polygonise(sim.ctx, mp, phi, buf)
        assert nt == nt_ref
        assert np.array_equal(buf.cpu().numpy()[:nt], tris_ref)
        # the fused path bench.py times (mc_extract: the SDF kernel writes the sign field, no k_mc_signs): same phi
        # bit for bit, hence the same mesh bit for bit
        buf2 = torch.zeros(nt_ref + 10, 3, 3, device="cuda")
        phi2 = torch.zeros(G ** 3, device="cuda")
        nt2 = B.mc_extract(sim.ctx, mp, buf2, phi=phi2)
        assert bool((phi2 == phi).all())
        assert nt2 == nt_ref and np.array_equal(buf2.cpu().numpy()[:nt2], tris_ref)


@pytest.mark.parametrize("idx,frames", [(2, 1000), (3, 100), (3, 400), (4, 60), (5, 20)])
def test_surface_of_an_evolved_state_at_full_size(idx, frames):
    """The surface pass on a state the simulation produced (the collapsed column / dam break after `frames` GPU frames:
    irregular spacing, a splashing free surface, boids inside), not on the initial lattice: phi of the whole field against
    the oracle on the same positions, the mesh of that phi bit for bit, and the fused mc_extract the same again."""
    cfg = W.config(idx)
    G, h = cfg["G"], cfg["sph"]["h"]
    with Sim(cfg, G=G) as sim:
        pos, vel, bpos, bvel = dev(cfg["pos"]), dev(cfg["vel"]), dev(cfg["bpos"]), dev(cfg["bvel"])
        for _ in range(frames):
            B.sph_step(sim.ctx, pos, vel, bpos, bvel, cfg["boid"])
            B.boid_step(sim.ctx, cfg["boid"], bpos, bvel)
        torch.cuda.synchronize()
        pos_np = pos.cpu().numpy()
        # it has moved (0.1 s of free fall: ~0.05; config 5's 20 frames: the compressed lattice pushes apart)
        assert np.isfinite(pos_np).all() and np.abs(pos_np[:, :3] - cfg["pos"][:, :3]).max() > (h if idx != 5 else 0.02 * h)
        mp = W.mc_params(cfg, pos_np)
        B.sph_build_grid(sim.ctx, pos, vel)
        phi = torch.zeros(G ** 3, device="cuda")
        buf = torch.zeros(4_000_000, 3, 3, device="cuda")
        nt = B.mc_extract(sim.ctx, mp, buf, phi=phi)
        phi_gpu = phi.cpu().numpy()
        phi_ref = R.voxel_sdf(cfg["sph"], mp, pos_np)
        assert np.abs(phi_gpu - phi_ref).max() <= 1e-5 * h
        tris_ref, nt_ref, _ = R.mc_polygonise(mp, phi_gpu)
        assert nt == nt_ref and nt > 1000
        assert np.array_equal(buf.cpu().numpy()[:nt], tris_ref)


# ---- N3: indexed mesh with per-vertex normals ------------------------------------------------------------------------
def _indexed_gpu(sim, mp, phi_np, vcap, tcap, with_normals=True):
    verts = torch.zeros(max(vcap, 1), 3, device="cuda")
    normals = torch.zeros(max(vcap, 1), 3, device="cuda") if with_normals else None
    idx = torch.zeros(max(tcap, 1), 3, dtype=torch.int32, device="cuda")
    nv, nt = B.mc_polygonise_indexed(sim.ctx, mp, dev(phi_np), verts, normals, idx)
    return (verts.cpu().numpy(), normals.cpu().numpy() if with_normals else None,
            idx.cpu().numpy().view(np.uint32), nv, nt)


@pytest.mark.parametrize("G,kind", [(23, "noise"), (33, "noise"), (40, "sphere"), (70, "sphere")])
def test_indexed_mesh_matches_oracle_stage_isolated(G, kind):
    # integers (vertex count, triangle count, every index) and vertex positions bit-exact; normals to 1e-5
    rng = np.random.default_rng(G)
    mp = dict(origin=(0.1, -0.2, 0.3), spacing=0.013, n_point_per_axis=G, radius=0.05, particle_radius=0.02,
              iso=0.1 if kind == "noise" else 0.0)
    if kind == "noise":
        phi = rng.standard_normal(G ** 3).astype(np.float32)
    else:
        k, j, i = np.meshgrid(np.arange(G), np.arange(G), np.arange(G), indexing="ij")
        x = np.stack([i, j, k], -1).reshape(-1, 3) * 0.013 + np.array(mp["origin"])
        c = np.array(mp["origin"]) + 0.013 * (G - 1) * np.array([0.5, 0.47, 0.52])
        phi = (np.linalg.norm(x - c, axis=1) - 0.013 * (G - 1) * 0.31).astype(np.float32)
    v_ref, n_ref, i_ref = R.mc_indexed(mp, phi)
    with Sim(dict(sph=W.config(1)["sph"], n=1), G=G) as sim:
        v, nrm, idx, nv, nt = _indexed_gpu(sim, mp, phi, v_ref.shape[0] + 5, i_ref.shape[0] + 5)
        assert nv == v_ref.shape[0] and nt == i_ref.shape[0] and nv > 0
        assert np.array_equal(idx[:nt], i_ref)
        assert np.array_equal(v[:nv], v_ref)
        assert np.abs(nrm[:nv] - n_ref).max() <= 1e-5
        # without normals, and with capacities that are too small: required counts reported, nothing past capacity
        v2, _, idx2, nv2, nt2 = _indexed_gpu(sim, mp, phi, nv, nt, with_normals=False)
        assert nv2 == nv and nt2 == nt and np.array_equal(v2[:nv], v_ref) and np.array_equal(idx2[:nt], i_ref)
        vcap, tcap = nv // 3, nt // 2
        verts = torch.full((vcap + 20, 3), -7.0, device="cuda")
        ind = torch.full((tcap + 20, 3), -7, dtype=torch.int32, device="cuda")
        import ctypes as C
        m = B._fill(B.McParams, mp)
        gv, gt = C.c_uint32(0), C.c_uint32(0)
        rc = B.lib().mc_polygonise_indexed(sim.ctx, C.byref(m), C.c_void_p(dev(phi).data_ptr()), None,
                                           C.c_void_p(verts.data_ptr()), None, vcap, C.c_void_p(ind.data_ptr()), tcap,
                                           C.byref(gv), C.byref(gt))
        assert rc == B.SPH_E_CAPACITY and gv.value == nv and gt.value == nt
        assert np.array_equal(verts.cpu().numpy()[:vcap], v_ref[:vcap]) and bool((verts[vcap:] == -7.0).all())
        assert np.array_equal(ind.cpu().numpy().view(np.uint32)[:tcap], i_ref[:tcap]) and bool((ind[tcap:] == -7).all())


def test_indexed_extract_on_config_matches_triangle_soup():
    # end to end on a fluid config: the indexed mesh expands to exactly the triangles mc_extract emits (same phi)
    cfg = W.config(2)
    mp = W.mc_params(cfg)
    G = mp["n_point_per_axis"]
    with Sim(cfg, G=G) as sim:
        B.sph_build_grid(sim.ctx, dev(cfg["pos"]))
        buf = torch.zeros(400000, 3, 3, device="cuda")
        phi = torch.zeros(G ** 3, device="cuda")
        nt = B.mc_extract(sim.ctx, mp, buf, phi=phi)
        verts = torch.zeros(3 * nt + 8, 3, device="cuda")
        normals = torch.zeros(3 * nt + 8, 3, device="cuda")
        idx = torch.zeros(nt + 8, 3, dtype=torch.int32, device="cuda")
        nv, nt2 = B.mc_extract_indexed(sim.ctx, mp, verts, normals, idx)
        assert nt2 == nt and 0 < nv < 3 * nt
        tri = verts.cpu().numpy()[idx.cpu().numpy()[:nt].astype(np.int64)]
        assert np.array_equal(tri, buf.cpu().numpy()[:nt])
        v_ref, n_ref, i_ref = R.mc_indexed(mp, phi.cpu().numpy())
        assert nv == v_ref.shape[0] and np.array_equal(idx.cpu().numpy().view(np.uint32)[:nt], i_ref)
        assert np.abs(normals.cpu().numpy()[:nv] - n_ref).max() <= 1e-5
        ln = np.linalg.norm(normals.cpu().numpy()[:nv].astype(np.float64), axis=1)
        assert np.abs(ln[ln > 0] - 1.0).max() < 1e-5


# ---- N3 connectivity (mc_mesh_components; reading D:A-CONNECT) -------------------------------------------------------
def _components(ctx, idx_np, n_verts):
    idx = dev(np.ascontiguousarray(idx_np, np.uint32).view(np.int32).reshape(-1, 3)) if len(idx_np) else None
    label = torch.full((max(n_verts, 1),), -3, dtype=torch.int32, device="cuda")
    nc, big = B.mc_mesh_components(ctx, idx, len(idx_np), n_verts, label)
    return host_u32(label)[:n_verts], nc, big


def test_mesh_components_match_oracle_on_synthetic_index_buffers():
    cfg = W.config(1)
    rng = np.random.default_rng(5)
    with Sim(cfg, G=8) as sim:
        cases = []
        for V, T in ((1, 0), (9, 0), (3, 1), (40, 9), (300, 120), (5000, 1700), (5000, 9000), (70001, 50021)):
            cases.append((rng.integers(0, V, size=(T, 3)).astype(np.uint32), V))
        # a long strip (the deepest trees a union-find can build), in order, reversed and shuffled
        strip = np.stack([np.arange(0, 200000), np.arange(1, 200001), np.arange(2, 200002)], 1).astype(np.uint32)
        cases += [(strip, 200002), (strip[::-1].copy(), 200002), (strip[rng.permutation(len(strip))], 200005)]
        # many small components: 30 000 triangles of their own, vertex ids scattered
        perm = rng.permutation(90000).astype(np.uint32)
        cases.append((perm.reshape(-1, 3), 90000))
        # scratch shrinks and grows between calls (context-owned, grows on demand)
        for idx, V in cases + cases[:4]:
            label, nc, big = _components(sim.ctx, idx, V)
            l_ref, nc_ref, big_ref = R.mesh_components(idx, V)
            assert (nc, big) == (nc_ref, big_ref)
            assert np.array_equal(label, l_ref)


def test_mesh_components_rejects_an_index_out_of_range():
    cfg = W.config(1)
    with Sim(cfg, G=8) as sim:
        idx = np.array([[0, 1, 2], [2, 3, 9]], np.uint32)
        with pytest.raises(Exception):
            _components(sim.ctx, idx, 9)
        label, nc, big = _components(sim.ctx, idx, 10)  # the context is usable afterwards
        assert (nc, big) == (6, 2) and label.tolist() == [0, 0, 0, 0, 4, 5, 6, 7, 8, 0]


def test_mesh_components_on_fluid_and_on_scattered_particles():
    # a fluid config: the mesh of mc_extract_indexed; then particles further apart than 2 R: one closed blob each
    cfg = W.config(2)
    mp = W.mc_params(cfg)
    G = mp["n_point_per_axis"]
    with Sim(cfg, G=G) as sim:
        B.sph_build_grid(sim.ctx, dev(cfg["pos"]))
        verts = torch.zeros(400000, 3, device="cuda")
        idx = torch.zeros(400000, 3, dtype=torch.int32, device="cuda")
        nv, nt = B.mc_extract_indexed(sim.ctx, mp, verts, None, idx)
        label = torch.zeros(nv, dtype=torch.int32, device="cuda")
        nc, big = B.mc_mesh_components(sim.ctx, idx, nt, nv, label)
        l_ref, nc_ref, big_ref = R.mesh_components(host_u32(idx)[:nt], nv)
        assert (nc, big) == (nc_ref, big_ref) and np.array_equal(host_u32(label), l_ref)
        assert 1 <= nc < nv and big <= nt
        # scattered: 64 lone particles ON voxel corners 16 spacings apart: phi = -rbar at that corner, > 0 at its six
        # neighbours, so every particle is an octahedron of 8 triangles on 6 vertices, connected to nothing else
        g = np.array([8, 24, 40, 56], np.float32) * np.float32(mp["spacing"])
        x, y, z = np.meshgrid(g, g, g, indexing="ij")
        pts = np.stack([x.ravel(), y.ravel(), z.ravel(), np.zeros(64, np.float32)], 1).astype(np.float32)
        B.sph_build_grid(sim.ctx, dev(pts))
        nv, nt = B.mc_extract_indexed(sim.ctx, mp, verts, None, idx)
        assert (nv, nt) == (64 * 6, 64 * 8)
        label = torch.zeros(nv, dtype=torch.int32, device="cuda")
        nc, big = B.mc_mesh_components(sim.ctx, idx, nt, nv, label)
        l_ref, nc_ref, big_ref = R.mesh_components(host_u32(idx)[:nt], nv)
        assert (nc, big) == (64, 8) == (nc_ref, big_ref) and np.array_equal(host_u32(label), l_ref)


# ---- cube ranges (mc_set_cube_range; the surface pass of the slab decomposition) ---------------------
def test_polygonise_cube_ranges_are_the_ordered_subsets_of_the_whole_mesh():
    # white noise on 70^3 corners (69 cubes per axis: segments of 32, 32 and 5 cubes).  The oracle gives every
    # triangle's cube (cube-major order, ntri[case] triangles each); a cube range must return exactly the triangles of
    # the cubes inside it, in the same order, bit for bit; a partition of an axis adds up to the whole mesh
    G = 70
    Q = G - 1
    rng = np.random.default_rng(17)
    phi = rng.standard_normal(G ** 3).astype(np.float32)
    mp = dict(origin=(0.1, -0.2, 0.3), spacing=0.013, n_point_per_axis=G, radius=0.05, particle_radius=0.02, iso=0.3)
    tris_ref, nt_ref, cases = R.mc_polygonise(mp, phi, want_cases=True)
    _, ntri, _ = R.mc_table()
    cube_of_tri = np.repeat(np.arange(Q ** 3), ntri[cases].astype(np.int64))
    assert cube_of_tri.shape[0] == nt_ref
    ci, cj, ck = cube_of_tri % Q, (cube_of_tri // Q) % Q, cube_of_tri // (Q * Q)
    coord = (ci, cj, ck)
    cfg = dict(sph=W.config(1)["sph"], n=1)
    with Sim(cfg, G=G) as sim:
        def run(ranges):
            B.mc_set_cube_range(sim.ctx, -1)
            keep = np.ones(nt_ref, bool)
            for axis, lo, hi in ranges:
                B.mc_set_cube_range(sim.ctx, axis, lo, hi)
                keep &= (coord[axis] >= lo) & (coord[axis] < hi)
            tris, nt = _polygonise_gpu(sim, mp, phi, nt_ref)
            assert nt == int(keep.sum()), ranges
            assert np.array_equal(tris[:nt], tris_ref[keep]), ranges
            return nt

        for ranges in ([(0, 0, 7)], [(0, 7, 40)], [(0, 31, 33)], [(0, 64, 1000)], [(0, 5, 5)], [(1, 3, 21)], [(2, 60, 69)],
                       [(0, 10, 50), (1, 0, 30), (2, 17, 18)], [(0, 33, 64), (2, 0, 0)]):
            run(ranges)
        for axis in range(3):  # a partition into four slabs adds up to the whole
            cuts = [0, 13, 32, 51, Q]
            assert sum(run([(axis, cuts[r], cuts[r + 1])]) for r in range(4)) == nt_ref
        B.mc_set_cube_range(sim.ctx, -1)
        tris, nt = _polygonise_gpu(sim, mp, phi, nt_ref)
        assert nt == nt_ref and np.array_equal(tris, tris_ref)
        with pytest.raises(B.SphError):
            B.mc_set_cube_range(sim.ctx, 0, 5, 4)
        with pytest.raises(B.SphError):
            B.mc_set_cube_range(sim.ctx, 3, 0, 4)


def test_extract_with_cube_ranges_on_the_tile_kernel_skips_tiles_but_not_triangles():
    # S14 -> S17 with the corner-tile kernel forced: under a cube range only the tiles holding corners of those cubes
    # are computed (the rest of phi keeps the NaN it was filled with), and the triangles are bit for bit the subset of
    # the unrestricted pass for those cubes
    from tests.slabutil import triangles_in_cube_range
    cfg = W.config(2)
    mp = W.mc_params(cfg)
    G = mp["n_point_per_axis"]
    Q = G - 1
    with Sim(cfg, G=G) as sim:
        B.mc_set_sdf_variant(sim.ctx, 2)
        B.sph_build_grid(sim.ctx, dev(cfg["pos"]))
        full = torch.zeros(400000, 3, 3, device="cuda")
        phi = torch.zeros(G ** 3, device="cuda")
        nt_full = B.mc_extract(sim.ctx, mp, full, phi=phi)
        phi_np = phi.cpu().numpy()
        t_ref, nt_ref, cases = R.mc_polygonise(mp, phi_np, want_cases=True)
        assert nt_ref == nt_full and np.array_equal(full.cpu().numpy()[:nt_full], t_ref)
        for ranges in ([(0, 10, 30)], [(1, 0, 9)], [(2, 50, 63)], [(0, 8, 16), (2, 4, 8)], [(0, 62, 63)], [(1, 7, 7)]):
            B.mc_set_cube_range(sim.ctx, -1)
            keep = np.ones(nt_full, bool)
            needed = np.ones((G, G, G), bool)  # [k, j, i]: corners of the cubes in range
            for axis, lo, hi in ranges:
                B.mc_set_cube_range(sim.ctx, axis, lo, hi)
                keep &= triangles_in_cube_range(mp, cases, axis, lo, hi)
                idx = np.arange(G)
                sel = (idx >= lo) & (idx <= hi) if hi > lo else np.zeros(G, bool)
                shape = [1, 1, 1]
                shape[2 - axis] = G
                needed &= sel.reshape(shape)
            part = torch.zeros(400000, 3, 3, device="cuda")
            phi2 = torch.full((G ** 3,), float("nan"), device="cuda")
            nt = B.mc_extract(sim.ctx, mp, part, phi=phi2)
            assert nt == int(keep.sum()), ranges
            assert np.array_equal(part.cpu().numpy()[:nt], t_ref[keep]), ranges
            p2 = phi2.cpu().numpy().reshape(G, G, G)
            written = ~np.isnan(p2)
            assert np.array_equal(p2[written], phi_np.reshape(G, G, G)[written])
            assert bool(written[needed].all()), ranges            # every corner a cube in range uses was computed
            assert written.sum() < G ** 3, ranges                 # and tiles outside the range were skipped
        B.mc_set_cube_range(sim.ctx, -1)
        again = torch.zeros(400000, 3, 3, device="cuda")
        assert B.mc_extract(sim.ctx, mp, again) == nt_full and bool((again[:nt_full] == full[:nt_full]).all())
