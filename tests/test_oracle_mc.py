"""Pins for the oracle's voxel SDF, generated marching-cubes table and polygoniser (S14-S17).  CPU only."""
import math
import os

import numpy as np
import pytest

from oracle import refbind as R
from tests import meshutil as M

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _sp(h=0.0625):
    return dict(box_min=(0.0, 0.0, 0.0), box_max=(1.0, 1.0, 1.0), h=h, rest_density=1000.0, mass=0.03,
                stiffness=3.0, viscosity=0.1, gravity=(0.0, -9.81, 0.0), dt=1e-3, wall_damping=0.5)


def _mp(G, origin=(0.0, 0.0, 0.0), spacing=None, R_=0.0625, rbar=0.03125, iso=0.0):
    return dict(origin=origin, spacing=spacing if spacing is not None else 1.0 / (G - 1), n_point_per_axis=G,
                radius=R_, particle_radius=rbar, iso=iso)


def _corners(mp):
    G = mp["n_point_per_axis"]
    k, j, i = np.meshgrid(np.arange(G), np.arange(G), np.arange(G), indexing="ij")
    o, s = np.float32(mp["origin"]), np.float32(mp["spacing"])
    return np.stack([o[0] + i.astype(np.float32) * s, o[1] + j.astype(np.float32) * s,
                     o[2] + k.astype(np.float32) * s], -1).reshape(-1, 3)


def test_sdf_single_particle_is_a_distance():
    # P:477 Eq. 48 with one neighbour: xbar = x1, so phi = |x - x1| - rbar inside R, and R - rbar outside (D:A-PHI0)
    mp = _mp(24, origin=(0.4, 0.4, 0.4), spacing=0.008)
    x1 = np.array([[0.4913, 0.5021, 0.4876, 0]], np.float32)
    phi = R.voxel_sdf(_sp(), mp, x1)
    d = np.linalg.norm(_corners(mp).astype(np.float64) - x1[0, :3].astype(np.float64), axis=1)
    inside = d < 0.0625 * (1 - 1e-6)
    outside = d > 0.0625 * (1 + 1e-6)
    assert inside.sum() > 1000 and outside.sum() > 1000
    assert np.allclose(phi[inside], d[inside] - 0.03125, atol=2e-7)
    assert np.all(phi[outside] == np.float32(0.0625 - 0.03125))


def test_sdf_symmetric_pair_and_brute_force():
    mp = _mp(9, origin=(0.5, 0.5, 0.5), spacing=0.0)  # every corner at the same point
    pts = np.array([[0.52, 0.5, 0.5, 0], [0.48, 0.5, 0.5, 0]], np.float32)
    phi = R.voxel_sdf(_sp(), mp, pts)
    assert np.allclose(phi, -0.03125, atol=1e-7)  # S1 = 0 -> phi = -rbar
    from paper_2311_15088_b200 import workloads as W
    cfg = W.config(1, scale=2)
    mp = _mp(20, spacing=0.3 / 19)
    a = R.voxel_sdf(cfg["sph"], mp, cfg["pos"])
    b = R.voxel_sdf(cfg["sph"], mp, cfg["pos"], brute=True)
    assert np.allclose(a, b, rtol=0, atol=1e-7)
    assert (a < 0).any() and (a > 0).any()


def _phi_at_one_corner(pts, x, R_, rbar, h=0.0625):
    """phi of the oracle at the single point x (a 2^3 voxel grid with spacing 0: every corner is x)."""
    mp = _mp(2, origin=tuple(float(v) for v in x), spacing=0.0, R_=R_, rbar=rbar)
    p4 = np.zeros((len(pts), 4), np.float32)
    p4[:, :3] = pts
    phi = R.voxel_sdf(_sp(h), mp, p4)
    assert np.all(phi == phi[0])
    return float(phi[0])


def test_sdf_weight_unequal_pair_closed_form():
    # P:477-487 (Eq. 48-50): two particles on a line through the corner x at UNEQUAL distances d1 (towards +x) and d2
    # (towards -x).  xbar - x = (k1 d1 - k2 d2)/(k1 + k2) along the line with k_i = (1 - d_i^2/R^2)^3, so
    # phi = |k1 d1 - k2 d2|/(k1 + k2) - rbar.  The weights do NOT cancel here: an exponent other than 3, or k(s) taken
    # as (1 - s)^3, moves phi by far more than the tolerance (checked below so the pin cannot go vacuous).
    Rn, rbar = 0.0625, 0.03125
    x = np.array([0.5, 0.5, 0.5], np.float32)
    for d1, d2 in ((0.05, 0.02), (0.01, 0.06), (0.031, 0.047), (0.0009765625, 0.0605)):
        pts = np.array([[0.5 + d1, 0.5, 0.5], [0.5 - d2, 0.5, 0.5]], np.float32)
        e1 = float(np.float64(pts[0, 0]) - np.float64(x[0]))      # the distances the float32 inputs really have
        e2 = float(np.float64(x[0]) - np.float64(pts[1, 0]))
        k1 = (1.0 - e1 * e1 / (Rn * Rn)) ** 3
        k2 = (1.0 - e2 * e2 / (Rn * Rn)) ** 3
        want = abs(k1 * e1 - k2 * e2) / (k1 + k2) - rbar
        got = _phi_at_one_corner(pts[:, :3], x, Rn, rbar)
        assert abs(got - want) < 2e-7, (d1, d2, got, want)
        # what plausible misreadings would give: each must be far from the closed form
        for kk in (lambda d: (1.0 - d * d / (Rn * Rn)) ** 2,      # exponent 2
                   lambda d: (1.0 - d / Rn) ** 3,                 # s where s^2 belongs
                   lambda d: 1.0 - d * d / (Rn * Rn),             # exponent 1
                   lambda d: 1.0):                                # unweighted mean
            wrong = abs(kk(e1) * e1 - kk(e2) * e2) / (kk(e1) + kk(e2)) - rbar
            assert abs(wrong - want) > 1e-5, (d1, d2)     # 50x the tolerance above


def test_sdf_weight_is_listing_9_written_out():
    # P:494-516 (Listing 9) evaluated exactly as printed, in numpy float64: loop 1 sums the kernel values
    # (weight_divisor), loop 2 forms w_i = k_i / sum k and the weighted mean position; phi = |x - xbar| - particle_size.
    # Also pins reading D:A-PHI (the oracle's one-pass |sum k (x_j - x)|/sum k is the two-loop form) and Eq. 50's
    # neighbourhood (only particles with |x - x_i| < R take part).
    rng = np.random.default_rng(5)
    Rn, rbar = 0.0625, 0.03125
    worst = 0.0
    for trial in range(40):
        npts = int(rng.integers(3, 9))
        x = (0.3 + 0.4 * rng.random(3)).astype(np.float32)
        d = rng.standard_normal((npts, 3))
        d *= (rng.random((npts, 1)) * 1.25 * Rn) / np.linalg.norm(d, axis=1, keepdims=True)   # some beyond R
        pts = (x.astype(np.float64) + d).astype(np.float32)
        cube_corner_pos = x.astype(np.float64)
        pp = pts.astype(np.float64)
        neigh = [p for p in pp if np.linalg.norm(cube_corner_pos - p) < Rn * (1 - 1e-6)]
        edge = [p for p in pp if abs(np.linalg.norm(cube_corner_pos - p) / Rn - 1) <= 1e-6]
        if edge or not neigh:
            continue
        kernel = lambda s: (1.0 - s * s) ** 3                                        # noqa: E731
        weight_divisor = 0.0
        for p in neigh:
            weight_divisor += kernel(np.linalg.norm(cube_corner_pos - p) / Rn)
        weight_multiplier = 1.0 / weight_divisor
        average_particle_pos = np.zeros(3)
        for p in neigh:
            weight_i = weight_multiplier * kernel(np.linalg.norm(cube_corner_pos - p) / Rn)
            average_particle_pos += weight_i * p
        want = np.linalg.norm(cube_corner_pos - average_particle_pos) - rbar
        got = _phi_at_one_corner(pts, x, Rn, rbar)
        worst = max(worst, abs(got - want))
        assert len(neigh) >= 1
    assert worst < 3e-7, worst


def test_sdf_weight_vanishes_continuously_at_R():
    # k(1) = 0, so a particle approaching the edge of the neighbourhood leaves the average continuously:
    # with a fixed particle at distance a on one side and a second at distance r -> R on the other side,
    # phi -> a - rbar, and the gap shrinks like k(r/R) ~ (2 (1 - r/R))^3 (the cube: exponent 3 and s^2 pinned again)
    Rn, rbar, a = 0.0625, 0.03125, 0.02
    x = np.array([0.5, 0.5, 0.5], np.float32)
    one = _phi_at_one_corner(np.array([[0.5 + a, 0.5, 0.5]], np.float32), x, Rn, rbar)
    gaps = []
    for eps in (0.08, 0.04, 0.02, 0.01):
        r = Rn * (1 - eps)
        pts = np.array([[0.5 + a, 0.5, 0.5], [0.5 - r, 0.5, 0.5]], np.float32)
        gaps.append(one - _phi_at_one_corner(pts, x, Rn, rbar))
    assert all(g > 0 for g in gaps) and gaps[-1] < 2e-6
    ratios = [gaps[i] / gaps[i + 1] for i in range(3)]
    # halving eps divides k by ~8 (exponent 3 of a simple zero of 1 - s^2); exponent 2 would give ~4, (1 - s)^3 also 8
    # but with k ~ eps^3 instead of (2 eps)^3: check the size too
    assert all(6.5 < q < 9.5 for q in ratios), ratios
    e = 0.01
    k2 = (1 - (1 - e) ** 2) ** 3
    k1 = (1 - (a / Rn) ** 2) ** 3
    want_gap = (a + Rn * (1 - e)) * k2 / (k1 + k2)
    assert abs(gaps[-1] / want_gap - 1) < 0.05
    # beyond R the particle is no neighbour at all
    pts = np.array([[0.5 + a, 0.5, 0.5], [0.5 - Rn * 1.001, 0.5, 0.5]], np.float32)
    assert _phi_at_one_corner(pts, x, Rn, rbar) == one


def test_table_worked_example_and_structure():
    tri, ntri, edge = R.mc_table()
    corners, edges = R.mc_numbering()
    # only corner 3 below the isolevel -> cube_index 8 -> edge_table[8] = 0x80c -> edges 2, 3, 11
    assert edge[8] == 0x80C and ntri[8] == 1 and sorted(tri[8][:3]) == [2, 3, 11] and tri[8][3] == -1
    assert {e for e in range(12) if 3 in edges[e]} == {2, 3, 11}
    assert ntri[0] == 0 and ntri[255] == 0 and edge[0] == 0 and edge[255] == 0
    for cs in range(256):
        below = [(cs >> n) & 1 for n in range(8)]
        crossed = {e for e in range(12) if below[edges[e][0]] != below[edges[e][1]]}
        used = {int(e) for e in tri[cs] if e >= 0}
        assert used == crossed, cs                                  # cover all sign-changing edges, and only them
        assert edge[cs] == sum(1 << e for e in crossed)
        n = ntri[cs]
        assert 0 <= n <= 5 and all(tri[cs][3 * n:] == -1) and all(tri[cs][:3 * n] >= 0)
        assert edge[cs] == edge[255 - cs]                            # complement has the same crossed edges
        # every triangle uses three distinct edges
        for t in range(n):
            assert len(set(tri[cs][3 * t:3 * t + 3])) == 3
    # a single corner below gives one triangle around it; its complement too
    for n in range(8):
        assert ntri[1 << n] == 1 and ntri[255 - (1 << n)] == 1


def test_table_matches_golden_counts():
    # tests/golden/mc_ntri.txt is written by tests/golden/make_golden.py from the oracle AFTER the pins here passed
    _, ntri, _ = R.mc_table()
    gold = np.loadtxt(os.path.join(GOLDEN, "mc_ntri.txt"), dtype=np.int64, comments="#")
    assert np.array_equal(gold.reshape(-1), ntri)


def _closed_field(G, seed, smooth):
    rng = np.random.default_rng(seed)
    f = rng.standard_normal((G, G, G))
    for _ in range(smooth):
        f = (f + np.roll(f, 1, 0) + np.roll(f, 1, 1) + np.roll(f, 1, 2)) / 4.0
    f = f - np.median(f)
    f[0], f[-1], f[:, 0], f[:, -1], f[:, :, 0], f[:, :, -1] = (1.0,) * 6  # outside everywhere on the boundary
    return f.astype(np.float32).reshape(-1)


@pytest.mark.parametrize("seed,smooth", [(0, 0), (1, 0), (2, 1), (3, 3)])
def test_random_fields_give_closed_consistently_oriented_meshes(seed, smooth):
    # white noise exercises all 256 cases and every pair of face-adjacent cases, ambiguous faces included:
    # crack-free <=> every mesh edge is shared by exactly two triangles, traversed once in each direction
    G = 14
    phi = _closed_field(G, seed, smooth)
    mp = _mp(G)
    tris, nt, cases = R.mc_polygonise(mp, phi, want_cases=True)
    assert nt == len(tris) and nt > 100
    if smooth == 0:
        assert len(np.unique(cases)) > 250
    ids, _ = M.weld(tris)
    _, ok, degenerate = M.edge_stats(ids)
    assert degenerate == 0
    assert ok
    # triangle count = sum over cubes of ntri[case]; order = cube-major (D:A-APPEND)
    _, ntri, _ = R.mc_table()
    assert nt == int(ntri[cases].sum())
    # volume enclosed (normals point to the >= iso side) is positive and below the grid volume
    _, vol, _ = M.area_volume(tris)
    assert 0 < vol < 1.0


@pytest.mark.parametrize("G,tol_area", [(32, 0.01), (64, 0.003)])
def test_sphere_isosurface(G, tol_area):
    # north_star pin: watertight sphere, area close to 4 pi r^2 (r = 10 voxels at G = 32)
    mp = _mp(G)
    c = np.array([0.5, 0.5, 0.5]) + 0.37 / (G - 1)
    r = 10.0 / 31.0
    x = _corners(mp).astype(np.float64)
    phi = (np.linalg.norm(x - c, axis=1) - r).astype(np.float32)
    tris, nt, _ = R.mc_polygonise(mp, phi)
    ids, nv = M.weld(tris)
    ne, ok, degenerate = M.edge_stats(ids)
    assert ok and degenerate == 0
    assert nv - ne + nt == 2                                     # Euler characteristic of a sphere
    area, vol, normals = M.area_volume(tris)
    assert abs(area / (4 * math.pi * r * r) - 1) < tol_area
    assert abs(vol / (4 / 3 * math.pi * r ** 3) - 1) < 2 * tol_area
    centroid = tris.astype(np.float64).mean(1)
    assert np.all(np.einsum("ij,ij->i", normals, centroid - c) > 0)  # outward
    # vertices lie on the sphere to O(spacing^2) (Eq. 51 linear interpolation)
    v = tris.reshape(-1, 3).astype(np.float64)
    assert np.abs(np.linalg.norm(v - c, axis=1) - r).max() < 0.6 * mp["spacing"] ** 2 / r + 1e-6


def test_capacity_is_respected():
    mp = _mp(16)
    x = _corners(mp).astype(np.float64)
    phi = (np.linalg.norm(x - 0.5, axis=1) - 0.3).astype(np.float32)
    full, nt, _ = R.mc_polygonise(mp, phi)
    part, nt2, _ = R.mc_polygonise(mp, phi, capacity=nt // 2)
    assert nt2 == nt and len(part) == nt // 2 and np.array_equal(part, full[:nt // 2])


def test_single_particle_through_sdf_and_mc_gives_sphere_of_radius_rbar():
    h = 0.0625
    G = 40
    mp = _mp(G, origin=(0.45, 0.45, 0.45), spacing=0.1 / (G - 1))
    x1 = np.array([[0.5003, 0.4991, 0.5007, 0]], np.float32)
    phi = R.voxel_sdf(_sp(h), mp, x1)
    tris, nt, _ = R.mc_polygonise(mp, phi)
    ids, nv = M.weld(tris)
    ne, ok, _ = M.edge_stats(ids)
    assert ok and nv - ne + nt == 2
    v = tris.reshape(-1, 3).astype(np.float64)
    # linear interpolation (Eq. 51) of a distance function along an edge errs by at most spacing^2 / (8 r)
    assert np.abs(np.linalg.norm(v - x1[0, :3], axis=1) - 0.5 * h).max() < 1.1 * mp["spacing"] ** 2 / (8 * 0.5 * h)


# ---- N3: indexed mesh with per-vertex normals (D:A-NORMAL, D:A-WELD) ------------------------------------------------
def _sphere_phi(mp, c, r):
    x = _corners(mp).astype(np.float64)
    return (np.linalg.norm(x - np.asarray(c), axis=1) - r).astype(np.float32)


def test_indexed_mesh_expands_to_the_triangle_soup_bitwise():
    # the welded mesh is the same mesh: verts[indices] == ref_mc_polygonise's triangles, bit for bit, on white noise
    # (all 256 cases) and on a sphere; and welding by bitwise vertex equality (meshutil) finds the same vertex count
    rng = np.random.default_rng(3)
    G = 14
    mp = _mp(G, origin=(0.1, -0.2, 0.3), spacing=0.013, iso=0.1)
    mp0 = dict(mp, iso=0.0)
    for mp, phi in ((mp, rng.standard_normal(G ** 3).astype(np.float32)), (mp0, _sphere_phi(mp0, (0.18, -0.12, 0.39), 0.055))):
        tris, nt, _ = R.mc_polygonise(mp, phi)
        verts, normals, idx = R.mc_indexed(mp, phi)
        assert idx.shape[0] == nt and nt > 0
        assert np.array_equal(verts[idx.astype(np.int64)], tris)
        # every vertex is used, and its id order is the ascending edge key (x-fastest point order, then axis)
        assert np.array_equal(np.unique(idx), np.arange(verts.shape[0]))
    ids, nv = M.weld(tris)  # sphere: no two crossing edges share a position, so bitwise welding agrees
    assert nv == verts.shape[0]


def test_indexed_sphere_is_a_closed_surface_by_index_and_normals_point_outwards():
    G = 40
    mp = _mp(G)
    c, r = (0.5, 0.52, 0.47), 0.3
    phi = _sphere_phi(mp, c, r)
    verts, normals, idx = R.mc_indexed(mp, phi)
    V, F = verts.shape[0], idx.shape[0]
    E, closed, degenerate = M.edge_stats(idx.astype(np.int64))
    assert closed and degenerate == 0
    assert V - E + F == 2  # Euler characteristic of a sphere, now on the index buffer itself
    # normals: unit length, within 2 degrees of the radial direction (central differences are O(spacing^2) accurate)
    radial = verts.astype(np.float64) - np.asarray(c)
    radial /= np.linalg.norm(radial, axis=1, keepdims=True)
    assert np.abs(np.linalg.norm(normals.astype(np.float64), axis=1) - 1.0).max() < 1e-6
    assert (np.einsum("ij,ij->i", normals.astype(np.float64), radial)).min() > math.cos(math.radians(2.0))
    # vertex ids ascend with the edge key 3 * (lower corner) + axis: recover corner and axis from the position (the
    # coordinate along the edge is the one off the lattice; the other two sit on it)
    t = (verts.astype(np.float64) - np.float64(mp["origin"])) / float(np.float32(mp["spacing"]))
    frac = np.abs(t - np.round(t))
    axis = np.argmax(frac, axis=1)
    cell = np.round(t).astype(np.int64)
    rows = np.arange(len(t))
    cell[rows, axis] = np.floor(t[rows, axis]).astype(np.int64)
    key = 3 * (cell[:, 0] + G * (cell[:, 1] + G * cell[:, 2])) + axis
    on_lattice = frac.max(axis=1) < 1e-4  # a vertex that coincides with a corner has no recoverable axis
    assert on_lattice.mean() < 0.01
    k = key[~on_lattice]
    assert np.all(np.diff(k) > 0)


def test_indexed_plane_normals_are_exact_and_border_is_one_sided():
    # phi = z - z0 is linear: central and one-sided differences are exact up to rounding, the normal is (0, 0, 1);
    # the plane z0 sits in the LAST layer of cubes, so the upper corners use the one-sided border formula
    G = 9
    mp = _mp(G, spacing=0.125)
    z0 = 0.125 * (G - 2) + 0.05
    x = _corners(mp).astype(np.float64)
    phi = (x[:, 2] - z0).astype(np.float32)
    verts, normals, idx = R.mc_indexed(mp, phi)
    assert verts.shape[0] == G * G and idx.shape[0] == 2 * (G - 1) ** 2
    assert np.abs(verts[:, 2] - z0).max() < 1e-6
    assert np.abs(normals - np.array([0, 0, 1], np.float32)).max() < 1e-6
    # flipped sign: fluid above the plane, normals point down
    v2, n2, _ = R.mc_indexed(mp, -phi)
    assert np.array_equal(v2, verts) and np.abs(n2 - np.array([0, 0, -1], np.float32)).max() < 1e-6


# ---- N3 connectivity (Table 2 last column; reading D:A-CONNECT) -----------------------------------------------
def test_mesh_components_match_scipy_on_random_triangle_sets():
    # a library routine as the pin: components of the graph with an edge between the vertices of every triangle
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    rng = np.random.default_rng(11)
    for V, T in ((1, 0), (7, 0), (3, 1), (40, 9), (300, 120), (5000, 1700), (5000, 9000)):
        idx = rng.integers(0, V, size=(T, 3)).astype(np.uint32)  # degenerate triangles (repeated ids) included
        label, nc, big = R.mesh_components(idx, V)
        i = idx.astype(np.int64)
        rows = np.concatenate([i[:, 0], i[:, 0]]) if T else np.zeros(0, np.int64)
        cols = np.concatenate([i[:, 1], i[:, 2]]) if T else np.zeros(0, np.int64)
        g = coo_matrix((np.ones(rows.size), (rows, cols)), shape=(V, V))
        n_ref, lab_ref = connected_components(g, directed=False)
        assert nc == n_ref
        # same partition, and the label is the smallest vertex id of the part
        smallest = np.full(n_ref, V, np.int64)
        np.minimum.at(smallest, lab_ref, np.arange(V))
        assert np.array_equal(label.astype(np.int64), smallest[lab_ref])
        per = np.bincount(lab_ref[i[:, 0]], minlength=n_ref) if T else np.zeros(1, np.int64)
        assert big == per.max()


def test_mesh_components_hand_made_chain_and_vertex_only_contact():
    # a strip of triangles sharing edges, one triangle touching it in a single vertex (connected, D:A-CONNECT),
    # one apart, one unused vertex
    idx = np.array([[0, 1, 2], [1, 2, 3], [2, 3, 4], [4, 5, 6], [8, 9, 10]], np.uint32)
    label, nc, big = R.mesh_components(idx, 11)
    assert label.tolist() == [0, 0, 0, 0, 0, 0, 0, 7, 8, 8, 8]
    assert nc == 3 and big == 4
    # relabelling the vertices changes the labels, not the partition sizes
    perm = np.random.default_rng(0).permutation(11).astype(np.uint32)
    _, nc2, big2 = R.mesh_components(perm[idx], 11)
    assert (nc2, big2) == (3, 4)


def test_mesh_components_of_separated_spheres():
    # k spheres further apart than a cube: k closed components with the triangle counts of the spheres extracted one
    # by one; one sphere: a single component holding 100 % of the triangles
    G = 36
    mp = _mp(G)
    centres = [(0.25, 0.25, 0.25), (0.72, 0.3, 0.3), (0.3, 0.74, 0.66), (0.7, 0.7, 0.72)]
    radii = [0.15, 0.12, 0.17, 0.1]
    each = [_sphere_phi(mp, c, r) for c, r in zip(centres, radii)]
    counts = []
    for phi in each:
        _, _, idx = R.mc_indexed(mp, phi)
        label, nc, big = R.mesh_components(idx, int(idx.max()) + 1)
        assert nc == 1 and big == idx.shape[0] and not label.any()
        counts.append(idx.shape[0])
    verts, _, idx = R.mc_indexed(mp, np.minimum.reduce(each))  # union of the spheres
    label, nc, big = R.mesh_components(idx, verts.shape[0])
    assert nc == 4 and idx.shape[0] == sum(counts) and big == max(counts)
    per = np.bincount(label[idx[:, 0].astype(np.int64)], minlength=verts.shape[0])
    assert sorted(per[per > 0].tolist()) == sorted(counts)
