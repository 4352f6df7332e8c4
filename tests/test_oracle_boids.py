"""Pins for the oracle's boid rules and SPH<->boid coupling (S7, S9, S11-S13).  CPU only.

The coupling READING (D:C-COUPLE) is ours, so beyond these invariants it stays "parity unpinned".
"""
import numpy as np

from oracle import refbind as R
from paper_2311_15088_b200 import workloads as W


def _cfg():
    return W.config(1)


def _far_fluid():
    # one fluid particle far from everything, so that boid rules can be looked at alone
    pos = np.array([[0.05, 0.05, 0.05, 0]], np.float32)
    return pos, np.zeros_like(pos), np.array([195.8], np.float32)


def test_two_boids_by_hand():
    cfg = _cfg()
    sp, bp = cfg["sph"], dict(cfg["boid"], protect_range=0.1, visible_range=0.2, w_sep=1.5, w_ali=0.7, w_coh=0.3)
    pos, vel, rho = _far_fluid()
    bpos = np.array([[0.5, 0.5, 0.5, 0], [0.56, 0.5, 0.5, 0]], np.float32)
    bvel = np.array([[0.1, 0.0, 0.0, 0], [0.0, 0.2, 0.0, 0]], np.float32)
    out = R.boid_step(sp, bp, pos, vel, rho, bpos, bvel)
    d = bpos[0, :3].astype(np.float64) - bpos[1, :3].astype(np.float64)
    dist = np.linalg.norm(d)
    sep = 1.5 * (1.0 - dist / 0.1) * d                      # P:284-291 with D:C-SEP
    vbar = 0.5 * (bvel[0, :3] + bvel[1, :3]).astype(np.float64)  # means include the boid itself (D:C-ALI)
    pbar = 0.5 * (bpos[0, :3] + bpos[1, :3]).astype(np.float64)
    ali = 0.7 * (vbar - bvel[0, :3])
    coh = 0.3 * (pbar - bpos[0, :3])
    parts = out["dv_parts"][0]
    assert np.allclose(parts[0, :3], sep, rtol=1e-5, atol=1e-9)
    assert np.allclose(parts[1, :3], ali, rtol=1e-5, atol=1e-9)
    assert np.allclose(parts[2, :3], coh, rtol=1e-5, atol=1e-9)
    assert not parts[3, :3].any()
    v_new = bvel[0, :3] + sep + ali + coh
    assert np.allclose(out["bvel"][0, :3], v_new, rtol=1e-5)
    assert np.allclose(out["bpos"][0, :3], bpos[0, :3] + 1e-3 * v_new, rtol=1e-6)
    # the second boid gets the mirrored separation
    assert np.allclose(out["dv_parts"][1, 0, :3], -sep, rtol=1e-5, atol=1e-9)


def test_lone_boid_and_speed_limits_and_edges():
    cfg = _cfg()
    sp = cfg["sph"]
    pos, vel, rho = _far_fluid()
    bp = dict(cfg["boid"], max_speed=0.5, min_speed=0.2)
    bpos = np.array([[0.5, 0.5, 0.5, 0]], np.float32)
    out = R.boid_step(sp, bp, pos, vel, rho, bpos, np.array([[0.3, 0.0, 0.0, 0]], np.float32))
    assert not out["dv_parts"][0, :3, :3].any()      # self-inclusive means: ali = coh = 0 exactly
    assert np.allclose(out["bvel"][0, :3], [0.3, 0, 0])
    out = R.boid_step(sp, bp, pos, vel, rho, bpos, np.array([[3.0, 4.0, 0.0, 0]], np.float32))
    assert np.allclose(out["bvel"][0, :3], [0.3, 0.4, 0.0], rtol=1e-6)  # scaled to max_speed (D:C-SPEED)
    out = R.boid_step(sp, bp, pos, vel, rho, bpos, np.array([[0.0, 0.03, 0.04, 0]], np.float32))
    assert np.allclose(out["bvel"][0, :3], [0.0, 0.12, 0.16], rtol=1e-6)  # scaled up to min_speed
    out = R.boid_step(sp, bp, pos, vel, rho, bpos, np.zeros((1, 4), np.float32))
    assert not out["bvel"][0, :3].any()                 # |v| = 0 untouched
    # edge rule (D:C-EDGE): outside the Boid Space -> turn back by edge_turn on that axis
    out_b = np.array([[1.2, -0.1, 0.5, 0]], np.float32)
    out = R.boid_step(sp, dict(bp, min_speed=0.0), pos, vel, rho, out_b, np.zeros((1, 4), np.float32))
    assert np.allclose(out["bvel"][0, :3], [-0.05, 0.05, 0.0])


def test_boid_grid_equals_brute_force_and_speed_cap():
    cfg = W.config(3, scale=8)  # boids inside the fluid column, push radius 2h (125-cell gather)
    out = R.step(cfg["sph"], cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"], cfg["boid"])
    g = R.boid_step(cfg["sph"], cfg["boid"], cfg["pos"], cfg["vel"], out["density"], cfg["bpos"], cfg["bvel"])
    b = R.boid_step(cfg["sph"], cfg["boid"], cfg["pos"], cfg["vel"], out["density"], cfg["bpos"], cfg["bvel"],
                    brute=True)
    assert np.allclose(g["bvel"], b["bvel"], rtol=1e-6, atol=1e-9)
    assert np.allclose(g["dv_parts"], b["dv_parts"], rtol=1e-6, atol=1e-9)
    assert np.abs(g["dv_parts"][:, 3]).max() > 0  # the fluid really pushes these boids
    speed = np.linalg.norm(g["bvel"][:, :3], axis=1)
    assert speed.max() <= 0.5 * (1 + 1e-6)
    # same for the particle side: touched / push identical under brute force
    ob = R.step(cfg["sph"], cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"], cfg["boid"], brute=True)
    assert np.array_equal(out["touched"], ob["touched"]) and out["touched"].max() > 0
    assert np.allclose(out["accel"], ob["accel"], rtol=1e-6, atol=1e-7)


def test_coupling_is_local():
    cfg = _cfg()  # boids in [0.6,0.9]^3, fluid in [0,0.5]^3, push radius h = 0.0625: out of reach
    with_b = R.step(cfg["sph"], cfg["pos"], cfg["vel"], cfg["bpos"], cfg["bvel"], cfg["boid"])
    without = R.step(cfg["sph"], cfg["pos"], cfg["vel"])
    assert not with_b["touched"].any()
    assert np.array_equal(with_b["accel"], without["accel"])
    out = R.boid_step(cfg["sph"], cfg["boid"], cfg["pos"], cfg["vel"], with_b["density"], cfg["bpos"], cfg["bvel"])
    assert not out["dv_parts"][:, 3].any()


def test_one_particle_one_boid_antisymmetry():
    cfg = _cfg()
    sp = dict(cfg["sph"], gravity=(0.0, 0.0, 0.0))
    bp = dict(cfg["boid"], push_radius=0.1, w_push=1.0, sph_factor=1.0, w_sep=0.0, w_ali=0.0, w_coh=0.0)
    pos = np.array([[0.5, 0.5, 0.5, 0]], np.float32)
    vel = np.array([[0.1, 0.0, -0.2, 0]], np.float32)
    bpos = np.array([[0.53, 0.52, 0.49, 0]], np.float32)
    bvel = np.array([[-0.2, 0.1, 0.0, 0]], np.float32)
    s = R.step(sp, pos, vel, bpos, bvel, bp)
    assert s["touched"][0] == 1
    b = R.boid_step(sp, bp, pos, vel, s["density"], bpos, bvel)
    a_fluid = s["accel"][0, :3].astype(np.float64)                 # = w_push * B_i / rho_i (no fluid neighbours)
    A_b = b["dv_parts"][0, 3, :3].astype(np.float64) / sp["dt"]    # dv_fluid = sph_factor * dt * A_b
    assert np.linalg.norm(a_fluid) > 0
    assert np.allclose(a_fluid, -A_b, rtol=2e-5)                   # equal masses: action = -reaction
    # probe density of the boid (D:C-COUPLE): own parcel + the one fluid particle within h
    h, m = sp["h"], sp["mass"]
    r = np.linalg.norm(pos[0, :3].astype(np.float64) - bpos[0, :3].astype(np.float64))
    rho_b = R.boid_density(sp, pos, bpos)
    assert np.allclose(rho_b[0], m * (R.w_poly6(0, h) + R.w_poly6(r, h)), rtol=1e-6)


# ---- N4: obstacle avoidance (P:261, P:336 step 7; reading D:C-OBST: parity unpinned beyond these invariants) --------
def _one_cell_grid(normal, cell=0.1, dims=(5, 5, 5), which=(2, 2, 2), w_obs=0.25, heavy=3.0):
    op = dict(origin=(0.0, 0.0, 0.0), cell=cell, dims=dims, w_obs=w_obs, heavy=heavy)
    normals = np.zeros((int(np.prod(dims)), 4), np.float32)
    normals[which[0] + dims[0] * (which[1] + dims[1] * which[2]), :3] = normal
    centre = (np.array(which) + 0.5) * cell
    return op, normals, centre


def test_obstacle_single_cell_hand_values():
    # one cell with normal n at centre x_c: inside the protection range the boid gets w * heavy * n, between the protection
    # and the visual range w * n, beyond the visual range nothing; the position is untouched (step 7 follows step 6)
    n = np.array([0.6, -0.8, 0.0], np.float32)
    op, normals, xc = _one_cell_grid(n)
    protect, visible = 0.05, 0.12
    bpos = np.zeros((4, 4), np.float32)
    bpos[0, :3] = xc + [0.03, 0.0, 0.0]    # inside protect
    bpos[1, :3] = xc + [0.0, 0.08, 0.0]    # between protect and visible
    bpos[2, :3] = xc + [0.0, 0.0, 0.13]    # outside visible
    bpos[3, :3] = xc + [0.12, 0.0, 0.0]    # exactly at the visible range: strict '<', nothing
    bvel = np.tile(np.array([0.1, 0.2, 0.3, 7.0], np.float32), (4, 1))
    out = R.boid_obstacles(op, normals, protect, visible, bpos, bvel)
    w, hv = np.float32(0.25), np.float32(3.0)
    assert np.allclose(out[0, :3], bvel[0, :3] + w * hv * n, atol=1e-7)
    assert np.allclose(out[1, :3], bvel[1, :3] + w * n, atol=1e-7)
    assert np.array_equal(out[2], bvel[2]) and np.array_equal(out[3], bvel[3])
    assert np.array_equal(out[:, 3], bvel[:, 3])  # payload lane carried through


def test_obstacle_zero_grid_is_identity_and_range_walk_equals_all_cells():
    from paper_2311_15088_b200 import workloads as W
    rng = np.random.default_rng(4)
    bpos = np.zeros((300, 4), np.float32)
    bpos[:, :3] = rng.uniform(-0.1, 1.1, (300, 3))  # some boids outside the grid
    bvel = rng.uniform(-0.2, 0.2, (300, 4)).astype(np.float32)
    op, normals = W.sphere_obstacle((0, 0, 0), (1, 1, 1), 0.05, (0.5, 0.45, 0.55), 0.25)
    assert np.array_equal(R.boid_obstacles(op, np.zeros_like(normals), 0.05, 0.1, bpos, bvel), bvel)
    a = R.boid_obstacles(op, normals, 0.06, 0.13, bpos, bvel)
    b = R.boid_obstacles(op, normals, 0.06, 0.13, bpos, bvel, brute=True)
    assert np.array_equal(a, b) and (a != bvel).any()


def test_obstacle_sphere_pushes_boids_outwards():
    # a boid near a spherical obstacle is pushed along the outward normal: the radial component of its velocity grows,
    # more for the one inside the protection range of the surface cells
    from paper_2311_15088_b200 import workloads as W
    c, r = np.array([0.5, 0.5, 0.5]), 0.2
    op, normals = W.sphere_obstacle((0, 0, 0), (1, 1, 1), 0.04, c, r, w_obs=0.1, heavy=2.0)
    dirs = np.array([[1, 0, 0], [0, -1, 0], [0.6, 0.0, 0.8]], np.float64)
    bpos = np.zeros((6, 4), np.float32)
    bpos[:3, :3] = c + dirs * (r + 0.01)   # hugging the surface
    bpos[3:, :3] = c + dirs * (r + 0.09)   # further out, still in visual range
    bvel = np.zeros((6, 4), np.float32)
    out = R.boid_obstacles(op, normals, 0.05, 0.12, bpos, bvel)
    radial = np.einsum("ij,ij->i", out[:, :3].astype(np.float64), np.vstack([dirs, dirs]))
    assert (radial > 0).all() and (radial[:3] > radial[3:]).all()
    far = np.zeros((1, 4), np.float32)
    far[0, :3] = c + [0.45, 0, 0]
    assert np.array_equal(R.boid_obstacles(op, normals, 0.05, 0.12, far, np.zeros((1, 4), np.float32)), np.zeros((1, 4), np.float32))
