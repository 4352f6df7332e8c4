"""Pins for the oracle's SPH density / force / integration (S6, S8, S10).  CPU only."""
import math

import numpy as np
import pytest

from oracle import refbind as R
from paper_2311_15088_b200 import workloads as W

A = 2.0 ** -5


def _sp(**kw):
    sp = dict(box_min=(0.0, 0.0, 0.0), box_max=(1.0, 1.0, 1.0), h=2 * A, rest_density=1000.0, mass=1000.0 * A ** 3,
              stiffness=3.0, viscosity=0.1, gravity=(0.0, -9.81, 0.0), dt=1e-3, wall_damping=0.5)
    sp.update(kw)
    return sp


def test_w_poly6_integrates_to_one():
    # int W dV = 1.  Composite Simpson on 4 pi r^2 W(r,h) over [0,h].
    for h in (0.0625, 0.3, 1.7):
        n = 2000
        r = np.linspace(0.0, h, n + 1)
        f = np.array([4.0 * math.pi * x * x * R.w_poly6(x, h) for x in r])
        integral = (h / n) / 3.0 * (f[0] + f[-1] + 4.0 * f[1:-1:2].sum() + 2.0 * f[2:-1:2].sum())
        assert abs(integral - 1.0) < 1e-9
        assert R.w_poly6(1.0001 * h, h) == 0.0


def _lattice_sum(ratio):
    """sum over integer offsets n with |n|*ratio < 2 of (4 - ratio^2 |n|^2)^3, in units of a^6 (h = 2a)."""
    s, cnt = 0.0, 0
    rng = range(-4, 5)
    for i in rng:
        for j in rng:
            for k in rng:
                r2 = ratio * ratio * (i * i + j * j + k * k)
                if r2 < 4.0:
                    s += (4.0 - r2) ** 3
                    cnt += 1
    return s, cnt


@pytest.mark.parametrize("ratio,count,rho_over_rho0", [(1.0, 27, 1.0097752), (0.8, 81, 1.944202)])
def test_lattice_interior_density_closed_form(ratio, count, rho_over_rho0):
    # SURVEY 8(c) pin: h = 2a, m = rho0 a^3: rho/rho0 = 315/(64 pi 512) * sum (4 - n^2)^3; = 315*330/(64 pi 512) at rest
    s, cnt = _lattice_sum(ratio)
    assert cnt == count
    closed = 315.0 * s / (64.0 * math.pi * 512.0)
    assert abs(closed - rho_over_rho0) < 2e-6
    if ratio == 1.0:
        assert s == 330.0
    pos = W.lattice(12, 12, 12, A * ratio, 0.0, 0)
    rho, cnt_o = R.density(_sp(), pos)
    centre = 5 + 12 * (5 + 12 * 5)
    assert cnt_o[centre] == count  # the six at r = h fail the strict < (D:A-PRED)
    assert abs(rho[centre] / 1000.0 - closed) < 2e-6 * closed
    # self term alone: 0.195835 rho0
    lone, c1 = R.density(_sp(), np.array([[0.5, 0.5, 0.5, 0]], np.float32))
    assert c1[0] == 1 and abs(lone[0] / 1000.0 - 0.195835) < 1e-6


def test_jittered_config1_interior_count():
    cfg = W.config(1)
    _, cnt = R.density(cfg["sph"], cfg["pos"])
    ijk = np.indices((16, 16, 16)).reshape(3, -1)  # k,j,i order irrelevant for an interior mask
    interior = np.all((ijk >= 2) & (ijk <= 13), axis=0)
    mean = cnt.reshape(16, 16, 16).transpose(0, 1, 2).reshape(-1)[interior].mean()
    assert 29.0 < mean < 31.0  # approx 29.9


def _pair_by_hand(m, R_, k, rho0, mu, pa, va, ra, pb, vb, rb):
    """Eq. 36 + Eq. 41 with the sign of Listing 3, float64, summand for j=b."""
    d = np.asarray(pa, np.float64) - np.asarray(pb, np.float64)
    dv = np.asarray(va, np.float64) - np.asarray(vb, np.float64)
    r = np.linalg.norm(d)
    q = r / R_
    press = 15.0 * k / (math.pi * R_ ** 4) * m * (ra + rb - 2 * rho0) / rb * (1 - q) ** 2 / q * d
    visc = -40.0 * mu / (math.pi * R_ ** 4) * m * dv / rb * (1 - q)
    return press + visc


def test_pair_term_hand_case_and_antisymmetry():
    m, h, k, rho0, mu = 0.03, 0.0625, 3.0, 1000.0, 0.1
    pa, pb = np.array([0.5, 0.5, 0.5], np.float32), np.array([0.52, 0.49, 0.515], np.float32)
    va, vb = np.array([0.1, -0.2, 0.3], np.float32), np.array([-0.3, 0.1, 0.05], np.float32)
    ra, rb = 1013.0, 998.5
    got = R.pair_term(m, h, k, rho0, mu, pa, va, ra, pb, vb, rb)
    want = _pair_by_hand(m, h, k, rho0, mu, pa, va, ra, pb, vb, rb)
    assert np.allclose(got, want, rtol=2e-6, atol=0)
    # Newton's third law under D:A-RHO: pair(a,b)/rho_a = -pair(b,a)/rho_b
    back = R.pair_term(m, h, k, rho0, mu, pb, vb, rb, pa, va, ra)
    assert np.allclose(got / ra, -back / rb, rtol=1e-5, atol=0)
    # early-outs: coincident and out-of-range pairs give zero
    assert not R.pair_term(m, h, k, rho0, mu, pa, va, ra, pa, vb, rb).any()
    far = pa + np.array([h * 1.001, 0, 0], np.float32)
    assert not R.pair_term(m, h, k, rho0, mu, pa, va, ra, far, vb, rb).any()


def test_two_particle_step_by_hand():
    sp = _sp(gravity=(0.0, 0.0, 0.0))
    h, m = sp["h"], sp["mass"]
    pos = np.array([[0.5, 0.5, 0.5, 0], [0.5 + 0.6 * h, 0.5, 0.5, 0]], np.float32)
    vel = np.array([[0.2, 0.0, 0.0, 0], [-0.1, 0.05, 0.0, 0]], np.float32)
    out = R.step(sp, pos, vel)
    r = float(pos[1, 0]) - float(pos[0, 0])
    rho = m * (R.w_poly6(0.0, h) + R.w_poly6(r, h))  # both particles see self + the other
    assert np.allclose(out["density"], rho, rtol=1e-6)
    assert list(out["ncount"]) == [2, 2]
    f0 = _pair_by_hand(m, h, 3.0, 1000.0, 0.1, pos[0, :3], vel[0, :3], rho, pos[1, :3], vel[1, :3], rho)
    assert np.allclose(out["accel"][0, :3], f0 / rho, rtol=1e-5, atol=1e-9)
    assert np.allclose(out["accel"][1, :3], -f0 / rho, rtol=1e-5, atol=1e-9)
    # Euler-Cromer: v first, then x with the NEW v (D:A-INTEG)
    v_new = vel[0, :3] + 1e-3 * out["accel"][0, :3]
    assert np.allclose(out["vel"][0, :3], v_new, rtol=1e-6, atol=1e-9)
    assert np.allclose(out["pos"][0, :3], pos[0, :3] + 1e-3 * v_new, rtol=1e-7)


def test_net_momentum_near_zero_and_reading_discriminates():
    cfg = W.config(1)
    vel = W.uniform_box(cfg["n"], (-0.5,) * 3, (0.5,) * 3, 1, 30)
    out = R.step(cfg["sph"], cfg["pos"], vel)
    g = np.array(cfg["sph"]["gravity"], np.float64)
    f = out["accel"][:, :3].astype(np.float64) - g
    ratio = np.linalg.norm(f.sum(0)) / np.linalg.norm(f, axis=1).sum()
    assert ratio < 1e-5  # symmetric pairwise force => near-zero net momentum (north_star pin)
    # the literal no-/rho_i variant (a_i = f_i + g) is NOT momentum conserving: this pin tells the two readings apart
    lit = f * out["density"][:, None].astype(np.float64)
    assert np.linalg.norm(lit.sum(0)) / np.linalg.norm(lit, axis=1).sum() > 1e-4


def test_lattice_interior_force_vanishes():
    pos = W.lattice(12, 12, 12, A, 0.0, 0)
    out = R.step(_sp(gravity=(0.0, 0.0, 0.0)), pos, np.zeros_like(pos))
    a = out["accel"].reshape(12, 12, 12, 4)[4:8, 4:8, 4:8, :3]
    assert np.abs(a).max() < 1e-4 * out["amag"].max()  # symmetric neighbourhood: pressure terms cancel


def test_viscosity_only_dissipates():
    cfg = W.config(1)
    sp = dict(cfg["sph"], stiffness=0.0, gravity=(0.0, 0.0, 0.0))
    vel = W.uniform_box(cfg["n"], (-0.2,) * 3, (0.2,) * 3, 2, 30)
    pos = cfg["pos"]
    ke = [(vel[:, :3].astype(np.float64) ** 2).sum()]
    for _ in range(3):
        out = R.step(sp, pos, vel)
        pos, vel = out["pos"], out["vel"]
        ke.append((vel[:, :3].astype(np.float64) ** 2).sum())
    assert all(b < a for a, b in zip(ke, ke[1:]))  # -40 mu v_ij is dissipative (D:A-VISC-SIGN)


def test_free_fall_and_wall():
    sp = _sp()
    pos = np.array([[0.5, 0.9, 0.5, 0]], np.float32)
    vel = np.zeros_like(pos)
    n = 50
    for _ in range(n):
        out = R.step(sp, pos, vel)
        pos, vel = out["pos"], out["vel"]
    g, dt = -9.81, 1e-3
    assert abs(vel[0, 1] - g * n * dt) < 1e-5
    assert abs(pos[0, 1] - (0.9 + g * dt * dt * n * (n + 1) / 2.0)) < 1e-5  # symplectic Euler closed form
    assert vel[0, 0] == 0 and vel[0, 2] == 0
    # wall: a particle heading out is clamped and that axis' velocity reversed and halved (D:A-WALL)
    pos = np.array([[0.9995, 0.5, 0.0002, 0]], np.float32)
    vel = np.array([[1.0, 0.0, -0.5, 0]], np.float32)
    out = R.step(_sp(gravity=(0.0, 0.0, 0.0)), pos, vel)
    assert out["pos"][0, 0] == np.float32(1.0) and out["vel"][0, 0] == np.float32(-0.5)
    assert out["pos"][0, 2] == np.float32(0.0) and out["vel"][0, 2] == np.float32(0.25)
    assert out["vel"][0, 1] == 0.0


def test_particles_stay_in_box_multi_step():
    cfg = W.config(1)
    pos, vel = cfg["pos"], cfg["vel"]
    for _ in range(10):
        out = R.step(cfg["sph"], pos, vel)
        pos, vel = out["pos"], out["vel"]
        assert pos[:, :3].min() >= 0.0 and pos[:, :3].max() <= 1.0
        assert np.isfinite(pos).all() and np.isfinite(vel).all()


def test_step_grid_equals_brute_force():
    cfg = W.config(1, scale=2)
    vel = W.uniform_box(cfg["n"], (-0.3,) * 3, (0.3,) * 3, 4, 30)
    a = R.step(cfg["sph"], cfg["pos"], vel, cfg["bpos"], cfg["bvel"], cfg["boid"], brute=False)
    b = R.step(cfg["sph"], cfg["pos"], vel, cfg["bpos"], cfg["bvel"], cfg["boid"], brute=True)
    for k in ("ncount", "touched", "density", "pos", "vel", "accel"):
        assert np.array_equal(a[k], b[k]), k
