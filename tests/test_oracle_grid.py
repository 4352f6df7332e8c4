"""Pins for the oracle's grid / counting sort / neighbour sets (S1-S6 counts).  CPU only."""
import numpy as np
import pytest

from oracle import refbind as R
from paper_2311_15088_b200 import workloads as W


def _sp(h, box_max=(1.0, 1.0, 1.0)):
    return dict(box_min=(0.0, 0.0, 0.0), box_max=box_max, h=h, rest_density=1000.0, mass=0.03, stiffness=3.0,
                viscosity=0.1, gravity=(0.0, -9.81, 0.0), dt=1e-3, wall_damping=0.5)


@pytest.mark.parametrize("h,box", [(0.0625, (1.0, 1.0, 1.0)), (0.11, (1.0, 0.7, 0.45)), (0.3, (1.0, 1.0, 0.2))])
def test_grid_invariants(h, box):
    sp = _sp(h, box)
    pos = W.random_cloud(2048, (0, 0, 0), box, seed=3)
    dims, C = R.grid_dims(sp)
    # D:A-DIMS: ceil of extent / h, host double
    assert dims == tuple(max(1, int(np.ceil(np.float64(np.float32(b)) / np.float64(np.float32(h))))) for b in box)
    cell, perm, start = R.build_grid(sp, pos)
    # cell index recomputed independently in numpy float32 (Eq. 47, P:395 hash)
    hf = np.float32(h)
    c = np.floor((pos[:, :3] - np.float32(0.0)) / hf).astype(np.int64)
    c = np.clip(c, 0, np.array(dims) - 1)
    key = c[:, 0] + dims[0] * (c[:, 1] + dims[1] * c[:, 2])
    assert np.array_equal(key, cell)
    # exclusive starts: monotone, start[0] = 0, start[C] = N, differences = histogram
    assert start[0] == 0 and start[-1] == len(pos)
    assert np.array_equal(np.diff(start.astype(np.int64)), np.bincount(key, minlength=C))
    # perm is a permutation, runs hold their own cell, ascending id inside a cell (stable sort, D:A-SORT)
    assert np.array_equal(np.sort(perm), np.arange(len(pos)))
    assert np.array_equal(perm, np.argsort(key, kind="stable"))


def test_clamped_cells_out_of_box():
    sp = _sp(0.25)
    pos = np.array([[-0.3, 0.5, 0.5, 0], [1.0, 1.0, 1.0, 0], [1.7, -2.0, 0.1, 0]], np.float32)
    cell, _, _ = R.build_grid(sp, pos)
    assert list(cell) == [0 + 4 * (2 + 4 * 2), 3 + 4 * (3 + 4 * 3), 3 + 4 * (0 + 4 * 0)]  # D:A-CLAMPCELL


@pytest.mark.parametrize("h", [0.0625, 0.11, 0.2])
def test_neighbour_counts_vs_brute_force(h):
    sp = _sp(h)
    pos = W.random_cloud(1500, (0, 0, 0), (0.6, 0.5, 0.4), seed=5)
    rho_g, cnt_g = R.density(sp, pos, brute=False)
    rho_b, cnt_b = R.density(sp, pos, brute=True)
    assert np.array_equal(cnt_g, cnt_b)
    assert np.array_equal(rho_g, rho_b)  # binary64 sums of identical binary32 terms round identically
    # independent numpy count with the D:A-FP r^2 (fma emulated exactly in float64: products of floats are exact)
    p = pos[:, :3].astype(np.float32)
    d = (p[:, None, :] - p[None, :, :]).astype(np.float32).astype(np.float64)
    t = np.float32(d[..., 0] * d[..., 0]).astype(np.float64)            # dx*dx rounded
    t = (d[..., 1] * d[..., 1] + t).astype(np.float32).astype(np.float64)  # fma: exact product + add, one rounding
    r2 = (d[..., 2] * d[..., 2] + t).astype(np.float32)
    h2 = np.float32(h) * np.float32(h)
    assert np.array_equal((r2 < h2).sum(1), cnt_b)
    assert cnt_b.min() >= 1  # self counts (D:A-SELF)


def test_neighbours_across_clamped_cells():
    # particles outside the box are binned into clamped border cells and must still be found (exactness of the 27-cell walk)
    sp = _sp(0.1)
    pos = W.random_cloud(600, (-0.15, -0.15, 0.8), (0.25, 0.25, 1.2), seed=9)
    _, cnt_g = R.density(sp, pos, brute=False)
    _, cnt_b = R.density(sp, pos, brute=True)
    assert np.array_equal(cnt_g, cnt_b)
