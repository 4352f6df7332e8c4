"""Parity of S1-S5 (cell hash, histogram, scan, counting sort, reorder) against the oracle: bit-exact."""
import numpy as np
import pytest
import torch

from oracle import refbind as R
from paper_2311_15088_b200 import binding as B
from paper_2311_15088_b200 import workloads as W
from tests.gpuutil import Sim, dev, host_u32

pytestmark = pytest.mark.gpu


def _check(sp, pos_np):
    cfg = dict(sph=sp, n=pos_np.shape[0])
    with Sim(cfg) as sim:
        cell, perm, start = sim.build_grid(dev(pos_np), dev(np.zeros_like(pos_np)))
        rc, rp, rs = R.build_grid(sp, pos_np)
        assert sim.C == len(rs) - 1
        assert np.array_equal(cell, rc)
        assert np.array_equal(start, rs)
        assert np.array_equal(perm, rp)


@pytest.mark.parametrize("idx,scale", [(1, None), (2, None), (3, 2), (4, 4), (5, 4)])
def test_grid_matches_oracle_on_configs(idx, scale):
    cfg = W.config(idx, scale=scale)
    _check(cfg["sph"], cfg["pos"])


@pytest.mark.parametrize("n", [1, 2, 255, 256, 257, 2047, 2048, 2049, 10000])
def test_grid_ragged_sizes_and_odd_cell_size(n):
    sp = dict(W.config(1)["sph"], h=0.0371, box_max=(1.0, 0.73, 0.41))  # C = 27*20*12 = 6480, not a tile multiple
    _check(sp, W.random_cloud(n, (-0.05, -0.05, -0.05), (1.05, 0.78, 0.46), seed=n))


def test_grid_degenerate_all_in_one_cell_and_tiny_grid():
    sp = dict(W.config(1)["sph"], h=0.5)  # 2x2x2 cells
    pos = W.random_cloud(3000, (0.1, 0.1, 0.1), (0.4, 0.4, 0.4), seed=1)  # everything in cell 0
    _check(sp, pos)
    sp = dict(W.config(1)["sph"], h=2.0)  # a single cell
    _check(sp, W.random_cloud(500, (0, 0, 0), (1, 1, 1), seed=2))


def test_grid_empty_input_and_scan_sizes():
    # n = 0: every start is 0; also grids whose C+1 straddles scan-tile boundaries (tile = 2048 cells)
    for h in (1.0 / 16, 1.0 / 12.7, 1.0 / 45):
        sp = dict(W.config(1)["sph"], h=h)
        cfg = dict(sph=sp, n=0)
        with Sim(cfg) as sim:
            start = torch.full((sim.C + 1,), -1, dtype=torch.int32, device="cuda")
            B.sph_build_grid(sim.ctx, None, None, cell_start=start)
            torch.cuda.synchronize()
            assert int(start.abs().sum()) == 0


def test_grid_rebuild_is_repeatable():
    # the histogram is cleared inside the scan and the scan state is epoch-tagged: many builds on one context
    cfg = W.config(2)
    with Sim(cfg) as sim:
        pos = dev(cfg["pos"])
        first = sim.build_grid(pos)
        for _ in range(5):
            again = sim.build_grid(pos)
            assert all(np.array_equal(a, b) for a, b in zip(first, again))


# ---- neighbour counts: sorted grid vs the paper's unsorted fixed-capacity hash grid (N4 baseline) ----------
@pytest.mark.parametrize("idx,scale", [(1, None), (2, None), (4, 4), (5, 4)])
def test_neighbor_counts_sorted_and_hashgrid_match_oracle(idx, scale):
    import torch
    from oracle import refbind as R
    from paper_2311_15088_b200 import binding as B
    cfg = W.config(idx, scale=scale)
    _, ref_cnt = R.density(cfg["sph"], cfg["pos"])
    with Sim(cfg) as sim:
        pos = dev(cfg["pos"])
        cnt = torch.zeros(cfg["n"], dtype=torch.int32, device="cuda")
        B.sph_neighbor_count(sim.ctx, pos, cnt)
        assert np.array_equal(host_u32(cnt), ref_cnt)
        cnt.zero_()
        dropped = B.sph_hashgrid_neighbor_count(sim.ctx, pos, 64, cnt)
        assert dropped == 0 and np.array_equal(host_u32(cnt), ref_cnt)
        # a capacity below the fullest cell: particles are dropped, reported, and the counts can only shrink
        cnt2 = torch.zeros_like(cnt)
        dropped = B.sph_hashgrid_neighbor_count(sim.ctx, pos, 4, cnt2)
        assert dropped > 0 and bool((cnt2 <= cnt).all()) and bool((cnt2 < cnt).any())


def test_invalidate_grid_after_rewriting_positions_in_place():
    """sph_step reuses a grid by pointer identity (include/sphboid.h): a caller that rewrites pos in place after
    sph_build_grid must call sph_invalidate_grid, after which the step sorts the new positions; mc_* then refuses the
    stale grid."""
    import torch
    from oracle import refbind as R
    from paper_2311_15088_b200 import binding as B
    from tests.gpuutil import vec_err
    cfg = W.config(1)
    other = W.uniform_box(cfg["n"], (0.1,) * 3, (0.6,) * 3, 3, 77)
    ref = R.step(cfg["sph"], other, cfg["vel"])
    with Sim(cfg, G=16) as sim:
        pos, vel = dev(cfg["pos"]), dev(cfg["vel"])
        B.sph_build_grid(sim.ctx, pos, vel)
        pos.copy_(dev(other))            # same pointer, new contents
        B.sph_invalidate_grid(sim.ctx)
        mp = dict(origin=(0.0, 0.0, 0.0), spacing=1.0 / 15, n_point_per_axis=16, radius=cfg["sph"]["h"],
                  particle_radius=0.5 * cfg["sph"]["h"], iso=0.0)
        with pytest.raises(B.SphError) as e:
            B.mc_voxel_sdf(sim.ctx, mp, torch.zeros(16 ** 3, device="cuda"))
        assert e.value.code == B.SPH_E_STALE_GRID
        out = sim.step(pos, vel)
    assert np.array_equal(out["ncount"], ref["ncount"])
    bad, worst = vec_err(out["pos"][:, :3], ref["pos"][:, :3])
    assert bad == 0, (bad, worst)


@pytest.mark.parametrize("n,h", [(16384, 1.0 / 20), (16385, 1.0 / 20), (16384, 1.0 / 20.2), (5000, 1.0 / 20.16), (5000, 1.0 / 21)])
def test_grid_small_and_large_paths_agree_at_their_boundary(n, h):
    """k_grid_small takes grids of <= 8192 cells and <= 16384 points, the four-kernel path everything else: both sides of
    either limit (20^3 = 8000 cells, 21^3 = 9261; 16384 / 16385 points), dense cells (a cloud in one corner: ~100 points
    per cell, the long-run ranking of k_reorder on the large path), against the oracle; and the two paths alternate on one
    context without disturbing each other (the large path's histogram must still be clear)."""
    sp = dict(W.config(1)["sph"], h=h)
    pos = W.random_cloud(n, (0.0, 0.0, 0.0), (0.3, 0.3, 0.25), seed=n)
    _check(sp, pos)
    with Sim(dict(sph=sp, n=n)) as sim:
        rc, rp, rs = R.build_grid(sp, pos)
        few = pos[:1000].copy()
        fc, fp, fs = R.build_grid(sp, few)
        for p_np, want in ((pos, (rc, rp, rs)), (few, (fc, fp, fs)), (pos, (rc, rp, rs))):
            cell, perm, start = sim.build_grid(dev(p_np), dev(np.zeros_like(p_np)))
            assert np.array_equal(cell, want[0]) and np.array_equal(perm, want[1]) and np.array_equal(start, want[2])
