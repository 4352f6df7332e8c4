"""sph_build_grid_static -- the entry point that allocates nothing (include/sphboid.h) -- against the existing path
(sph_build_grid on a context) and the oracle: integers, so bit-exact.  Two calls in a row share the static scratch; the
second is smaller and on another grid, so it runs over the first one's leftovers.  Collected last on purpose."""
import numpy as np
import pytest
import torch

from oracle import refbind as R
from paper_2311_15088_b200 import binding as B
from paper_2311_15088_b200 import workloads as W
from tests.gpuutil import Sim, dev, host_u32, u32

pytestmark = pytest.mark.gpu


def _existing(sp, pos_np):
    with Sim(dict(sph=sp, n=pos_np.shape[0])) as sim:
        cell, perm, start = sim.build_grid(dev(pos_np), dev(np.zeros_like(pos_np)))
        return sim.C, cell, perm, start


def _static(sp, pos_t, cell_t, perm_t, start_t):
    B.sph_build_grid_static(sp["box_min"], sp["box_max"], sp["h"], pos_t, cell_t, perm_t, start_t)
    torch.cuda.synchronize()


def _cases():
    base = W.config(1)["sph"]
    # the maximum size on 27 x 20 x 12 = 6480 cells (points outside the box included), then 5000 points on 16^3 cells
    sp1 = dict(base, h=0.0371, box_max=(1.0, 0.73, 0.41))
    pos1 = W.random_cloud(B.SPH_STATIC_MAX_POINTS, (-0.05, -0.05, -0.05), (1.05, 0.78, 0.46), seed=11)
    sp2 = dict(base)
    pos2 = W.random_cloud(5000, (0.0, 0.0, 0.0), (1.0, 1.0, 0.3), seed=12)
    return [(sp1, pos1), (sp2, pos2)]


def test_static_grid_build_matches_the_context_path_on_two_calls_in_a_row():
    cases = _cases()
    want = [_existing(sp, pos) for sp, pos in cases]
    # outputs and inputs first, then the two calls back to back
    bufs = []
    for (sp, pos), (C, _, _, _) in zip(cases, want):
        n = pos.shape[0]
        bufs.append((dev(pos), u32(n), u32(n), u32(C + 1)))
    for (sp, _), (pos_t, cell_t, perm_t, start_t) in zip(cases, bufs):
        B.sph_build_grid_static(sp["box_min"], sp["box_max"], sp["h"], pos_t, cell_t, perm_t, start_t)
    torch.cuda.synchronize()
    for (sp, pos), (C, cell, perm, start), (_, cell_t, perm_t, start_t) in zip(cases, want, bufs):
        assert np.array_equal(host_u32(cell_t), cell)
        assert np.array_equal(host_u32(start_t), start)
        assert np.array_equal(host_u32(perm_t), perm)
        rc, rp, rs = R.build_grid(sp, pos)
        assert C == len(rs) - 1
        assert np.array_equal(host_u32(cell_t), rc) and np.array_equal(host_u32(start_t), rs)
        assert np.array_equal(host_u32(perm_t), rp)
    # the same two calls again, in the other order, give the same results (the scratch carries nothing over)
    for k in (1, 0):
        sp, _ = cases[k]
        pos_t, cell_t, perm_t, start_t = bufs[k]
        cell_t.fill_(-1), perm_t.fill_(-1), start_t.fill_(-1)
        _static(sp, pos_t, cell_t, perm_t, start_t)
        assert np.array_equal(host_u32(cell_t), want[k][1])
        assert np.array_equal(host_u32(perm_t), want[k][2])
        assert np.array_equal(host_u32(start_t), want[k][3])


def test_static_grid_build_takes_no_device_memory_after_its_first_call():
    sp, pos = _cases()[1]
    C = 16 ** 3
    pos_t, cell_t, perm_t, start_t = dev(pos), u32(pos.shape[0]), u32(pos.shape[0]), u32(C + 1)
    _static(sp, pos_t, cell_t, perm_t, start_t)  # the first launch may load the kernel's module
    same = False
    for attempt in range(3):  # the figure is device-wide: another process may move it once, not three times in a row
        free0, _ = torch.cuda.mem_get_info()
        for _ in range(3):
            _static(sp, pos_t, cell_t, perm_t, start_t)
        free1, _ = torch.cuda.mem_get_info()
        same = same or free1 == free0
    assert same


def test_static_grid_build_rejects_sizes_beyond_its_maximum_and_bad_arguments():
    sp = W.config(1)["sph"]
    n = B.SPH_STATIC_MAX_POINTS + 1
    pos_t = dev(W.random_cloud(n, (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), seed=13))
    cell_t, perm_t = u32(n), u32(n)
    start_t = u32(16 ** 3 + 1)
    start_t.fill_(7)
    with pytest.raises(B.SphError) as e:
        B.sph_build_grid_static(sp["box_min"], sp["box_max"], sp["h"], pos_t, cell_t, perm_t, start_t)
    assert e.value.code == B.SPH_E_CAPACITY and "SPH_STATIC_MAX_POINTS" in str(e.value)
    with pytest.raises(B.SphError) as e:  # 32^3 cells
        B.sph_build_grid_static(sp["box_min"], sp["box_max"], 0.5 * sp["h"], pos_t[:100], cell_t, perm_t, u32(32 ** 3 + 1))
    assert e.value.code == B.SPH_E_CAPACITY and "SPH_STATIC_MAX_CELLS" in str(e.value)
    with pytest.raises(B.SphError) as e:  # cell_start too short
        B.sph_build_grid_static(sp["box_min"], sp["box_max"], sp["h"], pos_t[:100], cell_t, perm_t, u32(16 ** 3))
    assert e.value.code == B.SPH_E_INVALID
    torch.cuda.synchronize()
    assert bool((start_t == 7).all())  # nothing was launched
    # an empty input is fine: every start is 0
    B.sph_build_grid_static(sp["box_min"], sp["box_max"], sp["h"], None, None, None, start_t)
    torch.cuda.synchronize()
    assert bool((start_t == 0).all())
