"""CPU-side checks (no GPU): the C-ABI library loads and exports every symbol include/sphboid.h declares, the
binding's struct layouts match the header, the roofline bookkeeping adds up to SURVEY.md 8(d)'s figures, and the
N > 1 plumbing (replicas only) combines per-rank results correctly under gloo with world_size 2."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "sphboid.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return re.findall(r"^\s*(?:const\s+char\s*\*|int|uint32_t|uint64_t|void)\s+(\w+)\s*\(", text, flags=re.M)


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2311_15088_b200 import build as lib_build
    from paper_2311_15088_b200 import binding as B
    lib_build.build()
    names = _declared_functions()
    assert len(names) >= 16 and "sph_create" in names and "mc_extract" in names and "boid_step" in names
    L = B.lib()
    for name in names:
        assert hasattr(L, name), name
    assert sorted(names) == sorted(B.EXPORTS)
    # host-only calls that need no device
    tri, ntri = B.sph_mc_table()
    assert ntri[0] == 0 and ntri[255] == 0 and ntri[8] == 1 and sorted(tri[8][:3]) == [2, 3, 11]
    assert L.sph_kernel_name(0) == b"k_hash_count" and L.sph_kernel_name(1000) is None
    assert L.sph_last_error(None) == b"null context"


def test_library_has_sm100a_code_only():
    from paper_2311_15088_b200 import binding as B
    out = subprocess.run(["cuobjdump", "-lelf", B.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump not available")
    archs = set(re.findall(r"sm_\d+a?", out.stdout))
    assert archs == {"sm_100a"}, archs


def test_struct_sizes_match_header_layout():
    from paper_2311_15088_b200 import binding as B
    # all members are 4-byte scalars: size = 4 * member count, no padding
    assert C.sizeof(B.SphParams) == 4 * (3 + 3 + 1 + 4 + 3 + 2 + 3)
    assert C.sizeof(B.BoidParams) == 4 * (2 + 3 + 3 + 1 + 2 + 3 + 3)
    assert C.sizeof(B.McParams) == 4 * (3 + 1 + 1 + 3)


def test_create_without_device_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2311_15088_b200 import binding as B
    from paper_2311_15088_b200 import workloads as W
    with pytest.raises(B.SphError):
        B.sph_create(W.config(1)["sph"], 16)
    from paper_2311_15088_b200.pipeline import Frame
    with pytest.raises(RuntimeError):
        Frame(W.config(1))


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2311_15088_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "refbind" not in text and "libsphref" not in text and "oracle/" not in text.replace(
                    "oracle/ref_mc.cpp); tests compare", ""), (dirpath, f)


def test_roofline_bytes_match_survey_totals():
    from paper_2311_15088_b200 import roofline as RF
    n, c = 1 << 20, 1 << 18
    kb = RF.kernel_bytes(n, c, 0, 0, 256, 1_500_000)
    sph = sum(kb[k] for k in ("k_hash_count", "k_scan_cells", "k_reorder", "k_density", "k_force_list"))
    assert sph == 184 * n + 16 * c  # 184 B + 16 B C/N per particle-step
    mc = RF.pass_bytes(RF.MC_KERNELS, n, c, 0, 0, 256, 1_500_000)
    assert mc == 8 * 256 ** 3 + 16 * n + 8 * c + 36 * 1_500_000
    rows, dom = RF.summarise({"k_density": (10, 5.0), "k_force_list": (10, 15.0)}, n, c, 0, 0, 256, 0, 6557.4)
    assert dom == "k_force_list" and abs(rows[0]["share"] - 0.75) < 1e-12
    assert abs(rows[0]["gbs"] - 72 * n / 1.5e-3 / 1e9) < 1e-6


def test_workloads_are_reproducible_and_shaped_like_the_configs():
    from paper_2311_15088_b200 import workloads as W
    a, b = W.config(1), W.config(1)
    assert a["n"] == 4096 and a["n_boid"] == 64 and np.array_equal(a["pos"], b["pos"])
    assert not np.array_equal(a["pos"], W.config(1, seed=1)["pos"])
    c4 = W.config(4, scale=8)
    assert c4["sph"]["h"] == 2.0 ** -6 and c4["lattice"] == (16, 16, 8)
    jitter = np.abs(a["pos"][:, 0] - (np.arange(4096) % 16 + 0.5) * 2.0 ** -5).max()
    assert 0.0025 < jitter <= 0.003 + 1e-7  # BASELINE.json config 1: +-0.003


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
from paper_2311_15088_b200 import dist as D
r = D.Ranks(backend="gloo")
r.barrier()
seconds = 1.0 + 0.5 * r.rank          # rank 1 is the slow one
units = 100.0 * (r.rank + 1)
t, u = r.combine(seconds, units)
m = r.reduce_max([float(r.rank), 7.0 - r.rank])
assert (t, u) == (1.5, 300.0), (t, u)
assert m == [1.0, 7.0], m
assert abs(u / t - D.throughput([1.0, 1.5], [100.0, 200.0])) < 1e-12
r.barrier()
r.close()
print("rank", r.rank, "ok")
"""


def test_replicas_combine_under_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    port = 29600 + os.getpid() % 300
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for rank, p in enumerate(procs):
        out, _ = p.communicate(timeout=120)
        assert p.returncode == 0, out
        assert "rank %d ok" % rank in out


def test_bench_reference_arm_runs_on_cpu_small_config():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    import json
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["steps"] == 2
