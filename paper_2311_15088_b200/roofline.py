"""Algorithmic bytes per kernel launch -- bookkeeping for bench.py.

"Algorithmic" = the compulsory traffic of the method with SoA float4 state, every array touched once per
pass: what a perfect implementation would have to move through HBM.  Bytes the implementation moves on top
(scratch such as the arrival ranks, re-reads served by L2) are NOT counted, so achieved GB/s = these bytes /
measured time is a lower bound on nothing and an upper bound on nothing: it is the roofline coordinate.

N particles, C particle-grid cells, B boids, Cb boid-grid cells, G^3 voxel corners, T triangles.
"""


def kernel_bytes(n, c, nb, cb, g, t):
    v = g ** 3
    return {
        # S1-S2: read pos 16, write key 4
        "k_hash_count": 20 * n,
        # S3: read count 4, write start 4 per cell
        "k_scan_cells": 8 * c,
        # S4: read key 4, pos 16, vel 16; write posS 16, velS 16, perm 4
        "k_scatter": 0,        # implementation split of S4: its bytes are counted on k_reorder
        "k_reorder": 72 * n,
        "k_grid_small": 92 * n + 8 * c,                 # S1-S5 in one block (small grids): the four kernels' bytes
        "k_grid_small[boid grid]": 92 * nb + 8 * cb,
        "k_hash_count[boid grid]": 20 * nb,
        "k_scan_cells[boid grid]": 8 * cb,
        "k_scatter[boid grid]": 0,
        "k_reorder[boid grid]": 72 * nb,
        # S6: read posS 16 + cell table 8 per cell, write rho 4
        "k_density": 20 * n + 8 * c,
        # S7: read bpos 16, write rho_b 4 (the fluid it gathers is already counted)
        "k_boid_density": 20 * nb,
        # S8-S10: read posS 16, velS 16, rho 4, perm 4; write pos' 16, vel' 16
        "k_force_list": 72 * n,     # the stored-neighbour-list variant of the same rows
        "k_density_brick": 20 * n + 8 * c,   # S6 with a brick of cells staged per block (sph_brick.cu)
        "k_force_masks": 72 * n,
        # S11-S13: read bpos, bvel 32, rho_b 4, perm 4; write 32
        "k_boid_step": 72 * nb,
        # S14: write phi 4 per corner; read posS 16 per particle and the cell table 8 per cell
        "k_voxel_sdf": 4 * v + 16 * n + 8 * c,
        "k_voxel_sdf_tiles": 4 * v + 16 * n + 8 * c,    # the 2x2x2-corners-per-lane tile variant of the same row
        # S15-S17: read phi 4 per corner, write 36 per triangle
        "k_mc_signs": 4 * v,                            # S15 first half: read phi once -> 1 bit per corner
        "k_mc_count": v // 8,                           # S15 second half - S16 on the bit field (1 bit per corner)
        "k_mc_emit": 36 * t,                            # S17: 36 B per triangle (+ the few phi values it interpolates)
        # N3 (indexed mesh): bit field once more, 24 B per vertex (position + normal), 12 B per triangle
        "k_mc_edge_scan": v // 8 + v // 8,
        "k_mc_vertices": 0,
        "k_mc_emit_indices": 12 * t,
        "k_zero_u32": 4,
    }


SIM_KERNELS = ("k_hash_count", "k_scan_cells", "k_scatter", "k_reorder", "k_hash_count[boid grid]",
               "k_scan_cells[boid grid]", "k_scatter[boid grid]", "k_reorder[boid grid]", "k_density",
               "k_boid_density", "k_force_list", "k_boid_step")
# The surface pass in SURVEY.md 8(d)'s accounting: phi written once and read once (4 + 4 B per corner), particles and
# cell table read once, 36 B per triangle.  The fused path reads the sign bits instead of phi (k_mc_signs does not run),
# but the pass figure keeps the survey's 8 B per corner so that it stays comparable.
MC_KERNELS = ("k_voxel_sdf", "k_mc_signs", "k_mc_emit")


def summarise(profile, n, c, nb, cb, g, t, peak_gbs):
    """profile: {kernel: (launches, total_ms)}.  Returns (per-kernel rows, dominant kernel name).

    Row: dict(kernel, launches, avg_us, share, bytes, gbs, frac).  share = fraction of the summed kernel time.
    """
    kb = kernel_bytes(n, c, nb, cb, g, t)
    total = sum(ms for _, ms in profile.values()) or 1.0
    rows = []
    for name, (cnt, ms) in profile.items():
        avg_ms = ms / max(cnt, 1)
        b = kb.get(name, 0)
        gbs = b / (avg_ms * 1e-3) / 1e9 if avg_ms > 0 else 0.0
        rows.append(dict(kernel=name, launches=cnt, avg_us=avg_ms * 1e3, share=ms / total, bytes=b, gbs=gbs,
                         frac=gbs / peak_gbs))
    rows.sort(key=lambda r: -r["share"])
    return rows, (rows[0]["kernel"] if rows else None)


def pass_bytes(names, n, c, nb, cb, g, t):
    kb = kernel_bytes(n, c, nb, cb, g, t)
    return sum(kb[k] for k in names)


# ---- arithmetic roofline of the three pair kernels -------------------------------------------
# The hot kernels are bound by binary32 arithmetic, not by HBM, so bench.py also places the dominant kernel on the
# ALU roofline: algorithmic flops = (true pairs) x (flops of one pair as the paper's listing evaluates it), peak =
# 148 SMs x 128 lanes x 2 flop x SM clock (FMA counted as two).  Only true pairs count: candidates that fail the
# distance test, list building and filters are overhead of the implementation.
ALU_PEAK_TFLOPS_AT_MHZ = lambda mhz: 148 * 128 * 2 * mhz * 1e6 / 1e12

FLOP_PER_PAIR = {
    # Listing 9: d = x_j - x (3), r^2 (5), 1 - r^2/R^2 (2), k = u^3 (2), S0 += k (1), S1 += k d (6)
    "sdf": 19,
    # Eq. 27: d (3), r^2 (5), h^2 - r^2 (1), cube and accumulate (3)
    "density": 12,
    # Listing 3: d, dv (6), r^2 (5), sqrt + q, q2 (4), q2/q (1), pressure factor (4), coefficient (3),
    # three components of (pterm d - 40 mu dv) scaled and accumulated (12)
    "force": 35,
}
KERNEL_KIND = {"k_density_brick": "density", "k_force_masks": "force",
               "k_voxel_sdf_tiles": "sdf", "k_voxel_sdf": "sdf",
               "k_density": "density", "k_force_list": "force"}


def sdf_pairs(n, radius, spacing):
    """(corner, particle) pairs with r < R: every particle reaches the corners of a ball of radius R of the voxel
    lattice, 4/3 pi (R / spacing)^3 of them, when the voxel grid covers the fluid (it does in all five configs)."""
    import math
    return n * 4.0 / 3.0 * math.pi * (radius / spacing) ** 3


def alu_point(kernel, avg_us, pairs, sm_mhz):
    kind = KERNEL_KIND.get(kernel)
    if kind is None or not pairs or avg_us <= 0:
        return None
    flops = FLOP_PER_PAIR[kind] * pairs
    peak = ALU_PEAK_TFLOPS_AT_MHZ(sm_mhz)
    ach = flops / (avg_us * 1e-6) / 1e12
    return dict(achieved=ach, peak=peak, frac=ach / peak, flop_per_launch=flops, pairs=pairs,
                flop_per_pair=FLOP_PER_PAIR[kind])


def csrc_sha16():
    """Hash of the CUDA sources that hold the frame's kernels (everything under csrc/ except api.cu, which is host-side
    glue, and noalloc.cu, whose one kernel bench.py never launches): stamps profiles/traffic.csv, so that bench.py only
    quotes a DRAM-traffic figure captured on the kernels it is timing."""
    import hashlib
    import os
    d = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc")
    h = hashlib.sha256()
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".h", ".inc")) and name not in ("api.cu", "noalloc.cu"):
            h.update(name.encode())
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def read_traffic(path, kernel):
    """profiles/traffic.csv: first line '# csrc_sha16=<hash> capture=<id>', then kernel,dram_bytes_per_launch,source.
    Returns (bytes or None, capture id, stale?)."""
    import os
    if not os.path.exists(path):
        return None, None, None
    lines = open(path).read().splitlines()
    sha, cap = None, None
    if lines and lines[0].startswith("#"):
        for tok in lines[0][1:].split():
            if tok.startswith("csrc_sha16="):
                sha = tok.split("=", 1)[1]
            if tok.startswith("capture="):
                cap = tok.split("=", 1)[1]
    stale = sha != csrc_sha16()
    val = None
    for row in lines:
        c = row.split(",")
        if len(c) >= 2 and c[0] == kernel:
            try:
                val = float(c[1])
            except ValueError:
                val = None
    return (None if stale else val), cap, stale
