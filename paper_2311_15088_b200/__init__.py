"""paper_2311_15088_b200 -- the per-frame particle pipeline of arXiv 2311.15088 (uniform-grid neighbour search,
SPH, boids, voxel SDF, marching cubes) as hand-written CUDA for sm_100a behind a C ABI (include/sphboid.h).

`binding` is the thin ctypes layer (same names as the header); `workloads` builds the seeded synthetic configs;
`build` compiles libsphboid.so in-tree.  There is no CPU fallback.
"""
__all__ = ["binding", "workloads", "build"]
