// grid.cu -- S1-S5: cell hash, histogram, device-wide exclusive scan, counting-sort scatter, reorder.
// P:389-395 (get_cell, hash), P:421-439 + P:467 (Listing 8: set_particle_count, count_sort_particle_index).
#include "kernels.h"

namespace sphb {

namespace {

constexpr int kThreads = 256;
constexpr int kScanItems = 8;                     // cells per thread in the scan
constexpr int kScanTile = kThreads * kScanItems;  // 2048 cells per tile
constexpr int kLongRun = 64;                      // k_reorder: runs longer than this are ranked by the whole warp

// S1 + S2 (P:426-432 set_particle_count): key = hash(get_cell(p)); rank = atomicAdd(count[key], 1).
__global__ void __launch_bounds__(kThreads) k_hash_count(GridDesc g, const float4* __restrict__ pos, uint32_t n,
                                                         uint32_t* __restrict__ key, uint32_t* __restrict__ rank,
                                                         uint32_t* __restrict__ count, uint32_t* __restrict__ box_part,
                                                         uint32_t* __restrict__ aabb) {
  // the bounding box of this build starts empty (the scan kernel, which runs next, folds the partials into it)
  if (blockIdx.x == 0 && threadIdx.x < 6) aabb[threadIdx.x] = threadIdx.x < 3 ? 0xffffffffu : 0u;
  const uint32_t i = blockIdx.x * kThreads + threadIdx.x;
  const bool in = i < n;
  const float4 p = __ldg(pos + (in ? i : n - 1));
  if (in) {
    const int cx = cell_coord(p.x, g.lo[0], g.cell, g.dim[0]);
    const int cy = cell_coord(p.y, g.lo[1], g.cell, g.dim[1]);
    const int cz = cell_coord(p.z, g.lo[2], g.cell, g.dim[2]);
    const uint32_t k = cell_hash(g, cx, cy, cz);
    key[i] = k;
    rank[i] = atomicAdd(count + k, 1u);
  }
  // bounding box of the points (order-preserving uint encoding), used by the surface pass to skip corners that
  // are further than R from every particle: warp min / max, block min / max through shared memory, one partial
  // per block; the scan kernel folds the partials (no same-address atomics from 10^4 blocks)
  __shared__ uint32_t s_box[kThreads / 32][6];
  float lo[3] = {p.x, p.y, p.z}, hi[3] = {p.x, p.y, p.z};
#pragma unroll
  for (int o = 16; o > 0; o >>= 1)
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
    }
  if ((threadIdx.x & 31u) == 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      s_box[threadIdx.x >> 5][a] = encode_ordered(lo[a]);
      s_box[threadIdx.x >> 5][3 + a] = encode_ordered(hi[a]);
    }
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    uint32_t v = s_box[0][threadIdx.x];
#pragma unroll
    for (int w = 1; w < kThreads / 32; ++w)
      v = threadIdx.x < 3 ? min(v, s_box[w][threadIdx.x]) : max(v, s_box[w][threadIdx.x]);
    box_part[blockIdx.x * 6 + threadIdx.x] = v;
  }
}

// S3 (D:A-OFFSET): exclusive scan of the histogram in ONE pass -- block-local scan plus
// decoupled look-back over tile aggregates -- instead of the paper's up-sweep / down-sweep.  Scans C+1
// entries (entry C counts 0) so that start[C] = total, and clears the histogram for the next build.
__global__ void __launch_bounds__(kThreads) k_scan_cells(uint32_t* __restrict__ count, uint32_t* __restrict__ start,
                                                         uint32_t C, ScanState st,
                                                         const uint32_t* __restrict__ box_part, uint32_t n_parts,
                                                         uint32_t* __restrict__ aabb) {
  __shared__ uint32_t s_scan[33];
  if (n_parts == 0 && blockIdx.x == 0 && threadIdx.x < 6) aabb[threadIdx.x] = threadIdx.x < 3 ? 0xffffffffu : 0u;  // no points
  if (threadIdx.x >= 32 && threadIdx.x < 64) {  // warp 1 folds this block's share of the bounding-box partials
    const uint32_t lane = threadIdx.x - 32;
    uint32_t v[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
    for (uint32_t q = blockIdx.x + lane * gridDim.x; q < n_parts; q += 32 * gridDim.x) {
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        v[a] = min(v[a], __ldg(box_part + 6 * q + a));
        v[3 + a] = max(v[3 + a], __ldg(box_part + 6 * q + 3 + a));
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        v[a] = min(v[a], __shfl_xor_sync(0xffffffffu, v[a], o));
        v[3 + a] = max(v[3 + a], __shfl_xor_sync(0xffffffffu, v[3 + a], o));
      }
    if (lane == 0 && blockIdx.x < n_parts) {
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        atomicMin(aabb + a, v[a]);
        atomicMax(aabb + 3 + a, v[3 + a]);
      }
    }
  }
  __shared__ uint32_t s_tile, s_base, s_epoch;
  if (threadIdx.x == 0) s_tile = scan_begin(st, &s_epoch);
  __syncthreads();
  const uint32_t tile = s_tile;
  st.epoch = s_epoch;
  const uint32_t first = tile * kScanTile + threadIdx.x * kScanItems;
  const bool full = first + kScanItems <= C;
  uint32_t v[kScanItems];
  if (full) {  // two 16-byte loads, two 16-byte clears
    const uint4 a = *reinterpret_cast<const uint4*>(count + first);
    const uint4 b = *reinterpret_cast<const uint4*>(count + first + 4);
    v[0] = a.x, v[1] = a.y, v[2] = a.z, v[3] = a.w, v[4] = b.x, v[5] = b.y, v[6] = b.z, v[7] = b.w;
    *reinterpret_cast<uint4*>(count + first) = make_uint4(0, 0, 0, 0);
    *reinterpret_cast<uint4*>(count + first + 4) = make_uint4(0, 0, 0, 0);
  } else {
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
      v[k] = 0u;
      if (first + k < C) {
        v[k] = count[first + k];
        count[first + k] = 0u;
      }
    }
  }
  uint32_t sum = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) sum += v[k];
  uint32_t total;
  uint32_t excl = block_exclusive_scan(sum, s_scan, &total);
  if (threadIdx.x < 32) {
    const uint32_t base = lookback_exclusive(st, tile, total);
    if (threadIdx.x == 0) {
      s_base = base;
      scan_end(st, gridDim.x);
    }
  }
  __syncthreads();
  excl += s_base;
  uint32_t o[kScanItems];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    o[k] = excl;
    excl += v[k];
  }
  if (full) {
    *reinterpret_cast<uint4*>(start + first) = make_uint4(o[0], o[1], o[2], o[3]);
    *reinterpret_cast<uint4*>(start + first + 4) = make_uint4(o[4], o[5], o[6], o[7]);
  } else {
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
      if (first + k <= C) start[first + k] = o[k];
  }
}

// S4a (P:433-439 count_sort_particle_index): slot_id[start[key] + rank] = id.
__global__ void __launch_bounds__(kThreads) k_scatter(const uint32_t* __restrict__ key, const uint32_t* __restrict__ rank,
                                                      const uint32_t* __restrict__ start, uint32_t n,
                                                      uint32_t* __restrict__ slot_id) {
  const uint32_t i = blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  slot_id[__ldg(start + __ldg(key + i)) + __ldg(rank + i)] = i;
}

// S4b: the atomic ranks are in arrival order; the canonical order is ascending id inside a cell
// (D:A-SORT).  Each slot counts the smaller ids of its cell's run (a run is ~8 ids) and moves there, carrying
// the physical copies of pos / vel (the paper keeps an index indirection instead).
__global__ void __launch_bounds__(kThreads) k_reorder(const uint32_t* __restrict__ key, const uint32_t* __restrict__ start,
                                                      const uint32_t* __restrict__ slot_id,
                                                      const float4* __restrict__ pos, const float4* __restrict__ vel,
                                                      uint32_t n, uint32_t* __restrict__ perm,
                                                      float4* __restrict__ posS, float4* __restrict__ velS) {
  const uint32_t s_raw = blockIdx.x * kThreads + threadIdx.x;
  const bool live = s_raw < n;
  const uint32_t s = live ? s_raw : n - 1u;  // idle lanes shadow the last slot (the warp-wide part below needs them)
  const uint32_t id = __ldg(slot_id + s);
  const uint32_t c = __ldg(key + id);
  const uint32_t s0 = __ldg(start + c), s1 = __ldg(start + c + 1);
  uint32_t smaller = 0;
  // A run is ~8 ids and every slot counts the smaller ids of its run on its own.  A long run (a crowded cell: the boid
  // cluster of config 5 has ~600 boids per cell; a degenerate input has everything in one) would make that quadratic
  // per thread, so the slots of a long run are ranked by the whole warp, one slot at a time, the lanes striding the run.
  const bool long_run = s1 - s0 > (uint32_t)kLongRun;
  if (!long_run)
    for (uint32_t t = s0; t < s1; ++t) smaller += (__ldg(slot_id + t) < id) ? 1u : 0u;
  uint32_t todo = __ballot_sync(0xffffffffu, long_run);
  const uint32_t lane = threadIdx.x & 31u;
  while (todo) {
    const int src = __ffs(todo) - 1;
    todo &= todo - 1u;
    const uint32_t id_s = __shfl_sync(0xffffffffu, id, src), a = __shfl_sync(0xffffffffu, s0, src),
                   e = __shfl_sync(0xffffffffu, s1, src);
    uint32_t cnt = 0;
    for (uint32_t t = a + lane; t < e; t += 32u) cnt += (__ldg(slot_id + t) < id_s) ? 1u : 0u;
    cnt = warp_sum_u32(cnt);
    if ((int)lane == src) smaller = cnt;
  }
  if (!live) return;
  const uint32_t dst = s0 + smaller;
  perm[dst] = id;
  posS[dst] = __ldg(pos + id);
  if (vel) velS[dst] = __ldg(vel + id);
}

// ---- S1-S5 in ONE block, for small grids (the Boid Space grid of every config; the particle grid of config 1) ---------
// Four launches per grid build (hash + histogram, scan, scatter, reorder) are launch latency when the grid is small:
// here one block of 1024 threads keeps the histogram / cell starts (C + 1 entries) and the arrival-ordered ids (n
// entries), 16 bits each, in shared memory and does all four steps between block barriers.  Same results bit for bit: keys, exclusive
// starts, canonical order (ascending id inside a cell, D:A-SORT), sorted copies, bounding box.
constexpr int kSmallThreads = 1024;
// counts, starts and ids all fit 16 bits (n <= 16384): (C + 2) * 2 + n * 2 bytes of shared memory.  One block zeroes,
// scans and writes out the whole cell table through one SM, so the win over four launches ends at a few thousand cells:
// measured on B200 with 64 000 boid cells (configs 2 and 4) the block takes 45-56 us against 33 us for the four kernels;
// at 4 096 cells (config 1, both grids) it equals them (16 us / 9 us) with six launches fewer per frame.
constexpr uint32_t kSmallMaxCells = 8192, kSmallMaxPoints = 16384;

__global__ void __launch_bounds__(kSmallThreads) k_grid_small(GridDesc g, const float4* __restrict__ pos,
                                                              const float4* __restrict__ vel, uint32_t n,
                                                              uint32_t* __restrict__ key, uint32_t* __restrict__ rank,
                                                              uint32_t* __restrict__ start, uint32_t* __restrict__ perm,
                                                              float4* __restrict__ posS, float4* __restrict__ velS,
                                                              uint32_t* __restrict__ aabb) {
  extern __shared__ uint32_t s_small[];
  __shared__ uint32_t s_scan[33];
  __shared__ uint32_t s_box[6];
  const uint32_t tid = threadIdx.x, C = g.C;
  const uint32_t cell_words = (C + 2u + 1u) >> 1;                       // C + 1 entries (+ pad), two per word
  uint16_t* s_cell = reinterpret_cast<uint16_t*>(s_small);              // histogram, then exclusive starts
  uint16_t* s_id = reinterpret_cast<uint16_t*>(s_small + cell_words);   // [n]: ids in arrival order, slot = start + rank
  for (uint32_t w = tid; w < cell_words; w += kSmallThreads) s_small[w] = 0u;
  if (tid < 6) s_box[tid] = tid < 3 ? 0xffffffffu : 0u;
  __syncthreads();
  // S1 + S2: key, rank = arrival order in the cell (a 32-bit atomic on the word that holds the cell's
  // 16-bit count: a count never reaches 65536, so the halves do not carry into each other); bounding box of the points
  float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
  for (uint32_t i = tid; i < n; i += kSmallThreads) {
    const float4 p = __ldg(pos + i);
    const uint32_t k = cell_hash(g, cell_coord(p.x, g.lo[0], g.cell, g.dim[0]), cell_coord(p.y, g.lo[1], g.cell, g.dim[1]),
                                 cell_coord(p.z, g.lo[2], g.cell, g.dim[2]));
    const uint32_t sh = 16u * (k & 1u);
    key[i] = k;
    rank[i] = (atomicAdd(s_small + (k >> 1), 1u << sh) >> sh) & 0xffffu;
    lo[0] = fminf(lo[0], p.x), lo[1] = fminf(lo[1], p.y), lo[2] = fminf(lo[2], p.z);
    hi[0] = fmaxf(hi[0], p.x), hi[1] = fmaxf(hi[1], p.y), hi[2] = fmaxf(hi[2], p.z);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1)
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
    }
  if ((tid & 31u) == 0u && tid < n) {  // a warp without a point keeps its +-3e38
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      atomicMin(s_box + a, encode_ordered(lo[a]));
      atomicMax(s_box + 3 + a, encode_ordered(hi[a]));
    }
  }
  __syncthreads();
  if (tid < 6) aabb[tid] = s_box[tid];
  // S3: exclusive scan of the C + 1 counts (entry C counts 0, so start[C] = n), a contiguous piece
  // per thread
  const uint32_t per = (C + 1u + kSmallThreads - 1u) / kSmallThreads;
  const uint32_t c0 = min(tid * per, C + 1u), c1 = min(c0 + per, C + 1u);
  uint32_t sum = 0;
  for (uint32_t c = c0; c < c1; ++c) sum += s_cell[c];
  uint32_t total;
  uint32_t run = block_exclusive_scan(sum, s_scan, &total);
  for (uint32_t c = c0; c < c1; ++c) {
    const uint32_t v = s_cell[c];
    s_cell[c] = (uint16_t)run;
    start[c] = run;
    run += v;
  }
  __syncthreads();
  // S4a: ids in arrival order
  for (uint32_t i = tid; i < n; i += kSmallThreads) s_id[(uint32_t)s_cell[key[i]] + rank[i]] = (uint16_t)i;
  __syncthreads();
  // S4b: canonical order inside a run = ascending id (D:A-SORT), with the physical copies of pos / vel
  for (uint32_t s = tid; s < n; s += kSmallThreads) {
    const uint32_t id = s_id[s];
    const uint32_t c = key[id];
    const uint32_t a = s_cell[c], e = s_cell[c + 1];
    uint32_t smaller = 0;
    for (uint32_t t = a; t < e; ++t) smaller += (uint32_t)s_id[t] < id ? 1u : 0u;
    const uint32_t dst = a + smaller;
    perm[dst] = id;
    posS[dst] = __ldg(pos + id);
    if (vel) velS[dst] = __ldg(vel + id);
  }
}

static size_t small_grid_smem(uint32_t C, uint32_t n) { return (size_t)((C + 3u) >> 1) * 4 + (size_t)((n + 1u) >> 1) * 4; }

// The velocity half of k_reorder on its own, for a grid that was built from the positions alone while the
// velocities were still on their way to the device (sph_simulate_host).  velS[.].w already holds rho (k_density).
__global__ void __launch_bounds__(kThreads) k_gather_vel(const uint32_t* __restrict__ perm, const float4* __restrict__ vel,
                                                         uint32_t n, float4* __restrict__ velS) {
  const uint32_t s = blockIdx.x * kThreads + threadIdx.x;
  if (s >= n) return;
  float4 v = __ldg(vel + __ldg(perm + s));
  v.w = velS[s].w;
  velS[s] = v;
}

// ---- N4: the paper's FIRST neighbour search, kept as a measured baseline (K7) -------------
// compute_hash_grid (Listing 5): hash_grid[cell * max_per_cell + slot] = particle id, slot = the cell's running count
// (hash_grid_tracker).  Particles that find their cell full are dropped and counted (the paper leaves that case open).
__global__ void __launch_bounds__(kThreads) k_hashgrid_fill(GridDesc g, const float4* __restrict__ pos, uint32_t n,
                                                            uint32_t cap, uint32_t* __restrict__ tracker,
                                                            uint32_t* __restrict__ hash_grid,
                                                            uint32_t* __restrict__ dropped) {
  const uint32_t i = blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  const float4 p = __ldg(pos + i);
  const uint32_t k = cell_hash(g, cell_coord(p.x, g.lo[0], g.cell, g.dim[0]), cell_coord(p.y, g.lo[1], g.cell, g.dim[1]),
                               cell_coord(p.z, g.lo[2], g.cell, g.dim[2]));
  const uint32_t slot = atomicAdd(tracker + k, 1u);
  if (slot < cap)
    hash_grid[(size_t)k * cap + slot] = i;
  else
    atomicAdd(dropped, 1u);
}

// compute_neighbor_list (Listings 6-7) reduced to its count: the 27 cells around the particle's own (cells outside the
// grid skipped, D:A-BOUND), every stored id a potential neighbour read through the index, r^2 < h^2.
__global__ void __launch_bounds__(kThreads) k_hashgrid_count(GridDesc g, float h2, const float4* __restrict__ pos,
                                                             uint32_t n, uint32_t cap,
                                                             const uint32_t* __restrict__ tracker,
                                                             const uint32_t* __restrict__ hash_grid,
                                                             uint32_t* __restrict__ ncount) {
  const uint32_t i = blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  const float4 pi = __ldg(pos + i);
  const int cx = cell_coord(pi.x, g.lo[0], g.cell, g.dim[0]);
  const int cy = cell_coord(pi.y, g.lo[1], g.cell, g.dim[1]);
  const int cz = cell_coord(pi.z, g.lo[2], g.cell, g.dim[2]);
  uint32_t cnt = 0;
  for (int z = max(cz - 1, 0); z <= min(cz + 1, g.dim[2] - 1); ++z)
    for (int y = max(cy - 1, 0); y <= min(cy + 1, g.dim[1] - 1); ++y)
      for (int x = max(cx - 1, 0); x <= min(cx + 1, g.dim[0] - 1); ++x) {
        const uint32_t k = cell_hash(g, x, y, z);
        const uint32_t m = min(__ldg(tracker + k), cap);
        const uint32_t* ids = hash_grid + (size_t)k * cap;
        for (uint32_t j = 0; j < m; ++j) {
          const float4 pj = __ldg(pos + __ldg(ids + j));
          cnt += dist2(pi.x - pj.x, pi.y - pj.y, pi.z - pj.z) < h2 ? 1u : 0u;
        }
      }
  ncount[i] = cnt;
}

// ---- N2: slab decomposition support -- ordered selection of the particles of a coordinate range --
// select_i = lo <= pos_i[axis] < hi.  Three small kernels: per-block counts, one-block exclusive scan of the counts,
// per-block ordered scatter; the output keeps ascending particle index, so a decomposed run is reproducible.
__device__ __forceinline__ bool in_range(const float4& p, int axis, float lo, float hi) {
  const float x = axis == 0 ? p.x : (axis == 1 ? p.y : p.z);
  return x >= lo && x < hi;
}

__global__ void __launch_bounds__(kThreads) k_range_count(const float4* __restrict__ pos, uint32_t n, int axis, float lo,
                                                          float hi, uint32_t* __restrict__ block_count) {
  const uint32_t i = blockIdx.x * kThreads + threadIdx.x;
  const bool sel = i < n && in_range(__ldg(pos + i), axis, lo, hi);
  const uint32_t c = __syncthreads_count(sel);
  if (threadIdx.x == 0) block_count[blockIdx.x] = c;
}

__global__ void __launch_bounds__(1024) k_range_scan(uint32_t* __restrict__ block_count, uint32_t nb,
                                                     uint32_t* __restrict__ total) {
  __shared__ uint32_t s_scan[33];
  uint32_t carry = 0;
  for (uint32_t base = 0; base < nb; base += 1024) {
    const uint32_t j = base + threadIdx.x;
    const uint32_t v = j < nb ? block_count[j] : 0u;
    uint32_t sum;
    const uint32_t ex = block_exclusive_scan(v, s_scan, &sum);
    if (j < nb) block_count[j] = carry + ex;
    carry += sum;
  }
  if (threadIdx.x == 0) *total = carry;
}

__global__ void __launch_bounds__(kThreads) k_range_scatter(const float4* __restrict__ pos, const float4* __restrict__ vel,
                                                            uint32_t n, int axis, float lo, float hi,
                                                            const uint32_t* __restrict__ block_offset,
                                                            float4* __restrict__ out_pos, float4* __restrict__ out_vel,
                                                            uint32_t capacity) {
  __shared__ uint32_t s_scan[33];
  const uint32_t i = blockIdx.x * kThreads + threadIdx.x;
  float4 p = make_float4(0.f, 0.f, 0.f, 0.f);
  bool sel = false;
  if (i < n) {
    p = __ldg(pos + i);
    sel = in_range(p, axis, lo, hi);
  }
  uint32_t total;
  const uint32_t ex = block_exclusive_scan(sel ? 1u : 0u, s_scan, &total);
  const uint32_t dst = block_offset[blockIdx.x] + ex;
  if (sel && dst < capacity) {
    out_pos[dst] = p;
    if (vel) out_vel[dst] = __ldg(vel + i);
  }
}

}  // namespace

uint32_t grid_scan_tiles(uint32_t C) { return (C + 1 + kScanTile - 1) / kScanTile; }

void grid_init() {
  cudaFuncSetAttribute(k_grid_small, cudaFuncAttributeMaxDynamicSharedMemorySize,
                       (int)small_grid_smem(kSmallMaxCells, kSmallMaxPoints));
}

void launch_build_grid(const GridDesc& g, GridBuf& b, const float4* pos, const float4* vel, uint32_t n,
                       ScanState& scan, cudaStream_t s, Prof* prof, bool boid_grid) {
  const uint32_t blocks = (n + kThreads - 1) / kThreads;
  const int k0 = boid_grid ? K_BOID_HASH_COUNT : K_HASH_COUNT;
  if (n > 0 && n <= kSmallMaxPoints && g.C <= kSmallMaxCells) {  // one launch instead of four
    prof->begin(boid_grid ? K_BOID_GRID_SMALL : K_GRID_SMALL, s);
    k_grid_small<<<1, kSmallThreads, small_grid_smem(g.C, n), s>>>(g, pos, vel, n, b.key, b.rank, b.start, b.perm,
                                                                    b.posS, b.velS, b.aabb);
    prof->end(s);
    b.aabb_now = b.aabb;
    return;
  }
  if (n > 0) {
    prof->begin(k0 + 0, s);
    k_hash_count<<<blocks, kThreads, 0, s>>>(g, pos, n, b.key, b.rank, b.count, b.box_part, b.aabb);
    prof->end(s);
  }
  const uint32_t tiles = grid_scan_tiles(g.C);
  prof->begin(k0 + 1, s);
  k_scan_cells<<<tiles, kThreads, 0, s>>>(b.count, b.start, g.C, scan, b.box_part, n > 0 ? blocks : 0u, b.aabb);
  prof->end(s);
  if (n > 0) {
    prof->begin(k0 + 2, s);
    k_scatter<<<blocks, kThreads, 0, s>>>(b.key, b.rank, b.start, n, b.slot_id);
    prof->end(s);
    prof->begin(k0 + 3, s);
    k_reorder<<<blocks, kThreads, 0, s>>>(b.key, b.start, b.slot_id, pos, vel, n, b.perm, b.posS, b.velS);
    prof->end(s);
  }
  b.aabb_now = b.aabb;
}

void launch_gather_vel(const GridBuf& b, const float4* vel, uint32_t n, cudaStream_t s, Prof* prof) {
  if (n == 0) return;
  prof->begin(K_GATHER_VEL, s);
  k_gather_vel<<<(n + kThreads - 1) / kThreads, kThreads, 0, s>>>(b.perm, vel, n, b.velS);
  prof->end(s);
}

void launch_hashgrid_count(const GridDesc& g, float h2, const float4* pos, uint32_t n, uint32_t cap, uint32_t* tracker,
                           uint32_t* hash_grid, uint32_t* dropped, uint32_t* ncount, cudaStream_t s, Prof* prof) {
  cudaMemsetAsync(tracker, 0, (size_t)g.C * 4, s);
  cudaMemsetAsync(dropped, 0, 4, s);
  if (n == 0) return;
  const uint32_t blocks = (n + kThreads - 1) / kThreads;
  prof->begin(K_HASHGRID_FILL, s);
  k_hashgrid_fill<<<blocks, kThreads, 0, s>>>(g, pos, n, cap, tracker, hash_grid, dropped);
  prof->end(s);
  prof->begin(K_HASHGRID_COUNT, s);
  k_hashgrid_count<<<blocks, kThreads, 0, s>>>(g, h2, pos, n, cap, tracker, hash_grid, ncount);
  prof->end(s);
}

void launch_pack_range(const float4* pos, const float4* vel, uint32_t n, int axis, float lo, float hi,
                       uint32_t* block_count, uint32_t* total_dev, float4* out_pos, float4* out_vel, uint32_t capacity,
                       cudaStream_t s, Prof* prof) {
  const uint32_t blocks = (n + kThreads - 1) / kThreads;
  if (blocks == 0) {
    cudaMemsetAsync(total_dev, 0, 4, s);
    return;
  }
  prof->begin(K_RANGE_COUNT, s);
  k_range_count<<<blocks, kThreads, 0, s>>>(pos, n, axis, lo, hi, block_count);
  prof->end(s);
  prof->begin(K_RANGE_SCAN, s);
  k_range_scan<<<1, 1024, 0, s>>>(block_count, blocks, total_dev);
  prof->end(s);
  prof->begin(K_RANGE_SCATTER, s);
  k_range_scatter<<<blocks, kThreads, 0, s>>>(pos, vel, n, axis, lo, hi, block_count, out_pos, out_vel, capacity);
  prof->end(s);
}

}  // namespace sphb
