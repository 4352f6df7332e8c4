// noalloc.cu -- sph_build_grid_static: S1-S5 (D:A-DIMS, D:A-SORT) for callers that may not
// allocate: no context, no cudaMalloc / cudaFree, no allocating library routine.  It is the one-block grid build of
// grid.cu (k_grid_small) with its global scratch -- the key and the arrival rank of every point -- in a file-scope
// __device__ array instead of a context's buffers.  The caller passes the positions and the three output arrays.
//
// The array is shared by every call on a device and keeps the last call's contents.  Nothing in it has to start at
// zero: the kernel writes key[i] and rank[i] for every i < n before it reads them, and the histogram it does zero lives
// in shared memory.  Two calls that overlap on one GPU (different streams, or different host threads) race on it.
#include <math.h>
#include <stdio.h>

#include <mutex>

#include "../../include/sphboid.h"
#include "common.cuh"

// Stated maximum: SPH_STATIC_MAX_POINTS = 16 384 points, SPH_STATIC_MAX_CELLS = 8 192 cells.  Scratch = 2 x 16 384 x 4 B =
// 128 KB of device memory that every GPU which loads the library holds until exit.  key[max points], rank[max points].
static __device__ __align__(256) uint32_t g_static_scratch[2 * SPH_STATIC_MAX_POINTS];

namespace sphb {

namespace {

constexpr int kStaticThreads = 1024;
// shared memory = (C + 2) x 2 + n x 2 bytes <= 48 KB + 1 KB at the maximum
constexpr uint32_t kStaticMaxPoints = SPH_STATIC_MAX_POINTS, kStaticMaxCells = SPH_STATIC_MAX_CELLS;

// k_grid_small of grid.cu without the sorted copies and the bounding box; same keys, starts and canonical order.
__global__ void __launch_bounds__(kStaticThreads) k_grid_static(GridDesc g, const float4* __restrict__ pos, uint32_t n,
                                                                uint32_t* __restrict__ scratch,
                                                                uint32_t* __restrict__ cell_of_particle,
                                                                uint32_t* __restrict__ start,
                                                                uint32_t* __restrict__ perm) {
  extern __shared__ uint32_t s_static[];
  __shared__ uint32_t s_scan[33];
  uint32_t* key = scratch;
  uint32_t* rank = scratch + kStaticMaxPoints;
  const uint32_t tid = threadIdx.x, C = g.C;
  const uint32_t cell_words = (C + 2u + 1u) >> 1;                        // C + 1 entries (+ pad), two per word
  uint16_t* s_cell = reinterpret_cast<uint16_t*>(s_static);              // histogram, then exclusive starts
  uint16_t* s_id = reinterpret_cast<uint16_t*>(s_static + cell_words);   // [n]: ids in arrival order
  for (uint32_t w = tid; w < cell_words; w += kStaticThreads) s_static[w] = 0u;  // what must start at zero
  __syncthreads();
  // S1 + S2: key; rank = arrival order in the cell (a 32-bit atomic on the word holding the
  // cell's 16-bit count: a count never reaches 65536, so the halves do not carry into each other)
  for (uint32_t i = tid; i < n; i += kStaticThreads) {
    const float4 p = __ldg(pos + i);
    const uint32_t k = cell_hash(g, cell_coord(p.x, g.lo[0], g.cell, g.dim[0]), cell_coord(p.y, g.lo[1], g.cell, g.dim[1]),
                                 cell_coord(p.z, g.lo[2], g.cell, g.dim[2]));
    const uint32_t sh = 16u * (k & 1u);
    key[i] = k;
    cell_of_particle[i] = k;
    rank[i] = (atomicAdd(s_static + (k >> 1), 1u << sh) >> sh) & 0xffffu;
  }
  __syncthreads();
  // S3: exclusive scan of the C + 1 counts (entry C counts 0, so start[C] = n)
  const uint32_t per = (C + 1u + kStaticThreads - 1u) / kStaticThreads;
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
  for (uint32_t i = tid; i < n; i += kStaticThreads) s_id[(uint32_t)s_cell[key[i]] + rank[i]] = (uint16_t)i;
  __syncthreads();
  // S4b: canonical order inside a cell = ascending id (D:A-SORT)
  for (uint32_t s = tid; s < n; s += kStaticThreads) {
    const uint32_t id = s_id[s];
    const uint32_t c = key[id];
    const uint32_t a = s_cell[c], e = s_cell[c + 1];
    uint32_t smaller = 0;
    for (uint32_t t = a; t < e; ++t) smaller += (uint32_t)s_id[t] < id ? 1u : 0u;
    perm[a + smaller] = id;
  }
}

size_t static_smem(uint32_t C, uint32_t n) { return (size_t)((C + 3u) >> 1) * 4 + (size_t)((n + 1u) >> 1) * 4; }

// Set-up, once per device, with that device current: the array's name is a host-side stand-in in host code, the
// device address comes from cudaGetSymbolAddress.  Neither call allocates.
constexpr int kMaxDevices = 64;
std::mutex g_setup_lock;
uint32_t* g_scratch_ptr[kMaxDevices] = {};

thread_local char t_static_err[160] = "";

int static_fail(int code, const char* msg) {
  snprintf(t_static_err, sizeof(t_static_err), "%s", msg);
  return code;
}

int static_cuda_fail(cudaError_t e, const char* where) {
  snprintf(t_static_err, sizeof(t_static_err), "%s: %s", where, cudaGetErrorString(e));
  return SPH_E_CUDA;
}

int static_setup(int device, uint32_t** out) {
  std::lock_guard<std::mutex> hold(g_setup_lock);
  if (!g_scratch_ptr[device]) {
    uint32_t* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess) return static_cuda_fail(e, "cudaGetSymbolAddress(g_static_scratch)");
    e = cudaFuncSetAttribute(k_grid_static, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)static_smem(kStaticMaxCells, kStaticMaxPoints));
    if (e != cudaSuccess) return static_cuda_fail(e, "cudaFuncSetAttribute(k_grid_static)");
    g_scratch_ptr[device] = p;
  }
  *out = g_scratch_ptr[device];
  return SPH_OK;
}

}  // namespace

}  // namespace sphb

extern "C" {

const char* sph_static_last_error(void) { return sphb::t_static_err; }

int sph_build_grid_static(const float* box_min, const float* box_max, float h, const void* pos, uint32_t n,
                          void* stream, uint32_t* cell_of_particle, uint32_t* perm, uint32_t* cell_start,
                          uint32_t cell_start_entries) {
  using namespace sphb;
  if (!box_min || !box_max) return static_fail(SPH_E_INVALID, "box_min / box_max is NULL");
  if (!(h > 0.0f)) return static_fail(SPH_E_INVALID, "h must be positive");
  // D:A-DIMS: dim = max(1, ceil((hi - lo)/h)) in host double -- the rule of sph_create
  GridDesc g;
  g.cell = h;
  uint64_t C = 1;
  for (int a = 0; a < 3; ++a) {
    if (!(box_max[a] > box_min[a])) return static_fail(SPH_E_INVALID, "empty box");
    g.lo[a] = box_min[a];
    double d = ceil(((double)box_max[a] - (double)box_min[a]) / (double)h);
    if (!(d >= 1.0)) d = 1.0;
    if (d > 65535.0) return static_fail(SPH_E_CAPACITY, "grid exceeds SPH_STATIC_MAX_CELLS (8192) cells");
    g.dim[a] = (int)d;
    C *= (uint64_t)g.dim[a];
  }
  if (C > kStaticMaxCells) return static_fail(SPH_E_CAPACITY, "grid exceeds SPH_STATIC_MAX_CELLS (8192) cells");
  if (n > kStaticMaxPoints) return static_fail(SPH_E_CAPACITY, "n exceeds SPH_STATIC_MAX_POINTS (16384)");
  g.C = (uint32_t)C;
  if (!cell_start || (n > 0 && (!pos || !cell_of_particle || !perm)))
    return static_fail(SPH_E_INVALID, "pos / cell_of_particle / perm / cell_start is NULL");
  if (reinterpret_cast<uintptr_t>(pos) & 15u) return static_fail(SPH_E_INVALID, "pos is not 16-byte aligned");
  if (cell_start_entries < g.C + 1u) return static_fail(SPH_E_INVALID, "cell_start holds fewer than C + 1 entries");
  int device = 0;
  cudaError_t e = cudaGetDevice(&device);
  if (e != cudaSuccess) return static_cuda_fail(e, "cudaGetDevice");
  if (device < 0 || device >= kMaxDevices) return static_fail(SPH_E_INVALID, "device ordinal out of range");
  uint32_t* scratch = nullptr;
  const int rc = static_setup(device, &scratch);
  if (rc != SPH_OK) return rc;
  k_grid_static<<<1, kStaticThreads, static_smem(g.C, n), (cudaStream_t)stream>>>(
      g, (const float4*)pos, n, scratch, cell_of_particle, cell_start, perm);
  e = cudaGetLastError();
  if (e != cudaSuccess) return static_cuda_fail(e, "k_grid_static launch");
  return SPH_OK;
}

}  // extern "C"
