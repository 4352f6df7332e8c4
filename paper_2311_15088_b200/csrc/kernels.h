// kernels.h -- host-side launchers of libsphboid's CUDA kernels (internal; the public ABI is include/sphboid.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"

namespace sphb {

struct SphConst {       // values every SPH kernel needs, precomputed once on the host
  GridDesc grid;        // particle grid, cell = h
  float h, h2;          // h2 = h*h in binary32 (D:A-FP)
  float mass, rho0, stiffness, viscosity;
  float mass_c6;        // m * 315/(64 pi h^9), binary64 rounded once
  float gravity[3], dt, damp;
  float box_min[3], box_max[3];
};

struct BoidConst {
  GridDesc grid;        // Boid Space grid, cell = max(visible, protect, push radius) (D:C-BGRID)
  float protect, visible, prot2, vis2;
  float w_sep, w_ali, w_coh, min_speed, max_speed, edge_turn, sph_factor;
  float push_radius, w_push;
  float space_min[3], space_max[3];
  int reach_push;       // ceil(push_radius / h) particle cells
};

struct ObstacleConst {  // N4: Obstacle Grid, D:C-OBST
  float origin[3], cell;
  int dims[3];
  float w_obs, heavy;
};

struct McConst {
  float origin[3], spacing;
  uint32_t G;
  float R, R2, rbar, iso;
  int reach;            // ceil(R / h) particle cells (D:A-R)
  uint32_t cube_lo[3], cube_hi[3];  // cubes that are polygonised: lo <= index < hi per axis (mc_set_cube_range)
};

// Kernel ids for the per-kernel timing that bench.py's roofline object is built from (sph_profile_*).
enum KernelId {
  K_HASH_COUNT = 0, K_SCAN_CELLS, K_SCATTER, K_REORDER,          // particle grid
  K_BOID_HASH_COUNT, K_BOID_SCAN_CELLS, K_BOID_SCATTER, K_BOID_REORDER,  // same kernels on the Boid Space grid
  K_GRID_SMALL, K_BOID_GRID_SMALL, K_GATHER_VEL,
  K_DENSITY, K_DENSITY_BRICK, K_BOID_DENSITY, K_FORCE_LIST, K_FORCE_MASKS, K_BOID_STEP, K_BOID_OBSTACLES,
  K_VOXEL_SDF, K_VOXEL_SDF_TILES, K_MC_SIGNS, K_MC_COUNT, K_MC_EMIT, K_MC_EDGE_SCAN, K_MC_VERTICES, K_MC_EMIT_INDICES,
  K_ZERO_U32, K_CC_INIT, K_CC_LINK, K_CC_FLATTEN, K_CC_COUNT, K_CC_LARGEST,  // N3 connectivity
  K_HASHGRID_FILL, K_HASHGRID_COUNT, K_RANGE_COUNT, K_RANGE_SCAN, K_RANGE_SCATTER,
  K_NUM_KERNELS
};


// Launch bookkeeping: a counter always; when `on`, a CUDA event before and after every launch, recorded on
// the launching stream (the kernels of one call are serialised on that stream anyway).
struct Prof {
  uint64_t launches;
  bool on;
  struct Rec { int kid; cudaEvent_t a, b; };
  Rec* recs;
  uint32_t used, cap;
  bool open;
  double total_ms[K_NUM_KERNELS];
  uint64_t count[K_NUM_KERNELS];
  void begin(int kid, cudaStream_t s);
  void end(cudaStream_t s);
};

// Scratch of one grid (particles or boids).
struct GridBuf {
  uint32_t* key;        // [n] cell of each point (caller order)
  uint32_t* rank;       // [n] arrival rank inside the cell (atomic order)
  uint32_t* count;      // [C] histogram, zero between builds
  uint32_t* start;      // [C+1] exclusive starts
  uint32_t* slot_id;    // [n] ids in arrival order
  uint32_t* perm;       // [n] sorted slot -> id, ascending id inside a cell (D:A-SORT)
  float4* posS;         // [n] cell-sorted copies
  float4* velS;
  uint32_t* aabb;       // [2][6] bounding box of the points (min xyz, max xyz; order-preserving encoding), two slots
  uint32_t* box_part;   // [ceil(n/256)][6] per-block partial bounding boxes of the hash kernel
  int slot;             // slot the NEXT build fills (the scan of each build empties the other one)
  const uint32_t* aabb_now;  // slot of the last build
};

// Stored neighbour list (sph.cu): rows list[k * stride + i] of 16-bit entries, cnt[i] entries per sorted particle i.
struct NbrList {
  uint16_t* list;       // [nbr_rows() * stride]
  uint16_t* cnt;        // [n]
  uint32_t stride;      // elements between rows, a multiple of 64
};

// grid.cu
void launch_build_grid(const GridDesc& g, GridBuf& b, const float4* pos, const float4* vel, uint32_t n,
                       ScanState& scan, cudaStream_t s, Prof* prof, bool boid_grid);
uint32_t grid_scan_tiles(uint32_t C);
void grid_init();  // once per device: opt in to the dynamic shared memory of the one-block grid build
void launch_gather_vel(const GridBuf& b, const float4* vel, uint32_t n, cudaStream_t s, Prof* prof);
void launch_pack_range(const float4* pos, const float4* vel, uint32_t n, int axis, float lo, float hi,
                       uint32_t* block_count, uint32_t* total_dev, float4* out_pos, float4* out_vel, uint32_t capacity,
                       cudaStream_t s, Prof* prof);
void launch_hashgrid_count(const GridDesc& g, float h2, const float4* pos, uint32_t n, uint32_t cap, uint32_t* tracker,
                           uint32_t* hash_grid, uint32_t* dropped, uint32_t* ncount, cudaStream_t s, Prof* prof);
// sph.cu
void launch_density(const SphConst& c, const GridBuf& b, uint32_t n, float* rhoS, float* density_out,
                    uint32_t* ncount_out, const NbrList* nl, cudaStream_t s, Prof* prof);
uint32_t nbr_rows();
void launch_boid_density(const SphConst& c, const GridBuf& pg, const GridBuf& bg, uint32_t nb, float* rho_bS,
                         cudaStream_t s, Prof* prof);
void launch_force_list(const SphConst& c, const BoidConst* bc, const GridBuf& pg, const GridBuf& bg, uint32_t n,
                       uint32_t nb, const float* rhoS, const float* rho_bS, float4* pos, float4* vel, float4* accel_out,
                       uint32_t* touched_out, const NbrList& nl, cudaStream_t s, Prof* prof);
// sph_brick.cu: S6 with a brick of cells per block staged in shared memory, S8-S10 from the masks it stores.  masks = one
// word per target and chunk of 32 candidates, up to kNbrMaskWords words per sorted particle: masks[w * stride + i].
constexpr int kNbrMaskWords = 32;
void launch_density_brick(const SphConst& c, const GridBuf& b, uint32_t n, float* rhoS, float* density_out,
                          uint32_t* ncount_out, uint32_t* masks, uint32_t stride, cudaStream_t s, Prof* prof);
void launch_force_masks(const SphConst& c, const BoidConst* bc, const GridBuf& pg, const GridBuf& bg, uint32_t n,
                        uint32_t nb, const float* rhoS, const float* rho_bS, float4* pos, float4* vel, float4* accel_out,
                        uint32_t* touched_out, const uint32_t* masks, uint32_t stride, cudaStream_t s, Prof* prof);
// boid.cu
void launch_boid_step(const SphConst& c, const BoidConst& bc, const GridBuf& pg, const GridBuf& bg, uint32_t n,
                      uint32_t nb, const float* rhoS, const float* rho_bS, float4* bpos, float4* bvel,
                      float4* dv_parts, cudaStream_t s, Prof* prof);
void launch_boid_obstacles(const ObstacleConst& oc, const float4* normals, const BoidConst& bc, const float4* bpos,
                           float4* bvel, uint32_t nb, cudaStream_t s, Prof* prof);
// mc.cu
void upload_mc_tables();
void mc_table_host(int8_t* tri, uint8_t* ntri);
bool launch_voxel_sdf(const SphConst& c, const McConst& m, const GridBuf& pg, float* phi,
                      uint32_t* sign_bits /* optional */, int variant, cudaStream_t s,
                      Prof* prof);  // true if it also filled the corner sign bit field
void launch_mc_polygonise(const McConst& m, const float* phi, uint32_t* bits, bool bits_ready, float* tris,
                          uint32_t capacity, uint32_t* n_tris_dev, uint2* work, uint32_t* n_work, ScanState& scan,
                          cudaStream_t s, Prof* prof);
void launch_mc_indexed(const McConst& m, const float* phi, uint32_t* bits, bool bits_ready, uint32_t* prefix,
                       float* verts, float* normals, uint32_t vert_capacity, uint32_t* indices, uint32_t tri_capacity,
                       uint32_t* n_verts_dev, uint32_t* n_tris_dev, uint2* work, uint32_t* n_work, ScanState& scan,
                       cudaStream_t s, Prof* prof);
void launch_mesh_components(const uint32_t* indices, uint32_t n_tris, uint32_t n_verts, uint32_t* label,
                            uint32_t* tri_count, uint32_t* result /* [3] */, cudaStream_t s, Prof* prof);
uint32_t mc_word_tiles(uint32_t G);    // look-back tiles of the edge scan
uint64_t mc_num_segments(uint32_t G);  // size of the active-segment work list
uint64_t mc_bits_words(uint32_t G);  // size of the corner sign bit field
uint32_t mc_num_tiles(uint32_t G);

}  // namespace sphb
