// api.cu -- the C ABI of libsphboid (include/sphboid.h): context, scratch, argument checks, sequencing.
#include "../../include/sphboid.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "kernels.h"

using namespace sphb;

struct sph_ctx {
  int device;
  sph_params p;
  SphConst sc;
  GridBuf pg;   // particle grid
  GridBuf bg;   // boid grid
  uint32_t boid_cells_cap;
  float* rhoS;
  float* rho_bS;
  float* phi;   // [Gmax^3]
  uint32_t* mc_bits;  // [ceil(Gmax/32) * Gmax^2] corner sign bits of the surface pass
  NbrList nbr;           // stored neighbour list of the last sph_step
  int force_variant;     // 0 = cost model, 1 = stored neighbour list (k_density + k_force_list), 2 = neighbour masks (k_density_brick + k_force_masks)
  uint32_t cube_lo[3], cube_hi[3];  // mc_set_cube_range: cubes the polygoniser handles (default: all)
  int sdf_variant;       // 0 = cost model, 1 = per-corner, 2 = corner tiles (mc_set_sdf_variant)
  uint32_t* n_tris_dev;
  uint32_t* mc_prefix;   // [words of mc_bits] vertex-id prefix of the indexed mesh (N3)
  uint32_t* n_verts_dev;
  uint2* mc_work;        // [segments] active-segment work list of the surface pass (segment, first triangle)
  uint32_t* mc_nwork;    // [2] its length, two counters used alternately
  bool bits_ready;       // mc_bits was filled by the SDF kernel of the mc_extract in progress
  ScanState scan;
  uint32_t max_tiles;
  // sequencing
  const void* grid_pos;
  const void* grid_vel;
  uint32_t grid_n;
  bool grid_fresh;       // pg holds a grid of (grid_pos, grid_n) and positions have not moved since
  bool step_state;       // pg/rhoS hold the step-start state of the last sph_step
  BoidConst bc;
  uint32_t *pack_blocks, *pack_total;  // N2: scratch of sph_pack_range (lazy)
  uint32_t *hg_tracker, *hg_grid, *hg_dropped;  // N4 baseline: the paper's unsorted fixed-capacity hash grid (lazy)
  uint32_t hg_cap;
  uint32_t *cc_count, *cc_result;      // N3 connectivity: per-root triangle counts (lazy, grows), result words
  uint32_t cc_cap;
  ObstacleConst oc;      // N4: Obstacle Grid set by boid_set_obstacles (normals stay caller-owned)
  const float4* obst_normals;
  bool boid_state;       // bg/rho_bS hold the boids given to the last sph_step
  bool rho_event;        // ev_rho was recorded by that sph_step (boid_step may then use the side stream)
  const void* boid_pos;
  uint32_t boid_n;
  cudaStream_t side;     // the boid grid + probe density of sph_step run here, beside k_density
  cudaStream_t surf;     // mc_extract_async runs the surface pass here, beside the next frame's SPH step
  cudaEvent_t ev_surf_fork, ev_surf_done;
  cudaStream_t up;       // sph_simulate_host uploads the velocities here while the grid build and k_density run
  cudaEvent_t ev_up_go, ev_up_done;
  bool vel_pending;      // the grid was built from positions alone: sph_step gathers velS after ev_up_done
  bool surf_pending;     // a surface pass was forked and nothing has waited for it yet
  uint32_t surf_capacity;
  ScanState scan_mc;     // look-back state of the surface pass (its scans may run beside the grid scans)
  cudaEvent_t ev_fork, ev_join, ev_rho;  // ev_rho: k_density of the last sph_step has finished
  Prof prof;
  char err[256];
  // staging for the *_host entry point
  float4 *h_pos, *h_vel, *h_bpos, *h_bvel;
  float* h_tris;
  uint32_t h_tris_cap;
};

namespace sphb {

void Prof::begin(int kid, cudaStream_t s) {
  ++launches;
  if (!on) return;
  if (used == cap) {
    const uint32_t ncap = cap ? cap * 2 : 1024;
    Rec* nr = (Rec*)realloc(recs, (size_t)ncap * sizeof(Rec));
    if (!nr) {
      on = false;
      return;
    }
    recs = nr, cap = ncap;
  }
  Rec& r = recs[used];
  r.kid = kid;
  if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) {
    on = false;
    return;
  }
  cudaEventRecord(r.a, s);
  ++used;
  open = true;
}

void Prof::end(cudaStream_t s) {
  if (!open) return;
  cudaEventRecord(recs[used - 1].b, s);
  open = false;
}

}  // namespace sphb

namespace {

int fail(sph_ctx* c, int code, const char* msg) {
  if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
  return code;
}

int cuda_fail(sph_ctx* c, cudaError_t e, const char* where) {
  if (c) snprintf(c->err, sizeof(c->err), "%s: %s", where, cudaGetErrorString(e));
  return SPH_E_CUDA;
}

#define CK(call)                                           \
  do {                                                     \
    cudaError_t e_ = (call);                               \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); \
  } while (0)

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// D:A-DIMS: dim = max(1, ceil((hi - lo)/cell)) in host double.
bool make_grid(GridDesc& g, const float* lo, const float* hi, float cell) {
  if (!(cell > 0.0f)) return false;
  g.cell = cell;
  uint64_t C = 1;
  for (int a = 0; a < 3; ++a) {
    if (!(hi[a] > lo[a])) return false;
    g.lo[a] = lo[a];
    double d = ceil(((double)hi[a] - (double)lo[a]) / (double)cell);
    if (!(d >= 1.0)) d = 1.0;
    if (d > 65535.0) return false;
    g.dim[a] = (int)d;
    C *= (uint64_t)g.dim[a];
  }
  if (C > (1ull << 30)) return false;
  g.C = (uint32_t)C;
  return true;
}

int alloc_grid(sph_ctx* ctx, GridBuf& b, uint32_t n, uint32_t C) {
  const size_t nn = std::max<uint32_t>(n, 1);
  CK(cudaMalloc(&b.key, nn * 4));
  CK(cudaMalloc(&b.rank, nn * 4));
  CK(cudaMalloc(&b.count, ((size_t)C + 8) * 4));
  CK(cudaMalloc(&b.start, ((size_t)C + 9) * 4));
  CK(cudaMalloc(&b.slot_id, nn * 4));
  CK(cudaMalloc(&b.perm, nn * 4));
  CK(cudaMalloc(&b.posS, nn * 16));
  CK(cudaMalloc(&b.velS, nn * 16));
  CK(cudaMalloc(&b.aabb, 12 * 4));
  CK(cudaMalloc(&b.box_part, ((nn + 255) / 256) * 6 * 4));
  {
    const uint32_t empty[12] = {~0u, ~0u, ~0u, 0u, 0u, 0u, ~0u, ~0u, ~0u, 0u, 0u, 0u};
    CK(cudaMemcpy(b.aabb, empty, sizeof(empty), cudaMemcpyHostToDevice));
  }
  b.slot = 0;
  b.aabb_now = b.aabb;
  CK(cudaMemset(b.count, 0, ((size_t)C + 8) * 4));
  CK(cudaMemset(b.start, 0, ((size_t)C + 9) * 4));
  return SPH_OK;
}

void free_grid(GridBuf& b) {
  cudaFree(b.key), cudaFree(b.rank), cudaFree(b.count), cudaFree(b.start);
  cudaFree(b.slot_id), cudaFree(b.perm), cudaFree(b.posS), cudaFree(b.velS), cudaFree(b.aabb), cudaFree(b.box_part);
  memset(&b, 0, sizeof(b));
}

int set_boid_params(sph_ctx* ctx, const boid_params* bp) {
  if (!bp) return fail(ctx, SPH_E_INVALID, "boid_params is NULL");
  BoidConst& bc = ctx->bc;
  float cell = std::max(bp->visible_range, std::max(bp->protect_range, bp->push_radius));  // D:C-BGRID
  if (!(cell > 0.0f) || !(bp->push_radius > 0.0f) || !(bp->visible_range > 0.0f) || !(bp->protect_range > 0.0f))
    return fail(ctx, SPH_E_INVALID, "boid ranges must be positive");
  GridDesc g;
  if (!make_grid(g, bp->space_min, bp->space_max, cell)) return fail(ctx, SPH_E_INVALID, "bad Boid Space");
  if (g.C > ctx->boid_cells_cap) {
    // re-size the boid grid's cell arrays (host-side decision, rare: only when the ranges shrink)
    cudaFree(ctx->bg.count), cudaFree(ctx->bg.start);
    CK(cudaMalloc(&ctx->bg.count, ((size_t)g.C + 8) * 4));
    CK(cudaMalloc(&ctx->bg.start, ((size_t)g.C + 9) * 4));
    CK(cudaMemset(ctx->bg.count, 0, ((size_t)g.C + 8) * 4));
    ctx->boid_cells_cap = g.C;
    const uint32_t tiles = grid_scan_tiles(g.C);
    if (tiles > ctx->max_tiles) {
      cudaFree(ctx->scan.status);
      CK(cudaMalloc(&ctx->scan.status, (size_t)tiles * 8));
      CK(cudaMemset(ctx->scan.status, 0, (size_t)tiles * 8));
      ctx->max_tiles = tiles;
    }
  }
  bc.grid = g;
  bc.protect = bp->protect_range, bc.visible = bp->visible_range;
  bc.prot2 = bp->protect_range * bp->protect_range;
  bc.vis2 = bp->visible_range * bp->visible_range;
  bc.w_sep = bp->w_sep, bc.w_ali = bp->w_ali, bc.w_coh = bp->w_coh;
  bc.min_speed = bp->min_speed, bc.max_speed = bp->max_speed, bc.edge_turn = bp->edge_turn;
  bc.sph_factor = bp->sph_factor, bc.push_radius = bp->push_radius, bc.w_push = bp->w_push;
  for (int a = 0; a < 3; ++a) bc.space_min[a] = bp->space_min[a], bc.space_max[a] = bp->space_max[a];
  int r = (int)ceil((double)bp->push_radius / (double)ctx->p.h);
  bc.reach_push = r < 1 ? 1 : r;
  return SPH_OK;
}

int make_mc(sph_ctx* ctx, const mc_params* mp, McConst& m) {
  if (!mp) return fail(ctx, SPH_E_INVALID, "mc_params is NULL");
  if (mp->n_point_per_axis > ctx->p.max_mc_points_per_axis)
    return fail(ctx, SPH_E_INVALID, "n_point_per_axis exceeds max_mc_points_per_axis");
  if (!(mp->radius > 0.0f)) return fail(ctx, SPH_E_INVALID, "mc radius must be positive");
  if (!(mp->spacing > 0.0f)) return fail(ctx, SPH_E_INVALID, "mc spacing must be positive");
  for (int a = 0; a < 3; ++a) m.origin[a] = mp->origin[a];
  m.spacing = mp->spacing;
  m.G = mp->n_point_per_axis;
  m.R = mp->radius;
  m.R2 = mp->radius * mp->radius;
  m.rbar = mp->particle_radius;
  m.iso = mp->iso;
  int r = (int)ceil((double)mp->radius / (double)ctx->p.h);  // D:A-R
  m.reach = r < 1 ? 1 : r;
  for (int a = 0; a < 3; ++a) m.cube_lo[a] = ctx->cube_lo[a], m.cube_hi[a] = ctx->cube_hi[a];
  return SPH_OK;
}

int build_grid(sph_ctx* ctx, const void* pos, const void* vel, uint32_t n, cudaStream_t s) {
  // a surface pass forked by mc_extract_async still reads the sorted arrays and the cell table this overwrites
  if (ctx->surf_pending) cudaStreamWaitEvent(s, ctx->ev_surf_done, 0);
  launch_build_grid(ctx->sc.grid, ctx->pg, (const float4*)pos, (const float4*)vel, n, ctx->scan, s, &ctx->prof, false);
  ctx->grid_pos = pos;
  ctx->grid_vel = vel;
  ctx->grid_n = n;
  ctx->grid_fresh = true;
  ctx->step_state = false;
  ctx->vel_pending = false;
  return SPH_OK;
}

}  // namespace

extern "C" {

int sph_create(sph_ctx** out, const sph_params* p, int device) {
  if (!out) return SPH_E_INVALID;
  *out = nullptr;
  if (!p) return SPH_E_INVALID;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return SPH_E_CUDA;
  sph_ctx* ctx = new (std::nothrow) sph_ctx();
  if (!ctx) return SPH_E_CUDA;
  memset(ctx, 0, sizeof(*ctx));
  for (int a = 0; a < 3; ++a) ctx->cube_hi[a] = 0xffffffffu;
  ctx->device = device;
  ctx->p = *p;
  SphConst& sc = ctx->sc;
  if (!make_grid(sc.grid, p->box_min, p->box_max, p->h) || !(p->mass > 0.0f) || !(p->rest_density > 0.0f)) {
    delete ctx;
    return SPH_E_INVALID;
  }
  sc.h = p->h;
  sc.h2 = p->h * p->h;
  sc.mass = p->mass, sc.rho0 = p->rest_density, sc.stiffness = p->stiffness, sc.viscosity = p->viscosity;
  sc.mass_c6 = (float)((double)p->mass * 315.0 / (64.0 * M_PI * pow((double)p->h, 9.0)));
  for (int a = 0; a < 3; ++a)
    sc.gravity[a] = p->gravity[a], sc.box_min[a] = p->box_min[a], sc.box_max[a] = p->box_max[a];
  sc.dt = p->dt, sc.damp = p->wall_damping;

  auto bail = [&](int code) {
    sph_destroy(ctx);
    return code;
  };
  if (cudaSetDevice(device) != cudaSuccess) return bail(SPH_E_CUDA);
  if (alloc_grid(ctx, ctx->pg, p->max_particles, sc.grid.C) != SPH_OK) return bail(SPH_E_CUDA);
  ctx->boid_cells_cap = 1u << 15;
  if (alloc_grid(ctx, ctx->bg, p->max_boids, ctx->boid_cells_cap) != SPH_OK) return bail(SPH_E_CUDA);
  const size_t nn = std::max<uint32_t>(p->max_particles, 1), nb = std::max<uint32_t>(p->max_boids, 1);
  const size_t G = p->max_mc_points_per_axis;
  if (cudaMalloc(&ctx->rhoS, nn * 4) != cudaSuccess || cudaMalloc(&ctx->rho_bS, nb * 4) != cudaSuccess ||
      cudaMalloc(&ctx->phi, std::max<size_t>(G * G * G, 1) * 4) != cudaSuccess ||
      cudaMalloc(&ctx->mc_bits, std::max<size_t>(mc_bits_words((uint32_t)G), 1) * 4) != cudaSuccess ||
      cudaMalloc(&ctx->n_tris_dev, 4) != cudaSuccess || cudaMalloc(&ctx->n_verts_dev, 4) != cudaSuccess ||
      cudaMalloc(&ctx->mc_prefix, std::max<size_t>(mc_bits_words((uint32_t)G), 1) * 4) != cudaSuccess || cudaMalloc(&ctx->mc_nwork, 8) != cudaSuccess ||
      cudaMalloc(&ctx->mc_work, std::max<size_t>(mc_num_segments((uint32_t)G), 1) * 8) != cudaSuccess || cudaMalloc(&ctx->nbr.cnt, nn * 2) != cudaSuccess ||
      cudaMalloc(&ctx->nbr.list, (size_t)nbr_rows() * (ctx->nbr.stride = (uint32_t)((nn + 63) & ~(size_t)63)) * 2) != cudaSuccess ||
      cudaMalloc(&ctx->scan.ticket, 4) != cudaSuccess ||
      cudaMalloc(&ctx->scan.ctl, 8) != cudaSuccess)
    return bail(SPH_E_CUDA);
  ctx->max_tiles = std::max(std::max(grid_scan_tiles(sc.grid.C), grid_scan_tiles(ctx->boid_cells_cap)),
                            std::max(std::max(mc_num_tiles((uint32_t)G), mc_word_tiles((uint32_t)G)), 1u));
  if (cudaMalloc(&ctx->scan.status, (size_t)ctx->max_tiles * 8) != cudaSuccess) return bail(SPH_E_CUDA);
  cudaMemset(ctx->scan.status, 0, (size_t)ctx->max_tiles * 8);
  cudaMemset(ctx->scan.ticket, 0, 4);
  {
    const size_t mt = std::max(std::max(mc_num_tiles((uint32_t)G), mc_word_tiles((uint32_t)G)), 1u);
    if (cudaMalloc(&ctx->scan_mc.status, mt * 8) != cudaSuccess || cudaMalloc(&ctx->scan_mc.ticket, 4) != cudaSuccess ||
        cudaMalloc(&ctx->scan_mc.ctl, 8) != cudaSuccess)
      return bail(SPH_E_CUDA);
    cudaMemset(ctx->scan_mc.status, 0, mt * 8);
    cudaMemset(ctx->scan_mc.ticket, 0, 4);
    {
      const uint32_t ctl0[2] = {1u, 0u};  // epoch 1: status words of zeros read as "not ready"
      cudaMemcpy(ctx->scan_mc.ctl, ctl0, 8, cudaMemcpyHostToDevice);
      cudaMemcpy(ctx->scan.ctl, ctl0, 8, cudaMemcpyHostToDevice);
    }
    ctx->scan_mc.epoch = 0;
  }
  cudaMemset(ctx->n_tris_dev, 0, 4);
  cudaMemset(ctx->mc_nwork, 0, 8);
  cudaMemset(ctx->mc_bits, 0, std::max<size_t>(mc_bits_words((uint32_t)G), 1) * 4);
  ctx->scan.epoch = 0;
  if (cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking) != cudaSuccess ||
      cudaStreamCreateWithFlags(&ctx->surf, cudaStreamNonBlocking) != cudaSuccess ||
      cudaStreamCreateWithFlags(&ctx->up, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_up_go, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_up_done, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_surf_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_surf_done, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_rho, cudaEventDisableTiming) != cudaSuccess)
    return bail(SPH_E_CUDA);
  upload_mc_tables();
  grid_init();
  if (cudaDeviceSynchronize() != cudaSuccess) return bail(SPH_E_CUDA);
  *out = ctx;
  return SPH_OK;
}

int sph_destroy(sph_ctx* ctx) {
  if (!ctx) return SPH_OK;
  cudaSetDevice(ctx->device);
  free_grid(ctx->pg);
  free_grid(ctx->bg);
  cudaFree(ctx->nbr.list), cudaFree(ctx->nbr.cnt), cudaFree(ctx->rhoS), cudaFree(ctx->rho_bS), cudaFree(ctx->phi), cudaFree(ctx->mc_bits), cudaFree(ctx->n_tris_dev), cudaFree(ctx->n_verts_dev), cudaFree(ctx->mc_prefix), cudaFree(ctx->mc_work), cudaFree(ctx->mc_nwork);
  cudaFree(ctx->scan.status), cudaFree(ctx->scan.ticket), cudaFree(ctx->scan_mc.status), cudaFree(ctx->scan_mc.ticket), cudaFree(ctx->scan.ctl), cudaFree(ctx->scan_mc.ctl);
  sph_profile_enable(ctx, 0);
  free(ctx->prof.recs);
  if (ctx->side) cudaStreamDestroy(ctx->side);
  if (ctx->surf) cudaStreamDestroy(ctx->surf);
  if (ctx->up) cudaStreamDestroy(ctx->up);
  if (ctx->ev_up_go) cudaEventDestroy(ctx->ev_up_go);
  if (ctx->ev_up_done) cudaEventDestroy(ctx->ev_up_done);
  if (ctx->ev_surf_fork) cudaEventDestroy(ctx->ev_surf_fork);
  if (ctx->ev_surf_done) cudaEventDestroy(ctx->ev_surf_done);
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
  if (ctx->ev_rho) cudaEventDestroy(ctx->ev_rho);
  cudaFree(ctx->hg_tracker), cudaFree(ctx->hg_grid), cudaFree(ctx->hg_dropped);
  cudaFree(ctx->pack_blocks), cudaFree(ctx->pack_total);
  cudaFree(ctx->cc_count), cudaFree(ctx->cc_result);
  cudaFree(ctx->h_pos), cudaFree(ctx->h_vel), cudaFree(ctx->h_bpos), cudaFree(ctx->h_bvel), cudaFree(ctx->h_tris);
  delete ctx;
  return SPH_OK;
}

const char* sph_last_error(const sph_ctx* ctx) { return ctx ? ctx->err : "null context"; }

uint32_t sph_grid_dims(const sph_ctx* ctx, uint32_t dims_out[3]) {
  if (!ctx) return 0;
  if (dims_out)
    for (int a = 0; a < 3; ++a) dims_out[a] = (uint32_t)ctx->sc.grid.dim[a];
  return ctx->sc.grid.C;
}

uint64_t sph_launch_count(const sph_ctx* ctx) { return ctx ? ctx->prof.launches : 0; }

static const char* const kKernelNames[K_NUM_KERNELS] = {
    "k_hash_count", "k_scan_cells", "k_scatter", "k_reorder", "k_hash_count[boid grid]", "k_scan_cells[boid grid]",
    "k_scatter[boid grid]", "k_reorder[boid grid]", "k_grid_small", "k_grid_small[boid grid]", "k_gather_vel",
    "k_density", "k_density_brick", "k_boid_density", "k_force_list", "k_force_masks", "k_boid_step", "k_boid_obstacles",
    "k_voxel_sdf", "k_voxel_sdf_tiles", "k_mc_signs", "k_mc_count", "k_mc_emit", "k_mc_edge_scan", "k_mc_vertices",
    "k_mc_emit_indices", "k_zero_u32", "k_cc_init", "k_cc_link", "k_cc_flatten", "k_cc_count", "k_cc_largest",
    "k_hashgrid_fill", "k_hashgrid_count", "k_range_count", "k_range_scan", "k_range_scatter"};


const char* sph_kernel_name(uint32_t kernel_id) { return kernel_id < K_NUM_KERNELS ? kKernelNames[kernel_id] : nullptr; }

int sph_profile_enable(sph_ctx* ctx, int enable) {
  if (!ctx) return SPH_E_INVALID;
  CK(cudaSetDevice(ctx->device));
  Prof& pr = ctx->prof;
  for (uint32_t i = 0; i < pr.used; ++i) cudaEventDestroy(pr.recs[i].a), cudaEventDestroy(pr.recs[i].b);
  pr.used = 0;
  for (int k = 0; k < K_NUM_KERNELS; ++k) pr.total_ms[k] = 0.0, pr.count[k] = 0;
  pr.on = enable != 0;
  return SPH_OK;
}

int sph_profile_read(sph_ctx* ctx, uint32_t kernel_id, uint64_t* launches_host, double* total_ms_host) {
  if (!ctx || kernel_id >= K_NUM_KERNELS) return SPH_E_INVALID;
  CK(cudaSetDevice(ctx->device));
  Prof& pr = ctx->prof;
  for (uint32_t i = 0; i < pr.used; ++i) {  // fold the pending event pairs into the totals
    CK(cudaEventSynchronize(pr.recs[i].b));
    float ms = 0.0f;
    CK(cudaEventElapsedTime(&ms, pr.recs[i].a, pr.recs[i].b));
    pr.total_ms[pr.recs[i].kid] += (double)ms;
    pr.count[pr.recs[i].kid] += 1;
    cudaEventDestroy(pr.recs[i].a), cudaEventDestroy(pr.recs[i].b);
  }
  pr.used = 0;
  if (launches_host) *launches_host = pr.count[kernel_id];
  if (total_ms_host) *total_ms_host = pr.total_ms[kernel_id];
  return SPH_OK;
}

void sph_mc_table(int8_t* tri_host, uint8_t* ntri_host) { mc_table_host(tri_host, ntri_host); }

int sph_build_grid(sph_ctx* ctx, const void* pos, const void* vel, uint32_t n, void* stream,
                   uint32_t* cell_of_particle, uint32_t* perm, uint32_t* cell_start) {
  if (!ctx) return SPH_E_INVALID;
  if (n > ctx->p.max_particles) return fail(ctx, SPH_E_INVALID, "n exceeds max_particles");
  if (n > 0 && (!pos || !aligned16(pos) || !aligned16(vel)))
    return fail(ctx, SPH_E_INVALID, "pos/vel must be 16-byte aligned device pointers");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  build_grid(ctx, pos, vel, n, s);
  if (cell_of_particle && n) CK(cudaMemcpyAsync(cell_of_particle, ctx->pg.key, (size_t)n * 4, cudaMemcpyDeviceToDevice, s));
  if (perm && n) CK(cudaMemcpyAsync(perm, ctx->pg.perm, (size_t)n * 4, cudaMemcpyDeviceToDevice, s));
  if (cell_start)
    CK(cudaMemcpyAsync(cell_start, ctx->pg.start, ((size_t)ctx->sc.grid.C + 1) * 4, cudaMemcpyDeviceToDevice, s));
  CK(cudaGetLastError());
  return SPH_OK;
}

int sph_invalidate_grid(sph_ctx* ctx) {
  if (!ctx) return SPH_E_INVALID;
  ctx->grid_fresh = false;
  ctx->grid_pos = ctx->grid_vel = nullptr;
  return SPH_OK;
}

int sph_particle_aabb(sph_ctx* ctx, void* stream, float* lo_hi_host) {
  if (!ctx || !lo_hi_host) return SPH_E_INVALID;
  if (!ctx->grid_fresh || ctx->grid_n == 0) return fail(ctx, SPH_E_STALE_GRID, "no current grid (or no particles)");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  uint32_t e[6];
  CK(cudaMemcpyAsync(e, ctx->pg.aabb_now, sizeof(e), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  for (int a = 0; a < 6; ++a) {  // inverse of encode_ordered (common.cuh)
    const uint32_t b = (e[a] & 0x80000000u) ? (e[a] & 0x7fffffffu) : ~e[a];
    memcpy(lo_hi_host + a, &b, 4);
  }
  return SPH_OK;
}

int sph_step(sph_ctx* ctx, void* pos, void* vel, uint32_t n, const void* bpos, const void* bvel, uint32_t n_boid,
             const boid_params* bp, void* stream, float* density, void* accel, uint32_t* ncount, uint32_t* touched) {
  if (!ctx) return SPH_E_INVALID;
  if (n > ctx->p.max_particles) return fail(ctx, SPH_E_INVALID, "n exceeds max_particles");
  if (n_boid > ctx->p.max_boids) return fail(ctx, SPH_E_INVALID, "n_boid exceeds max_boids");
  if (n > 0 && (!pos || !vel || !aligned16(pos) || !aligned16(vel) || !aligned16(accel)))
    return fail(ctx, SPH_E_INVALID, "pos/vel/accel must be 16-byte aligned device pointers");
  if (n_boid > 0 && (!bpos || !bvel || !bp || !aligned16(bpos) || !aligned16(bvel)))
    return fail(ctx, SPH_E_INVALID, "boid arrays / params missing or misaligned");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  if (!(ctx->grid_fresh && ctx->grid_pos == pos && ctx->grid_vel == vel && ctx->grid_n == n))
    build_grid(ctx, pos, vel, n, s);
  ctx->boid_state = false;
  // 0 = cost model from what the host knows (n and the cell count).  Measured on B200: the mask path
  // wins where the passes are throughput-bound -- 1 M particles at ~8 per occupied cell: frame -3 %, SPH half -8 %;
  // 4 M at ~15 per cell: frame -14 % -- and loses where they are latency-bound (its density pass launches a block per
  // brick of the whole grid): 4 K .. 262 K particles, +1 .. +10 % per frame.
  const bool brick = ctx->force_variant == 2 ||
                     (ctx->force_variant == 0 && (n >= (1u << 19) || (double)n >= 6.0 * (double)ctx->sc.grid.C));
  if (n_boid > 0) {
    int rc = set_boid_params(ctx, bp);
    if (rc != SPH_OK) return rc;
    // S7 / K14 (Boid Space hash, same machinery as the particle grid) and the boids' probe density depend only on the
    // particle grid, not on rho: they run on the context's side stream beside k_density and join before the forces
    // (with per-kernel timing on they stay on the caller's stream, so that every event pair brackets one kernel alone)
    const bool fork = !ctx->prof.on;
    cudaStream_t sb = fork ? ctx->side : s;
    if (fork) {
      CK(cudaEventRecord(ctx->ev_fork, s));
      CK(cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
    }
    launch_build_grid(ctx->bc.grid, ctx->bg, (const float4*)bpos, (const float4*)bvel, n_boid, ctx->scan, sb, &ctx->prof,
                      true);
    launch_boid_density(ctx->sc, ctx->pg, ctx->bg, n_boid, ctx->rho_bS, sb, &ctx->prof);
    if (fork) CK(cudaEventRecord(ctx->ev_join, ctx->side));
  }
  if (brick)
    launch_density_brick(ctx->sc, ctx->pg, n, ctx->rhoS, density, ncount, (uint32_t*)ctx->nbr.list, ctx->nbr.stride, s,
                         &ctx->prof);
  else
    launch_density(ctx->sc, ctx->pg, n, ctx->rhoS, density, ncount, &ctx->nbr, s, &ctx->prof);
  if (ctx->vel_pending) {  // sph_simulate_host: the velocities arrived on the upload stream while the above ran
    CK(cudaStreamWaitEvent(s, ctx->ev_up_done, 0));
    launch_gather_vel(ctx->pg, (const float4*)vel, n, s, &ctx->prof);
    ctx->vel_pending = false;
  }
  ctx->rho_event = n_boid > 0 && !ctx->prof.on;
  if (ctx->rho_event) {
    CK(cudaEventRecord(ctx->ev_rho, s));
    CK(cudaStreamWaitEvent(s, ctx->ev_join, 0));
  }
  if (brick)
    launch_force_masks(ctx->sc, n_boid > 0 ? &ctx->bc : nullptr, ctx->pg, ctx->bg, n, n_boid, ctx->rhoS, ctx->rho_bS,
                       (float4*)pos, (float4*)vel, (float4*)accel, touched, (const uint32_t*)ctx->nbr.list,
                       ctx->nbr.stride, s, &ctx->prof);
  else
    launch_force_list(ctx->sc, n_boid > 0 ? &ctx->bc : nullptr, ctx->pg, ctx->bg, n, n_boid, ctx->rhoS, ctx->rho_bS,
                      (float4*)pos, (float4*)vel, (float4*)accel, touched, ctx->nbr, s, &ctx->prof);
  ctx->grid_fresh = false;  // positions moved
  ctx->step_state = true;   // pg / rhoS still describe the step-start state (for boid_step)
  if (n_boid > 0) {
    ctx->boid_state = true;
    ctx->boid_pos = bpos;
    ctx->boid_n = n_boid;
  }
  CK(cudaGetLastError());
  return SPH_OK;
}

int boid_step(sph_ctx* ctx, const boid_params* bp, void* bpos, void* bvel, uint32_t n_boid, void* stream,
              void* dv_parts) {
  if (!ctx) return SPH_E_INVALID;
  if (n_boid == 0) return SPH_OK;
  if (!bp || !bpos || !bvel || !aligned16(bpos) || !aligned16(bvel) || !aligned16(dv_parts))
    return fail(ctx, SPH_E_INVALID, "boid arrays / params missing or misaligned");
  if (!(ctx->step_state && ctx->boid_state && ctx->boid_pos == bpos && ctx->boid_n == n_boid))
    return fail(ctx, SPH_E_STALE_GRID, "boid_step must follow sph_step called with the same boids");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  const GridDesc keep = ctx->bc.grid;
  int rc = set_boid_params(ctx, bp);  // weights may differ from sph_step's; the grid must not
  if (rc != SPH_OK) return rc;
  if (memcmp(&keep, &ctx->bc.grid, sizeof(GridDesc)) != 0)
    return fail(ctx, SPH_E_STALE_GRID, "boid ranges / space changed since sph_step");
  // S11-S13 need the step-start sorted state, rho and rho_b, not the forces: the kernel goes to the side stream, behind
  // the boid grid / probe density it already ran there and behind k_density (ev_rho), so it runs beside k_force_list;
  // the caller's stream then waits for it, so everything enqueued after this call still sees the new boid state
  // (with per-kernel timing on it stays on the caller's stream)
  if (!ctx->prof.on && ctx->rho_event) {
    // bpos / bvel are untouched since sph_step by contract, so ordering after k_density (ev_rho) is enough for them and
    // the kernel runs beside k_force_list.  dv_parts is a caller buffer that may have been written on `stream` just
    // before this call (a fill): with it, the side stream is ordered after everything enqueued on `stream` so far.
    if (dv_parts) {
      CK(cudaEventRecord(ctx->ev_fork, s));
      CK(cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
    } else {
      CK(cudaStreamWaitEvent(ctx->side, ctx->ev_rho, 0));
    }
    launch_boid_step(ctx->sc, ctx->bc, ctx->pg, ctx->bg, ctx->grid_n, n_boid, ctx->rhoS, ctx->rho_bS, (float4*)bpos,
                     (float4*)bvel, (float4*)dv_parts, ctx->side, &ctx->prof);
    if (ctx->obst_normals)  // step 7 follows the position update
      launch_boid_obstacles(ctx->oc, ctx->obst_normals, ctx->bc, (const float4*)bpos, (float4*)bvel, n_boid, ctx->side,
                            &ctx->prof);
    CK(cudaEventRecord(ctx->ev_join, ctx->side));
    CK(cudaStreamWaitEvent(s, ctx->ev_join, 0));
  } else {
    launch_boid_step(ctx->sc, ctx->bc, ctx->pg, ctx->bg, ctx->grid_n, n_boid, ctx->rhoS, ctx->rho_bS, (float4*)bpos,
                     (float4*)bvel, (float4*)dv_parts, s, &ctx->prof);
    if (ctx->obst_normals)
      launch_boid_obstacles(ctx->oc, ctx->obst_normals, ctx->bc, (const float4*)bpos, (float4*)bvel, n_boid, s,
                            &ctx->prof);
  }
  ctx->boid_state = false;  // boids moved
  CK(cudaGetLastError());
  return SPH_OK;
}

static int voxel_sdf(sph_ctx* ctx, const mc_params* mp, void* stream, float* phi, bool want_bits) {
  if (!ctx) return SPH_E_INVALID;
  if (ctx->surf_pending) cudaStreamWaitEvent((cudaStream_t)stream, ctx->ev_surf_done, 0);  // shared phi / sign field
  McConst m;
  int rc = make_mc(ctx, mp, m);
  if (rc != SPH_OK) return rc;
  if (!phi) return fail(ctx, SPH_E_INVALID, "phi is NULL");
  if (!ctx->grid_fresh) return fail(ctx, SPH_E_STALE_GRID, "mc needs sph_build_grid on the current positions");
  CK(cudaSetDevice(ctx->device));
  ctx->bits_ready = launch_voxel_sdf(ctx->sc, m, ctx->pg, phi,
                                     want_bits ? ctx->mc_bits : nullptr, ctx->sdf_variant, (cudaStream_t)stream,
                                     &ctx->prof);
  CK(cudaGetLastError());
  return SPH_OK;
}

int mc_voxel_sdf(sph_ctx* ctx, const mc_params* mp, void* stream, float* phi) {
  return voxel_sdf(ctx, mp, stream, phi, false);
}

int boid_set_obstacles(sph_ctx* ctx, const obstacle_params* op, const void* normals) {
  if (!ctx) return SPH_E_INVALID;
  if (!op || !normals) {  // clear
    ctx->obst_normals = nullptr;
    return SPH_OK;
  }
  if (!(op->cell > 0.0f) || op->dims[0] == 0 || op->dims[1] == 0 || op->dims[2] == 0 || !aligned16(normals) ||
      (uint64_t)op->dims[0] * op->dims[1] * op->dims[2] > (1ull << 31))
    return fail(ctx, SPH_E_INVALID, "bad obstacle grid");
  for (int a = 0; a < 3; ++a) ctx->oc.origin[a] = op->origin[a], ctx->oc.dims[a] = (int)op->dims[a];
  ctx->oc.cell = op->cell;
  ctx->oc.w_obs = op->w_obs;
  ctx->oc.heavy = op->heavy;
  ctx->obst_normals = (const float4*)normals;
  return SPH_OK;
}

int mc_set_cube_range(sph_ctx* ctx, int axis, uint32_t lo, uint32_t hi) {
  if (!ctx) return SPH_E_INVALID;
  if (axis < -1 || axis > 2) return fail(ctx, SPH_E_INVALID, "axis must be -1 (reset), 0, 1 or 2");
  if (axis >= 0 && lo > hi) return fail(ctx, SPH_E_INVALID, "empty ranges are lo == hi, not lo > hi");
  for (int a = 0; a < 3; ++a)
    if (axis < 0) ctx->cube_lo[a] = 0u, ctx->cube_hi[a] = 0xffffffffu;
    else if (a == axis) ctx->cube_lo[a] = lo, ctx->cube_hi[a] = hi;
  return SPH_OK;
}

int mc_set_sdf_variant(sph_ctx* ctx, int variant) {
  if (!ctx) return SPH_E_INVALID;
  if (variant < 0 || variant > 2) return fail(ctx, SPH_E_INVALID, "sdf variant must be 0, 1 or 2");
  ctx->sdf_variant = variant;
  return SPH_OK;
}

int sph_pack_range(sph_ctx* ctx, const void* pos, const void* vel, uint32_t n, int axis, float lo, float hi, void* stream,
                   void* out_pos, void* out_vel, uint32_t capacity, uint32_t* count_host) {
  if (!ctx) return SPH_E_INVALID;
  if (axis < 0 || axis > 2) return fail(ctx, SPH_E_INVALID, "axis must be 0, 1 or 2");
  if (n > ctx->p.max_particles) return fail(ctx, SPH_E_INVALID, "n exceeds max_particles");
  if (n > 0 && (!pos || !aligned16(pos) || !aligned16(vel) || !aligned16(out_pos) || !aligned16(out_vel) ||
                (capacity > 0 && !out_pos) || (vel && capacity > 0 && !out_vel)))
    return fail(ctx, SPH_E_INVALID, "pos / out arrays missing or misaligned");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  if (!ctx->pack_blocks) {
    CK(cudaMalloc(&ctx->pack_blocks, ((size_t)ctx->p.max_particles / 256 + 2) * 4));
    CK(cudaMalloc(&ctx->pack_total, 4));
  }
  launch_pack_range((const float4*)pos, (const float4*)vel, n, axis, lo, hi, ctx->pack_blocks, ctx->pack_total,
                    (float4*)out_pos, (float4*)out_vel, capacity, s, &ctx->prof);
  CK(cudaGetLastError());
  if (count_host) {
    CK(cudaMemcpyAsync(count_host, ctx->pack_total, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    if (*count_host > capacity) return fail(ctx, SPH_E_CAPACITY, "pack buffer too small");
  }
  return SPH_OK;
}

int sph_neighbor_count(sph_ctx* ctx, const void* pos, uint32_t n, void* stream, uint32_t* ncount) {
  if (!ctx) return SPH_E_INVALID;
  if (n > ctx->p.max_particles) return fail(ctx, SPH_E_INVALID, "n exceeds max_particles");
  if (n > 0 && (!pos || !aligned16(pos) || !ncount)) return fail(ctx, SPH_E_INVALID, "pos / ncount missing or misaligned");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  build_grid(ctx, pos, nullptr, n, s);
  launch_density(ctx->sc, ctx->pg, n, ctx->rhoS, nullptr, ncount, nullptr, s, &ctx->prof);
  CK(cudaGetLastError());
  return SPH_OK;
}

int sph_hashgrid_neighbor_count(sph_ctx* ctx, const void* pos, uint32_t n, uint32_t max_per_cell, void* stream,
                                uint32_t* ncount, uint32_t* dropped_host) {
  if (!ctx) return SPH_E_INVALID;
  if (n > ctx->p.max_particles) return fail(ctx, SPH_E_INVALID, "n exceeds max_particles");
  if (max_per_cell == 0 || (uint64_t)max_per_cell * ctx->sc.grid.C > (1ull << 31))
    return fail(ctx, SPH_E_INVALID, "max_per_cell out of range");
  if (n > 0 && (!pos || !aligned16(pos) || !ncount)) return fail(ctx, SPH_E_INVALID, "pos / ncount missing or misaligned");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  if (!ctx->hg_tracker) {
    CK(cudaMalloc(&ctx->hg_tracker, (size_t)ctx->sc.grid.C * 4));
    CK(cudaMalloc(&ctx->hg_dropped, 4));
  }
  if (max_per_cell > ctx->hg_cap) {
    cudaFree(ctx->hg_grid);
    ctx->hg_grid = nullptr;
    CK(cudaMalloc(&ctx->hg_grid, (size_t)ctx->sc.grid.C * max_per_cell * 4));
    ctx->hg_cap = max_per_cell;
  }
  launch_hashgrid_count(ctx->sc.grid, ctx->sc.h2, (const float4*)pos, n, max_per_cell, ctx->hg_tracker, ctx->hg_grid,
                        ctx->hg_dropped, ncount, s, &ctx->prof);
  CK(cudaGetLastError());
  if (dropped_host) {
    CK(cudaMemcpyAsync(dropped_host, ctx->hg_dropped, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
  }
  return SPH_OK;
}

int sph_set_force_variant(sph_ctx* ctx, int variant) {
  if (!ctx) return SPH_E_INVALID;
  if (variant < 0 || variant > 2) return fail(ctx, SPH_E_INVALID, "force variant must be 0, 1 or 2");
  ctx->force_variant = variant;
  return SPH_OK;
}

static int polygonise(sph_ctx* ctx, const mc_params* mp, const float* phi, bool bits_ready, void* stream, float* tris,
                      uint32_t tri_capacity, uint32_t* n_tris_host, uint32_t* n_tris_dev) {
  if (!ctx) return SPH_E_INVALID;
  if (ctx->surf_pending) cudaStreamWaitEvent((cudaStream_t)stream, ctx->ev_surf_done, 0);
  McConst m;
  int rc = make_mc(ctx, mp, m);
  if (rc != SPH_OK) return rc;
  if (!phi || (tri_capacity > 0 && !tris)) return fail(ctx, SPH_E_INVALID, "phi / tris is NULL");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  launch_mc_polygonise(m, phi, ctx->mc_bits, bits_ready, tris, tri_capacity, ctx->n_tris_dev, ctx->mc_work,
                       ctx->mc_nwork, ctx->scan_mc, s, &ctx->prof);
  if (n_tris_dev) CK(cudaMemcpyAsync(n_tris_dev, ctx->n_tris_dev, 4, cudaMemcpyDeviceToDevice, s));
  CK(cudaGetLastError());
  if (n_tris_host) {
    CK(cudaMemcpyAsync(n_tris_host, ctx->n_tris_dev, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    if (*n_tris_host > tri_capacity) return fail(ctx, SPH_E_CAPACITY, "triangle buffer too small");
  }
  return SPH_OK;
}

int mc_polygonise(sph_ctx* ctx, const mc_params* mp, const float* phi, void* stream, float* tris,
                  uint32_t tri_capacity, uint32_t* n_tris_host, uint32_t* n_tris_dev) {
  return polygonise(ctx, mp, phi, false, stream, tris, tri_capacity, n_tris_host, n_tris_dev);
}

static int polygonise_indexed(sph_ctx* ctx, const mc_params* mp, const float* phi, bool bits_ready, void* stream,
                              float* verts, float* normals, uint32_t vert_capacity, uint32_t* indices,
                              uint32_t tri_capacity, uint32_t* n_verts_host, uint32_t* n_tris_host) {
  if (!ctx) return SPH_E_INVALID;
  if (ctx->surf_pending) cudaStreamWaitEvent((cudaStream_t)stream, ctx->ev_surf_done, 0);
  McConst m;
  int rc = make_mc(ctx, mp, m);
  if (rc != SPH_OK) return rc;
  if (!phi || (vert_capacity > 0 && !verts) || (tri_capacity > 0 && !indices))
    return fail(ctx, SPH_E_INVALID, "phi / verts / indices is NULL");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  launch_mc_indexed(m, phi, ctx->mc_bits, bits_ready, ctx->mc_prefix, verts, normals, vert_capacity, indices,
                    tri_capacity, ctx->n_verts_dev, ctx->n_tris_dev, ctx->mc_work, ctx->mc_nwork, ctx->scan_mc, s,
                    &ctx->prof);
  CK(cudaGetLastError());
  if (n_verts_host || n_tris_host) {
    uint32_t nv = 0, nt = 0;
    CK(cudaMemcpyAsync(&nv, ctx->n_verts_dev, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(&nt, ctx->n_tris_dev, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    if (n_verts_host) *n_verts_host = nv;
    if (n_tris_host) *n_tris_host = nt;
    if (nv > vert_capacity || nt > tri_capacity) return fail(ctx, SPH_E_CAPACITY, "vertex / index buffer too small");
  }
  return SPH_OK;
}

int mc_polygonise_indexed(sph_ctx* ctx, const mc_params* mp, const float* phi, void* stream, float* verts,
                          float* normals, uint32_t vert_capacity, uint32_t* indices, uint32_t tri_capacity,
                          uint32_t* n_verts_host, uint32_t* n_tris_host) {
  return polygonise_indexed(ctx, mp, phi, false, stream, verts, normals, vert_capacity, indices, tri_capacity,
                            n_verts_host, n_tris_host);
}

int mc_extract_indexed(sph_ctx* ctx, const mc_params* mp, void* stream, float* phi, float* verts, float* normals,
                       uint32_t vert_capacity, uint32_t* indices, uint32_t tri_capacity, uint32_t* n_verts_host,
                       uint32_t* n_tris_host) {
  if (!ctx) return SPH_E_INVALID;
  float* field = phi ? phi : ctx->phi;
  int rc = voxel_sdf(ctx, mp, stream, field, true);
  if (rc != SPH_OK) return rc;
  return polygonise_indexed(ctx, mp, field, ctx->bits_ready, stream, verts, normals, vert_capacity, indices,
                            tri_capacity, n_verts_host, n_tris_host);
}

int mc_mesh_components(sph_ctx* ctx, const uint32_t* indices, uint32_t n_tris, uint32_t n_verts, void* stream,
                       uint32_t* label, uint32_t* n_components_host, uint32_t* largest_tris_host) {
  if (!ctx) return SPH_E_INVALID;
  if ((n_tris > 0 && !indices) || (n_verts > 0 && !label)) return fail(ctx, SPH_E_INVALID, "indices / label is NULL");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  if (!ctx->cc_result) CK(cudaMalloc(&ctx->cc_result, 3 * 4));
  if (n_verts > ctx->cc_cap || !ctx->cc_count) {
    CK(cudaStreamSynchronize(s));  // an earlier call on this stream may still use the old scratch
    cudaFree(ctx->cc_count);
    ctx->cc_count = nullptr;
    ctx->cc_cap = 0;
    CK(cudaMalloc(&ctx->cc_count, (size_t)std::max<uint32_t>(n_verts, 1u) * 4));
    ctx->cc_cap = std::max<uint32_t>(n_verts, 1u);
  }
  launch_mesh_components(indices, n_tris, n_verts, label, ctx->cc_count, ctx->cc_result, s, &ctx->prof);
  CK(cudaGetLastError());
  if (n_components_host || largest_tris_host) {
    uint32_t r[3] = {0, 0, 0};
    CK(cudaMemcpyAsync(r, ctx->cc_result, sizeof(r), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    if (r[2]) return fail(ctx, SPH_E_INVALID, "vertex index out of range");
    if (n_components_host) *n_components_host = r[0];
    if (largest_tris_host) *largest_tris_host = r[1];
  }
  return SPH_OK;
}

int mc_extract(sph_ctx* ctx, const mc_params* mp, void* stream, float* phi, float* tris, uint32_t tri_capacity,
               uint32_t* n_tris_host) {
  if (!ctx) return SPH_E_INVALID;
  float* field = phi ? phi : ctx->phi;
  int rc = voxel_sdf(ctx, mp, stream, field, true);
  if (rc != SPH_OK) return rc;
  return polygonise(ctx, mp, field, ctx->bits_ready, stream, tris, tri_capacity, n_tris_host, nullptr);
}

int mc_extract_async(sph_ctx* ctx, const mc_params* mp, void* stream, float* phi, float* tris, uint32_t tri_capacity) {
  if (!ctx) return SPH_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  if (ctx->prof.on) {  // per-kernel timing: everything stays on the caller's stream
    int rc = mc_extract(ctx, mp, stream, phi, tris, tri_capacity, nullptr);
    if (rc != SPH_OK) return rc;
    CK(cudaEventRecord(ctx->ev_surf_done, s));
  } else {
    CK(cudaEventRecord(ctx->ev_surf_fork, s));
    CK(cudaStreamWaitEvent(ctx->surf, ctx->ev_surf_fork, 0));
    int rc = mc_extract(ctx, mp, ctx->surf, phi, tris, tri_capacity, nullptr);
    if (rc != SPH_OK) return rc;
    CK(cudaEventRecord(ctx->ev_surf_done, ctx->surf));
  }
  ctx->surf_pending = true;
  ctx->surf_capacity = tri_capacity;
  return SPH_OK;
}

int mc_wait(sph_ctx* ctx, void* stream, uint32_t* n_tris_host) {
  if (!ctx) return SPH_E_INVALID;
  if (!ctx->surf_pending) return fail(ctx, SPH_E_INVALID, "mc_wait without a pending mc_extract_async");
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  CK(cudaStreamWaitEvent(s, ctx->ev_surf_done, 0));
  ctx->surf_pending = false;
  if (n_tris_host) {
    CK(cudaMemcpyAsync(n_tris_host, ctx->n_tris_dev, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    if (*n_tris_host > ctx->surf_capacity) return fail(ctx, SPH_E_CAPACITY, "triangle buffer too small");
  }
  return SPH_OK;
}

int sph_simulate_host(sph_ctx* ctx, float* pos_host, float* vel_host, uint32_t n, float* bpos_host, float* bvel_host,
                      uint32_t n_boid, const boid_params* bp, uint32_t steps, const mc_params* mp, float* tris_host,
                      uint32_t tri_capacity, uint32_t* n_tris_host) {
  if (!ctx) return SPH_E_INVALID;
  if (n > ctx->p.max_particles || n_boid > ctx->p.max_boids) return fail(ctx, SPH_E_INVALID, "n exceeds capacity");
  if (n > 0 && (!pos_host || !vel_host)) return fail(ctx, SPH_E_INVALID, "host state is NULL");
  if (n_boid > 0 && (!bpos_host || !bvel_host || !bp)) return fail(ctx, SPH_E_INVALID, "host boid state is NULL");
  CK(cudaSetDevice(ctx->device));
  if (!ctx->h_pos) {
    const size_t nn = std::max<uint32_t>(ctx->p.max_particles, 1), nb = std::max<uint32_t>(ctx->p.max_boids, 1);
    CK(cudaMalloc(&ctx->h_pos, nn * 16));
    CK(cudaMalloc(&ctx->h_vel, nn * 16));
    CK(cudaMalloc(&ctx->h_bpos, nb * 16));
    CK(cudaMalloc(&ctx->h_bvel, nb * 16));
  }
  if (mp && tri_capacity > ctx->h_tris_cap) {
    cudaFree(ctx->h_tris);
    ctx->h_tris = nullptr;
    CK(cudaMalloc(&ctx->h_tris, (size_t)tri_capacity * 36));
    ctx->h_tris_cap = tri_capacity;
  }
  cudaStream_t s = nullptr;
  // upload order: boids (small), positions, then the velocities on the upload stream: the first step's grid build and
  // density pass need positions only and run while the velocities are still crossing the bus; sph_step gathers the
  // sorted velocities (k_gather_vel) once they are there
  const bool split = steps > 0 && n > 0;
  if (n_boid) {
    CK(cudaMemcpyAsync(ctx->h_bpos, bpos_host, (size_t)n_boid * 16, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(ctx->h_bvel, bvel_host, (size_t)n_boid * 16, cudaMemcpyHostToDevice, s));
  }
  CK(cudaMemcpyAsync(ctx->h_pos, pos_host, (size_t)n * 16, cudaMemcpyHostToDevice, s));
  if (split) {
    CK(cudaEventRecord(ctx->ev_up_go, s));
    CK(cudaStreamWaitEvent(ctx->up, ctx->ev_up_go, 0));
    CK(cudaMemcpyAsync(ctx->h_vel, vel_host, (size_t)n * 16, cudaMemcpyHostToDevice, ctx->up));
    CK(cudaEventRecord(ctx->ev_up_done, ctx->up));
  } else {
    CK(cudaMemcpyAsync(ctx->h_vel, vel_host, (size_t)n * 16, cudaMemcpyHostToDevice, s));
  }
  for (uint32_t t = 0; t < steps; ++t) {
    int rc;
    if (t == 0 && split) {
      build_grid(ctx, ctx->h_pos, nullptr, n, s);
      CK(cudaGetLastError());
      ctx->grid_vel = ctx->h_vel;  // sph_step below takes this grid as its own and completes velS itself
      ctx->vel_pending = true;
      rc = SPH_OK;
    } else {
      rc = sph_build_grid(ctx, ctx->h_pos, ctx->h_vel, n, s, nullptr, nullptr, nullptr);
    }
    if (rc != SPH_OK) return rc;
    rc = sph_step(ctx, ctx->h_pos, ctx->h_vel, n, ctx->h_bpos, ctx->h_bvel, n_boid, bp, s, nullptr, nullptr, nullptr,
                  nullptr);
    if (rc != SPH_OK) return rc;
    rc = boid_step(ctx, bp, ctx->h_bpos, ctx->h_bvel, n_boid, s, nullptr);
    if (rc != SPH_OK) return rc;
  }
  // the final state goes back to the host on the side stream while the surface pass runs (pinned host buffers
  // make the two overlap; pageable ones are still correct)
  CK(cudaEventRecord(ctx->ev_fork, s));
  CK(cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
  CK(cudaMemcpyAsync(pos_host, ctx->h_pos, (size_t)n * 16, cudaMemcpyDeviceToHost, ctx->side));
  CK(cudaMemcpyAsync(vel_host, ctx->h_vel, (size_t)n * 16, cudaMemcpyDeviceToHost, ctx->side));
  if (n_boid) {
    CK(cudaMemcpyAsync(bpos_host, ctx->h_bpos, (size_t)n_boid * 16, cudaMemcpyDeviceToHost, ctx->side));
    CK(cudaMemcpyAsync(bvel_host, ctx->h_bvel, (size_t)n_boid * 16, cudaMemcpyDeviceToHost, ctx->side));
  }
  int result = SPH_OK;
  uint32_t nt = 0;
  if (mp) {
    int rc = sph_build_grid(ctx, ctx->h_pos, nullptr, n, s, nullptr, nullptr, nullptr);
    if (rc != SPH_OK) return rc;
    rc = mc_extract(ctx, mp, s, nullptr, ctx->h_tris, tri_capacity, &nt);
    if (rc != SPH_OK && rc != SPH_E_CAPACITY) return rc;
    result = rc;
    const uint32_t got = std::min(nt, tri_capacity);
    if (got && tris_host) CK(cudaMemcpyAsync(tris_host, ctx->h_tris, (size_t)got * 36, cudaMemcpyDeviceToHost, s));
  }
  if (n_tris_host) *n_tris_host = nt;
  CK(cudaStreamSynchronize(ctx->side));
  CK(cudaStreamSynchronize(s));
  return result;
}

}  // extern "C"
