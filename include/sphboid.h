/* sphboid.h -- C ABI of libsphboid: the per-frame particle pipeline of arXiv 2311.15088
 * ("A GPU-based Hydrodynamic Simulator with Boid Interactions") as hand-written CUDA for sm_100a.
 *
 * Citations: "P:n" = line n of the paper text; "D:X" = reading X in DESIGN.md section 3.
 *
 * Conventions
 *   - Every array argument is a DEVICE pointer unless its name ends in _host or the comment says
 *     "host".  Particle / boid state is SoA float4: pos[i] = (x,y,z,-), vel[i] = (vx,vy,vz,-),
 *     16-byte aligned; the 4th lane is carried through untouched.
 *   - The caller owns every state and output array.  The library owns only the scratch it sized in
 *     sph_create from the max_* fields (cell keys, histogram, starts, permutation, sorted copies,
 *     densities, boid grid, phi, scan state).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls only
 *     enqueue work on it; the single host synchronisation is the optional triangle-count read in
 *     mc_extract / mc_polygonise (pass n_tris_host = NULL to skip it) and the *_host entry points.
 *   - Outputs are in the CALLER'S particle order; the cell-sorted copy is internal.
 *   - Every function returns SPH_OK (0) or a negative sph_status; nothing throws or aborts.
 *     sph_last_error(ctx) gives a message for the last failure on that context.
 *   - There is no CPU fallback: without a CUDA device sph_create fails with SPH_E_CUDA.
 */
#ifndef SPHBOID_H
#define SPHBOID_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sph_ctx sph_ctx; /* opaque, library-owned */

typedef enum {
  SPH_OK = 0,
  SPH_E_INVALID = -1,    /* null / misaligned pointer, n > max, h <= 0, empty box, bad params */
  SPH_E_CAPACITY = -2,   /* triangle buffer too small: nothing past capacity written, count still returned */
  SPH_E_STALE_GRID = -3, /* call needs a grid / step state that is not current */
  SPH_E_CUDA = -4        /* CUDA runtime error, see sph_last_error */
} sph_status;

/* SPH parameters.  bound = {min,max} and cell size d (Eq. 47); h, rho0, k, mu
 * (Eq. 27-45); Euler-Cromer step and damped walls. */
typedef struct {
  float box_min[3], box_max[3];
  float h;                                   /* smoothing length == grid cell size d (D:A-CELLSIZE) */
  float rest_density, mass, stiffness, viscosity; /* rho0, m, k (bulk_modulus), mu */
  float gravity[3], dt, wall_damping;
  uint32_t max_particles, max_boids, max_mc_points_per_axis; /* scratch sizing */
} sph_params;

/* Boid parameters: separation inside protect_range, alignment + cohesion inside
 * visible_range, weights "sep", "mat", "cen"; speed limits, edge rule (D:C-EDGE); fluid->boid gain
 * sph_factor; boid->fluid radius R_p and gain (D:C-COUPLE); Boid Space. */
typedef struct {
  float protect_range, visible_range;
  float w_sep, w_ali, w_coh;
  float min_speed, max_speed, edge_turn;
  float sph_factor;
  float push_radius, w_push;
  float space_min[3], space_max[3];
} boid_params;

/* Surface pass (P:475-517 voxel density, P:531-562 marching cubes).
 * corner(i,j,k) = origin + (i,j,k)*spacing, linear index i + G*(j + G*k); (G-1)^3 cubes. */
typedef struct {
  float origin[3], spacing;
  uint32_t n_point_per_axis;                 /* G */
  float radius, particle_radius, iso;        /* R, r-bar, isolevel */
} mc_params;

/* Create a context on CUDA device `device`, allocating all scratch.  *out is NULL on failure. */
int sph_create(sph_ctx** out, const sph_params* p, int device);
int sph_destroy(sph_ctx* ctx);
const char* sph_last_error(const sph_ctx* ctx); /* host string, valid until the next call on ctx */

/* Grid dimensions dim = max(1, ceil((max-min)/h)) (D:A-DIMS); returns C = product. */
uint32_t sph_grid_dims(const sph_ctx* ctx, uint32_t dims_out[3] /* host */);

/* S1-S5: uniform-grid neighbour structure.
 *   key = hash(get_cell(p)), clamped cells (D:A-CLAMPCELL); histogram; device-wide exclusive scan;
 *   counting-sort scatter with the canonical within-cell order = ascending particle id (D:A-SORT);
 *   cell-sorted copies of pos (and of vel when given) kept in the context.
 * pos[n]; vel may be NULL (mc_extract needs positions only).
 * Optional outputs (NULL to skip): cell_of_particle[n], perm[n] (sorted slot -> particle id),
 * cell_start[C+1] (exclusive starts, cell_start[C] = n). */
int sph_build_grid(sph_ctx* ctx, const void* pos, const void* vel, uint32_t n, void* stream,
                   uint32_t* cell_of_particle, uint32_t* perm, uint32_t* cell_start);

/* Forget the current grid: the next sph_step rebuilds it, the next mc_* call returns SPH_E_STALE_GRID until
 * sph_build_grid is called.  For callers that rewrite pos in place between sph_build_grid and sph_step / mc_*. */
int sph_invalidate_grid(sph_ctx* ctx);

/* Bounding box of the particles of the last sph_build_grid (the grid build computes it on the device; the surface pass
 * uses it to skip corner tiles beyond R of every particle).  lo_hi_host = 6 host floats: min x, y, z, max x, y, z, exact
 * (binary32 min / max of the coordinates).  Synchronises `stream`.  SPH_E_STALE_GRID without a current grid or with no
 * particles.  Lets a caller lay the voxel grid over the fluid's bounding box at extraction time (BASELINE config 4). */
int sph_particle_aabb(sph_ctx* ctx, void* stream, float* lo_hi_host);

/* S6-S10: one SPH step, in place on pos / vel.
 *   density rho_i = sum_j m W_poly6 (self included), neighbour count;
 *   f_i = sum_j Listing-3 pair term; boids push the fluid (D:C-COUPLE); a_i = f_i/rho_i + g (D:A-RHO);
 *   v += a dt, x += v dt (Euler-Cromer), damped wall clamp (D:A-WALL).
 * Builds the grid itself unless the last sph_build_grid was on this (pos, vel, n) -- "this" means the same POINTERS and
 * count, and the library trusts that the arrays were not rewritten in between: a caller that modifies pos in place after
 * sph_build_grid (or whose allocator hands a new array the old address) must call sph_invalidate_grid first, otherwise
 * the step runs on the stale sort.  The mc_* calls trust the same flag.
 * bpos / bvel [n_boid] are the step-start boids (not modified); bp may be NULL iff n_boid == 0.
 * Optional outputs in caller order (NULL to skip): density[n], accel[n] (float4, total a_i),
 * ncount[n], touched[n] (number of boids inside the push radius). */
int sph_step(sph_ctx* ctx, void* pos, void* vel, uint32_t n, const void* bpos, const void* bvel,
             uint32_t n_boid, const boid_params* bp /* host */, void* stream, float* density, void* accel,
             uint32_t* ncount, uint32_t* touched);

/* S11-S13: one boid step, in place on bpos / bvel.
 *   separation / alignment / cohesion on step-start state (D:C-JACOBI), fluid force on the boid from the
 *   step-start fluid state retained by the sph_step of the same frame (D:C-COUPLE), edge rule, speed
 *   clamp, position update.
 * Must follow sph_step called with these same (unmodified) bpos / bvel; otherwise SPH_E_STALE_GRID.
 * Stream contract: bpos / bvel must not be written by anything enqueued between that sph_step and this call (the
 * library runs this step beside the force pass of sph_step, ordered after its density pass only; work enqueued on
 * `stream` AFTER this call sees the new boid state).
 * Optional dv_parts[n_boid*4] float4: the sep, ali, coh, fluid velocity increments per boid; when given, the step is
 * ordered after everything enqueued on `stream` before the call (so a fill of dv_parts on `stream` is safe). */
int boid_step(sph_ctx* ctx, const boid_params* bp /* host */, void* bpos, void* bvel, uint32_t n_boid,
              void* stream, void* dv_parts);

/* N4 (P:261 Obstacle Grid, P:336 step 7 "Obstacle Avoidance"; reading D:C-OBST).  An Obstacle Grid of
 * dims[0]*dims[1]*dims[2] cells of size `cell` from `origin`; normals = DEVICE float4[cells], cell
 * c = cx + dims0*(cy + dims1*cz) holds the averaged mesh normal of the obstacle surface in that cell (zero = none),
 * caller-owned and read by every later boid_step until cleared (op or normals NULL).  After its position update each
 * boid gets v_b += w_obs * sum over the cells whose centre lies within visible_range of the boid of g * n_c, g = heavy
 * inside protect_range ("weighed heavier"), else 1. */
typedef struct {
  float origin[3], cell;
  uint32_t dims[3];
  float w_obs, heavy;
} obstacle_params;
int boid_set_obstacles(sph_ctx* ctx, const obstacle_params* op /* host */, const void* normals);

/* N2 (the paper only names a multi-node decomposition as future work): support for
 * a slab decomposition.  Copies, in ascending index order, the particles with lo <= pos[axis] < hi (use -INFINITY /
 * INFINITY for an open side) to out_pos / out_vel (DEVICE float4[capacity]; vel / out_vel may both be NULL).
 * *count_host (host, optional; passing it synchronises) gets the number selected; SPH_E_CAPACITY if it exceeds capacity
 * (nothing past capacity is written). */
int sph_pack_range(sph_ctx* ctx, const void* pos, const void* vel, uint32_t n, int axis, float lo, float hi, void* stream,
                   void* out_pos, void* out_vel, uint32_t capacity, uint32_t* count_host);

/* S5-S6 without the density: the neighbour count of every particle (P:440-464 compute_neighbor_count; self counted,
 * r^2 < h^2) through the sorted grid (builds it on pos first).  ncount = DEVICE u32[n], caller order. */
int sph_neighbor_count(sph_ctx* ctx, const void* pos, uint32_t n, void* stream, uint32_t* ncount);

/* N4 baseline: the same counts through the paper's FIRST neighbour search (Listings 5-7):
 * an unsorted hash_grid[cell * max_per_cell + slot] of particle ids filled with atomic slot counters, then the 27-cell
 * walk reading positions through the ids.  Kept to measure the paper's claim that the sorted search is better
 * (P:589).  A particle that finds its cell full is dropped (the paper leaves that case open); *dropped_host (host,
 * optional; passing it synchronises) gets their number -- the counts equal sph_neighbor_count's iff it is 0. */
int sph_hashgrid_neighbor_count(sph_ctx* ctx, const void* pos, uint32_t n, uint32_t max_per_cell, void* stream,
                                uint32_t* ncount, uint32_t* dropped_host);

/* S6 / S8 exist twice, computing the same densities and forces (DESIGN.md sections 6 and 10): 1 = the density pass
 * stores each particle's neighbour list as 16-bit entries (the paper's section 9 design) and the force pass
 * reads it; 2 = the density pass stages a brick of cells per block in shared memory and stores the neighbour predicate
 * as one bit per candidate, the force pass walks those bits.  Measured on B200, whole frame: 2 is 3 % faster at 1 M
 * particles (config 4), 14 % at 4 M compressed ones (config 5), 1 is 1-10 % faster at 4 K - 262 K (configs 1-3, where
 * the passes are latency-bound).  0 (default) picks by a cost model: 2 when n >= 2^19 or the box holds at least 6
 * particles per grid cell on average (n >= 6 C), else 1.  Host-side setting, takes effect with the next
 * sph_step.  Any other value: SPH_E_INVALID. */
int sph_set_force_variant(sph_ctx* ctx, int variant);

/* S14: voxel signed distance phi(x) = |x - xbar| - rbar, xbar the kernel-weighted mean neighbour position
 * (Eq. 48-50, Listing 9; D:A-PHI, D:A-PHI0).  Needs a current grid (sph_build_grid on the
 * positions to mesh) else SPH_E_STALE_GRID.  phi[G^3]. */
int mc_voxel_sdf(sph_ctx* ctx, const mc_params* mp /* host */, void* stream, float* phi);

/* Restrict S15-S17 (mc_polygonise, mc_extract, their async / indexed forms) to the cubes whose index along `axis`
 * is in [lo, hi) (clamped to the grid); the other two axes keep their ranges; axis = -1 resets all three to the whole
 * grid (the default).  Triangles keep the order of D:A-APPEND among the cubes that remain, so the meshes of a partition
 * of the cubes add up to the mesh of the whole grid.  Used by the slab decomposition: a rank
 * polygonises the cubes of its own slab from its own and its ghost particles.  The vertices of the indexed form still
 * cover the whole grid.  S14 may skip what the range does not need: on fine grids (the corner-tile kernel) phi and the
 * sign field are only written for the 8 x 8 x 4 corner tiles that hold corners of the cubes in range, the rest of a phi
 * buffer keeps its old contents.  Host-side setting, takes effect with the next call. */
int mc_set_cube_range(sph_ctx* ctx, int axis, uint32_t lo, uint32_t hi);

/* S14 has two kernels that compute the same phi: 1 = one thread per corner (coarse voxel grids),
 * 2 = a warp per tile of 8x8x4 corners, 2x2x2 corners per lane, with per-lane candidate lists (fine grids).  0 (default)
 * picks by a cost model from the voxel spacing; the others force one (tests, A/B measurements). */
int mc_set_sdf_variant(sph_ctx* ctx, int variant);

/* S15-S17: marching cubes on a given phi[G^3] (Listing 10-11, Eq. 51): case per cube,
 * triangle count, device-wide exclusive scan, ordered emit (cube-major, then table order; D:A-APPEND).
 * tris = tri_capacity * 9 floats (3 vertices x xyz).  *n_tris_host (host, optional) gets the REQUIRED
 * count; if it exceeds tri_capacity the return value is SPH_E_CAPACITY and nothing past capacity is written.
 * n_tris_dev (device, optional) receives the same count without a host sync. */
int mc_polygonise(sph_ctx* ctx, const mc_params* mp /* host */, const float* phi, void* stream, float* tris,
                  uint32_t tri_capacity, uint32_t* n_tris_host, uint32_t* n_tris_dev);

/* S14-S17 in one call: phi may be NULL (library scratch is used) or a G^3 buffer that receives phi. */
int mc_extract(sph_ctx* ctx, const mc_params* mp /* host */, void* stream, float* phi, float* tris,
               uint32_t tri_capacity, uint32_t* n_tris_host);

/* The surface pass of frame t and the SPH step of frame t+1 are independent once the grid on the new positions exists
 * (the mesh is only rendered), and they stress different units (FMA pipe vs L1 / load latency).
 * mc_extract_async enqueues S14-S17 on a stream of the context, ordered after everything already enqueued on `stream`,
 * and returns without making `stream` wait; sph_step / boid_step enqueued afterwards on `stream` run beside it.  The
 * library itself orders the next sph_build_grid (which overwrites what the pass reads) and any other mc_* call after
 * the pending pass.  phi / tris must stay untouched until mc_wait, which makes `stream` wait for the pass and, if
 * n_tris_host (host) is given, synchronises and returns the required count (SPH_E_CAPACITY as for mc_extract).
 * One pass can be pending at a time; results are those of mc_extract, bit for bit. */
int mc_extract_async(sph_ctx* ctx, const mc_params* mp /* host */, void* stream, float* phi, float* tris,
                     uint32_t tri_capacity);
int mc_wait(sph_ctx* ctx, void* stream, uint32_t* n_tris_host);

/* N3 ("normals ... for each vertex", P:595-602 connectivity; readings D:A-NORMAL, D:A-WELD):
 * the same surface as mc_polygonise / mc_extract as an INDEXED mesh.  One vertex per grid edge whose end corners lie on
 * different sides of iso, in ascending edge key 3 * (point index of the lower corner) + axis; verts / normals are
 * vert_capacity * 3 floats (normals optional: NULL), position = Eq. 51 (bitwise the vertex mc_polygonise emits for that
 * edge), normal = normalise(g_a + w (g_b - g_a)) with g = grad phi by central differences (one-sided on the grid border).
 * indices = tri_capacity * 3 vertex ids, triangles in mc_polygonise's order.  *n_verts_host / *n_tris_host (host,
 * optional; passing either makes the call synchronise) get the REQUIRED counts; SPH_E_CAPACITY if one exceeds its
 * capacity, nothing past a capacity is written.  All buffers are DEVICE pointers. */
int mc_polygonise_indexed(sph_ctx* ctx, const mc_params* mp /* host */, const float* phi, void* stream, float* verts,
                          float* normals, uint32_t vert_capacity, uint32_t* indices, uint32_t tri_capacity,
                          uint32_t* n_verts_host, uint32_t* n_tris_host);
int mc_extract_indexed(sph_ctx* ctx, const mc_params* mp /* host */, void* stream, float* phi, float* verts,
                       float* normals, uint32_t vert_capacity, uint32_t* indices, uint32_t tri_capacity,
                       uint32_t* n_verts_host, uint32_t* n_tris_host);

/* N3 connectivity ("... for the triangles to connect with each other", Table 2's last column P:595-602; reading
 * D:A-CONNECT): connected components of an indexed mesh, two triangles being connected when they share a vertex.
 * indices = n_tris * 3 vertex ids below n_verts (DEVICE, e.g. mc_extract_indexed's output); label = n_verts words
 * (DEVICE, out): the smallest vertex id of the vertex's component.  *n_components_host (host, optional) = number of
 * components (a vertex no triangle uses is one, with no triangle); *largest_tris_host (host, optional) = triangles of
 * the component that has most, so 100 * largest / n_tris is the "percent of connected triangles" under D:A-CONNECT.
 * Passing either host pointer makes the call synchronise; an index >= n_verts is then reported as SPH_E_INVALID
 * (the labels are unspecified in that case).  Scratch (n_verts words) is kept in the context and grows on demand. */
int mc_mesh_components(sph_ctx* ctx, const uint32_t* indices, uint32_t n_tris, uint32_t n_verts, void* stream,
                       uint32_t* label, uint32_t* n_components_host, uint32_t* largest_tris_host);

/* End-to-end frame with HOST buffers (pinned or pageable): copies pos/vel/bpos/bvel to the device, runs
 * `steps` frames of sph_build_grid + sph_step + boid_step, optionally one surface pass on the final
 * positions (mp != NULL), copies the state (and triangles) back and synchronises.
 * tris_host may be NULL when mp is NULL. */
int sph_simulate_host(sph_ctx* ctx, float* pos_host, float* vel_host, uint32_t n, float* bpos_host,
                      float* bvel_host, uint32_t n_boid, const boid_params* bp, uint32_t steps,
                      const mc_params* mp, float* tris_host, uint32_t tri_capacity, uint32_t* n_tris_host);

/* The marching-cubes table the library uses (generated, D:M-TABLE): tri[256*16] edge ids, -1 terminated. */
void sph_mc_table(int8_t* tri_host, uint8_t* ntri_host);

/* Number of kernel launches this context has enqueued so far (bench.py's gpu_launches). */
uint64_t sph_launch_count(const sph_ctx* ctx);

/* Per-kernel device timing (measurement only, no effect on results).  While enabled, every kernel launch of
 * this context is bracketed by two CUDA events recorded on the launching stream.  sph_profile_enable resets the
 * totals.  sph_profile_read synchronises on the pending events (a host sync) and returns, for kernel
 * `kernel_id`, the number of launches and their summed duration in milliseconds (both host pointers, optional).
 * sph_kernel_name returns the kernel's name, or NULL once kernel_id is past the last kernel. */
int sph_profile_enable(sph_ctx* ctx, int enable);
int sph_profile_read(sph_ctx* ctx, uint32_t kernel_id, uint64_t* launches_host, double* total_ms_host);
const char* sph_kernel_name(uint32_t kernel_id);

/* ---- An entry point that allocates nothing -----------------------------------------------------------------------------
 * sph_build_grid_static: S1-S5 without a context -- for callers that may not call
 * cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  It calls no cudaMalloc,
 * cudaFree or allocating library routine, on its first call or any later one; its scratch (the key and the arrival rank
 * of every point) is a file-scope __device__ array of 2 x SPH_STATIC_MAX_POINTS x 4 B = 128 KB that every GPU which
 * loads the library holds until the process exits.  Runs on the CURRENT device, asynchronously on `stream`.
 *   box_min, box_max (host, 3 floats each), h: the grid of sph_create with these values (D:A-DIMS); C = its cell count.
 *   pos (device, n x float4, 16-byte aligned): the points; .w ignored.
 *   cell_of_particle[n], perm[n] (sorted slot -> id, ascending id inside a cell), cell_start[C + 1] (device, all
 *   required, caller-owned): the same values sph_build_grid returns, bit for bit.  cell_start_entries = the number of
 *   entries cell_start can hold (>= C + 1, else SPH_E_INVALID).
 * Limits: n <= SPH_STATIC_MAX_POINTS and C <= SPH_STATIC_MAX_CELLS, else SPH_E_CAPACITY and nothing is launched.
 * The scratch is shared by every call on a device and keeps the last call's contents (nothing in it needs clearing: every
 * word a call reads it has written first); calls that overlap on one GPU -- two streams, two host threads -- race on it.
 * Errors: sph_status as elsewhere; the message of the calling thread's last failure is sph_static_last_error(). */
#define SPH_STATIC_MAX_POINTS 16384u
#define SPH_STATIC_MAX_CELLS 8192u
int sph_build_grid_static(const float* box_min, const float* box_max, float h, const void* pos, uint32_t n,
                          void* stream, uint32_t* cell_of_particle, uint32_t* perm, uint32_t* cell_start,
                          uint32_t cell_start_entries);
const char* sph_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
