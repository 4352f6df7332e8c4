/* oracle/ref.h -- CPU ORACLE for the per-frame particle pipeline of arXiv 2311.15088.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may build, link or call anything under oracle/.
 * It shares no code, header, table or constant generator with the CUDA path
 * (paper_2311_15088_b200/csrc, include/sphboid.h); neither side includes the other.
 *
 * Citations: "P:n" = line n of PAPER.md (arXiv 2311.15088 text); "D:X" = reading X listed in
 * DESIGN.md section 3 (the readings of what the paper leaves silent, ambiguous or garbled).
 *
 * Precision (D:A-FP).  The paper computes in HLSL `float`.  Here every DECISION that
 * produces an integer (cell index, neighbour predicate, MC case bit) and every PER-PAIR TERM is
 * evaluated in IEEE binary32 with the operation order written in the code (compiled with
 * -ffp-contract=off; the only fused operations are the explicit fmaf calls in r2()).  Every SUM
 * over neighbours is accumulated in binary64 and rounded to binary32 once: the paper's threads sum
 * in an unspecified order, and the binary64 sum of binary32 terms is the order-free value every
 * legal order approximates.
 *
 * Pin status (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   grid / counting sort / neighbour sets ... pinned (brute force O(N^2), permutation invariants)
 *   W_poly6 normalisation, lattice density .. pinned (numerical integral = 1, closed form 1.0097752 rho0)
 *   pair force ............................... pinned (hand-evaluated two-particle case, antisymmetry,
 *                                                      zero net momentum, lattice interior f = 0)
 *   integrate + wall ......................... pinned (free-fall closed form, wall reflection)
 *   boid rules ............................... pinned (hand-evaluated two-boid case, lone boid, speed cap)
 *   SPH<->boid coupling ...................... invariants only (antisymmetry, locality, brute force);
 *                                              the coupling READING is ours (D:C-COUPLE): PARITY UNPINNED
 *   voxel SDF ................................ pinned (one particle: phi = |x-x1| - rbar; symmetric pair; the weight
 *                                              k(s) = (1-s^2)^3 of P:487: unequal pair closed form, Listing 9 written
 *                                              out as its two loops in numpy, k -> 0 like (2 eps)^3 at the edge of R)
 *   MC table ................................. pinned (P:542 worked example edge_table[8]=0x80c, crack-free
 *                                                      faces, edge cover, orientation)
 *   indexed mesh (N3) ........................ welding pinned (expands to the triangle soup bitwise, Euler characteristic
 *                                              on the index buffer); the NORMAL formula is ours (D:A-NORMAL): invariants
 *                                              only (exact on a plane, radial on a sphere): PARITY UNPINNED
 *   mesh connectivity (N3) ................... pinned (scipy.sparse.csgraph.connected_components on random triangle sets,
 *                                              k separated spheres -> k equal components, hand-made chains)
 *   obstacle avoidance (N4) .................. invariants only (hand-evaluated single cell, zero grid, range walk = all
 *                                              cells, sphere pushes outwards); the rule is ours (D:C-OBST): PARITY UNPINNED
 *   MC end to end ............................ pinned (analytic sphere: closed, Euler char 2, area, volume)
 */
#ifndef ORACLE_REF_H
#define ORACLE_REF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* P:389-395 (bound, d), P:182-251 (h, rho0, k, mu), P:43, P:345 (walls, Euler-Cromer) */
typedef struct {
  float box_min[3], box_max[3];
  float h;                 /* smoothing length == cell size d (D:A-CELLSIZE) */
  float rest_density, mass, stiffness, viscosity;
  float gravity[3], dt, wall_damping;
} ref_sph_params;

/* P:256-337 (boid rules), P:377 (sph_factor), D:C-COUPLE (push radius / gain) */
typedef struct {
  float protect_range, visible_range;
  float w_sep, w_ali, w_coh;
  float min_speed, max_speed, edge_turn;
  float sph_factor;
  float push_radius, w_push;
  float space_min[3], space_max[3];
} ref_boid_params;

/* P:475-517 (voxel density), P:531-547 (marching cubes) */
typedef struct {
  float origin[3], spacing;
  uint32_t n_point_per_axis;     /* G points per axis, (G-1)^3 cubes (D:A-MCGRID) */
  float radius, particle_radius, iso;
} ref_mc_params;

/* All pointers are HOST pointers.  pos/vel/bpos/bvel are float[4*n] (x,y,z,unused). */

/* D:A-DIMS: dims[a] = max(1, ceil((hi-lo)/h)) ; returns C = product. */
uint32_t ref_grid_dims(const ref_sph_params* p, uint32_t dims[3]);

/* S1-S5: cell key per particle, stable counting sort, exclusive starts.
 * cell_of_particle[n], perm[n] (sorted position -> original id), cell_start[C+1]. */
int ref_build_grid(const ref_sph_params* p, const float* pos, uint32_t n,
                   uint32_t* cell_of_particle, uint32_t* perm, uint32_t* cell_start);

/* S6: density and neighbour count.  brute != 0 -> all-pairs O(N^2). */
int ref_density(const ref_sph_params* p, const float* pos, uint32_t n, int brute,
                float* density, uint32_t* ncount);

/* S7 (D:C-COUPLE): boid probe density rho_b = m W(0) + sum_fluid m W_poly6. */
int ref_boid_density(const ref_sph_params* p, const float* pos, uint32_t n,
                     const float* bpos, uint32_t n_boid, int brute, float* rho_b);

/* S6-S10: one SPH step in place (pos, vel updated).  bp may be NULL iff n_boid == 0.
 * Optional outputs (may be NULL): density[n], accel[4n] (total a_i incl. gravity), ncount[n],
 * touched[n], amag[n] (sum of |term|/rho_i + |g|: the magnitude the float error scales with). */
int ref_step(const ref_sph_params* p, float* pos, float* vel, uint32_t n,
             const float* bpos, const float* bvel, uint32_t n_boid, const ref_boid_params* bp,
             int brute,
             float* density, float* accel, uint32_t* ncount, uint32_t* touched, float* amag);

/* S11-S13: one boid step in place, from the STEP-START fluid state (pos, vel, density of the same
 * frame's ref_step input; D:C-JACOBI).  Optional dv_parts[nb*16]: sep, ali, coh, fluid (4 floats each). */
int ref_boid_step(const ref_sph_params* p, const ref_boid_params* bp,
                  const float* pos, const float* vel, const float* density, uint32_t n,
                  float* bpos, float* bvel, uint32_t n_boid, int brute, float* dv_parts);

/* N4 (P:261 Obstacle Grid, P:336 step 7; reading D:C-OBST): obstacle avoidance, applied to the boids'
 * state AFTER the position update (step 7 follows step 6).  The Obstacle Grid is dims[0]*dims[1]*dims[2] cells of size
 * `cell` from `origin`; normals[4*c] holds the averaged mesh normal of cell c = cx + dims0*(cy + dims1*cz) (zero =
 * no obstacle there), x_c its centre.  bvel_b += w_obs * sum over cells with |bpos_b - x_c| < visible of g * n_c,
 * g = heavy if |bpos_b - x_c| < protect else 1.  brute != 0 visits every cell instead of the cells in range. */
typedef struct {
  float origin[3], cell;
  uint32_t dims[3];
  float w_obs, heavy;
} ref_obstacle_params;
int ref_boid_obstacles(const ref_obstacle_params* op, const float* normals, float protect_range, float visible_range,
                       const float* bpos, float* bvel, uint32_t n_boid, int brute);

/* S14: phi[G^3], corner index i + G*(j + G*k). */
int ref_voxel_sdf(const ref_sph_params* p, const ref_mc_params* mp, const float* pos, uint32_t n,
                  int brute, float* phi);

/* S15-S17: polygonise a given phi.  tris = capacity*9 floats (may be NULL if capacity 0);
 * n_tris gets the REQUIRED count; nothing past capacity is written.  Optional case_of_cube[(G-1)^3]. */
int ref_mc_polygonise(const ref_mc_params* mp, const float* phi, float* tris, uint32_t tri_capacity,
                      uint32_t* n_tris, uint8_t* case_of_cube);

/* N3 (D:A-NORMAL, D:A-WELD): the same mesh as ref_mc_polygonise, indexed: one vertex per crossing grid edge in
 * ascending edge key 3*point + axis, verts / normals = vert_capacity*3 floats (normals may be NULL),
 * indices = tri_capacity*3 vertex ids in ref_mc_polygonise's triangle order.  n_verts / n_tris get the REQUIRED counts;
 * nothing past a capacity is written.  Returns 1 if a capacity was too small. */
int ref_mc_indexed(const ref_mc_params* mp, const float* phi, float* verts, float* normals, uint32_t vert_capacity,
                   uint32_t* indices, uint32_t tri_capacity, uint32_t* n_verts, uint32_t* n_tris);

/* N3 connectivity (Table 2; D:A-CONNECT): connected components of an indexed mesh, two triangles
 * being connected when they share a vertex.  label[n_verts] (may be NULL) = smallest vertex id of the vertex's
 * component; n_components counts every vertex's component (an unused vertex is one, with no triangle);
 * largest_tris = triangles of the component that has most.  Returns -1 if an index is out of range. */
int ref_mesh_components(const uint32_t* indices, uint32_t n_tris, uint32_t n_verts, uint32_t* label,
                        uint32_t* n_components, uint32_t* largest_tris);

/* The generated table (D:M-TABLE): tri[256][16] edge ids terminated by -1, ntri[256], edge_table[256]. */
void ref_mc_table(int8_t* tri, uint8_t* ntri, uint16_t* edge_table);
/* Bourke numbering used by the table: corner offsets [8][3], edge endpoints [12][2]. */
void ref_mc_numbering(int* corner_offsets, int* edge_corners);

/* W_poly6(r,h) in binary64, for the normalisation pin. */
double ref_w_poly6(double r, double h);
/* Listing 3 pair term in binary32 arithmetic; out[3]. */
void ref_pair_term(float mass, float radius, float stiffness, float rest_density, float viscosity,
                   const float* pos_a, const float* vel_a, float rho_a,
                   const float* pos_b, const float* vel_b, float rho_b, float* out);

int ref_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
