// oracle/ref_sim.cpp -- CPU ORACLE (test infrastructure, see ref.h): grid, SPH step, boids, voxel SDF.
// Plain and slow on purpose; OpenMP over the outer particle / boid / corner index only.
// "P:n" = PAPER.md line n; "D:X" = reading X in DESIGN.md section 3.
#include "ref.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <cmath>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// D:A-FP  r^2 = fma(dz,dz, fma(dy,dy, dx*dx)) in binary32; the one place fused ops are used.
inline float r2f(float dx, float dy, float dz) { return fmaf(dz, dz, fmaf(dy, dy, dx * dx)); }

// Uniform grid over [lo, lo + dim*cell) with clamped cells (D:A-CLAMPCELL, D:A-DIMS).
struct Grid {
  float lo[3];
  float cell;
  uint32_t dim[3];
  uint32_t C;
  std::vector<uint32_t> key, perm, start;

  void init(const float* lo_, const float* hi_, float cell_) {
    cell = cell_;
    C = 1;
    for (int a = 0; a < 3; ++a) {
      lo[a] = lo_[a];
      double e = ((double)hi_[a] - (double)lo_[a]) / (double)cell_;
      double d = ceil(e);
      if (!(d >= 1.0)) d = 1.0;
      dim[a] = (uint32_t)d;
      C *= dim[a];
    }
  }
  // P:391 Eq. 47: c = floor((p - m)/d), clamped into [0, dim-1].
  inline int coord(float p, int a) const {
    float t = (p - lo[a]) / cell;
    int c = (int)floorf(t);
    if (c < 0) c = 0;
    if (c > (int)dim[a] - 1) c = (int)dim[a] - 1;
    return c;
  }
  // hash(cx,cy,cz) = cx + dimx*(cy + dimy*cz)
  inline uint32_t hash(int cx, int cy, int cz) const {
    return (uint32_t)cx + dim[0] * ((uint32_t)cy + dim[1] * (uint32_t)cz);
  }
  inline uint32_t key_of(const float* x) const { return hash(coord(x[0], 0), coord(x[1], 1), coord(x[2], 2)); }

  // histogram, exclusive scan (D:A-OFFSET), stable counting sort (D:A-SORT).
  void build(const float* pts, uint32_t n) {
    key.assign(n, 0);
    perm.assign(n, 0);
    start.assign((size_t)C + 1, 0);
    std::vector<uint32_t> count(C, 0);
    for (uint32_t i = 0; i < n; ++i) {
      key[i] = key_of(pts + 4 * (size_t)i);
      ++count[key[i]];
    }
    uint32_t run = 0;
    for (uint32_t c = 0; c < C; ++c) {
      start[c] = run;
      run += count[c];
    }
    start[C] = run;
    std::vector<uint32_t> fill(start.begin(), start.end() - 1);
    for (uint32_t i = 0; i < n; ++i) perm[fill[key[i]]++] = i;  // ascending id within a cell
  }

  // Visit every stored point whose cell is within `reach` cells of x's cell, in ascending sorted
  // position (D:A-ORDER); cells outside the grid are skipped (D:A-BOUND).
  template <class F>
  inline void visit(const float* x, int reach, F&& f) const {
    int cx = coord(x[0], 0), cy = coord(x[1], 1), cz = coord(x[2], 2);
    for (int z = cz - reach; z <= cz + reach; ++z) {
      if (z < 0 || z >= (int)dim[2]) continue;
      for (int y = cy - reach; y <= cy + reach; ++y) {
        if (y < 0 || y >= (int)dim[1]) continue;
        int x0 = cx - reach < 0 ? 0 : cx - reach;
        int x1 = cx + reach > (int)dim[0] - 1 ? (int)dim[0] - 1 : cx + reach;
        uint32_t s0 = start[hash(x0, y, z)], s1 = start[hash(x1, y, z) + 1];
        for (uint32_t s = s0; s < s1; ++s) f(perm[s]);
      }
    }
  }
};

// Candidate enumeration: the grid walk, or (pins) every point in ascending id.
template <class F>
inline void candidates(const Grid& g, uint32_t n, const float* x, int reach, int brute, F&& f) {
  if (brute) {
    for (uint32_t j = 0; j < n; ++j) f(j);
  } else {
    g.visit(x, reach, f);
  }
}

inline int reach_cells(float radius, float cell) {
  int r = (int)ceil((double)radius / (double)cell);
  return r < 1 ? 1 : r;
}

void make_particle_grid(const ref_sph_params* p, Grid& g) { g.init(p->box_min, p->box_max, p->h); }

// m * 315/(64 pi h^9), evaluated in binary64 and rounded once (Eq. 27).
float mass_c6(const ref_sph_params* p) {
  double h = (double)p->h;
  return (float)((double)p->mass * 315.0 / (64.0 * M_PI * pow(h, 9.0)));
}

// P:172 Eq. 25 with A = rho, Eq. 27: sum_j (h^2 - r^2)^3 over r^2 < h^2 (D:A-PRED, D:A-SELF).
inline void density_at(const Grid& g, const float* pos, uint32_t n, const float* x, float h2, int brute,
                       double* sum, uint32_t* count) {
  double S = 0.0;
  uint32_t cnt = 0;
  candidates(g, n, x, 1, brute, [&](uint32_t j) {
    const float* pj = pos + 4 * (size_t)j;
    float r2 = r2f(x[0] - pj[0], x[1] - pj[1], x[2] - pj[2]);
    if (r2 < h2) {
      ++cnt;
      float t = h2 - r2;
      float t3 = t * t * t;
      S += (double)t3;
    }
  });
  *sum = S;
  *count = cnt;
}

// Listing 3, binary32, radius R.  Returns false on the two early-outs.
inline bool pair_term(float mass, float R, float k, float rho0, float mu, const float* pa, const float* va,
                      float rho_a, const float* pb, const float* vb, float rho_b, float out[3]) {
  float d[3] = {pa[0] - pb[0], pa[1] - pb[1], pa[2] - pb[2]};
  float dv[3] = {va[0] - vb[0], va[1] - vb[1], va[2] - vb[2]};
  float R2 = R * R;
  float r2 = r2f(d[0], d[1], d[2]);
  if (r2 > R2 || r2 == 0.0f) return false;
  const float pi = 3.14159265358979323846f;
  float q = sqrtf(r2) / R, q2 = 1.0f - q;
  float R4 = R2 * R2;
  float coef = mass * q2 / (pi * R4 * rho_b);
  float pterm = 15.0f * k * (rho_a + rho_b - 2.0f * rho0) * q2 / q;
  float visc = 40.0f * mu;
  for (int c = 0; c < 3; ++c) out[c] = coef * (pterm * d[c] - visc * dv[c]);
  return true;
}

void boid_grid_init(const ref_boid_params* bp, Grid& g) {
  float d = bp->visible_range;
  if (bp->push_radius > d) d = bp->push_radius;
  if (bp->protect_range > d) d = bp->protect_range;
  g.init(bp->space_min, bp->space_max, d);  // D:C-BGRID
}

void boid_density(const ref_sph_params* p, const Grid& pg, const float* pos, uint32_t n, const float* bpos,
                  uint32_t nb, int brute, float* rho_b) {
  const float h2 = p->h * p->h;
  const float mc6 = mass_c6(p);
  const float self3 = h2 * h2 * h2;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t b = 0; b < (int64_t)nb; ++b) {
    double S;
    uint32_t cnt;
    density_at(pg, pos, n, bpos + 4 * b, h2, brute, &S, &cnt);
    rho_b[b] = (float)((double)mc6 * (S + (double)self3));  // D:C-COUPLE: own parcel m W(0) + fluid
  }
}

}  // namespace

extern "C" {

int ref_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

uint32_t ref_grid_dims(const ref_sph_params* p, uint32_t dims[3]) {
  Grid g;
  make_particle_grid(p, g);
  for (int a = 0; a < 3; ++a) dims[a] = g.dim[a];
  return g.C;
}

int ref_build_grid(const ref_sph_params* p, const float* pos, uint32_t n, uint32_t* cell_of_particle,
                   uint32_t* perm, uint32_t* cell_start) {
  Grid g;
  make_particle_grid(p, g);
  g.build(pos, n);
  if (cell_of_particle) memcpy(cell_of_particle, g.key.data(), sizeof(uint32_t) * n);
  if (perm) memcpy(perm, g.perm.data(), sizeof(uint32_t) * n);
  if (cell_start) memcpy(cell_start, g.start.data(), sizeof(uint32_t) * ((size_t)g.C + 1));
  return 0;
}

int ref_density(const ref_sph_params* p, const float* pos, uint32_t n, int brute, float* density,
                uint32_t* ncount) {
  Grid g;
  make_particle_grid(p, g);
  if (!brute) g.build(pos, n);
  const float h2 = p->h * p->h;
  const float mc6 = mass_c6(p);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < (int64_t)n; ++i) {
    double S;
    uint32_t cnt;
    density_at(g, pos, n, pos + 4 * i, h2, brute, &S, &cnt);
    if (density) density[i] = (float)((double)mc6 * S);
    if (ncount) ncount[i] = cnt;
  }
  return 0;
}

int ref_boid_density(const ref_sph_params* p, const float* pos, uint32_t n, const float* bpos, uint32_t n_boid,
                     int brute, float* rho_b) {
  Grid g;
  make_particle_grid(p, g);
  if (!brute) g.build(pos, n);
  boid_density(p, g, pos, n, bpos, n_boid, brute, rho_b);
  return 0;
}

int ref_step(const ref_sph_params* p, float* pos, float* vel, uint32_t n, const float* bpos, const float* bvel,
             uint32_t n_boid, const ref_boid_params* bp, int brute, float* density, float* accel,
             uint32_t* ncount, uint32_t* touched, float* amag) {
  if (n_boid > 0 && !bp) return -1;
  Grid g;
  make_particle_grid(p, g);
  if (!brute) g.build(pos, n);
  const float h2 = p->h * p->h;
  const float mc6 = mass_c6(p);

  // S6: density (+ neighbour count)
  std::vector<float> rho(n);
  std::vector<uint32_t> cnt(n);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < (int64_t)n; ++i) {
    double S;
    uint32_t c;
    density_at(g, pos, n, pos + 4 * i, h2, brute, &S, &c);
    rho[i] = (float)((double)mc6 * S);
    cnt[i] = c;
  }

  // S7: boid grid + probe density
  Grid bg;
  std::vector<float> rho_b(n_boid);
  if (n_boid > 0) {
    boid_grid_init(bp, bg);
    if (!brute) bg.build(bpos, n_boid);
    boid_density(p, g, pos, n, bpos, n_boid, brute, rho_b.data());
  }

  // S8-S10 into fresh buffers (every thread reads step-start state only)
  std::vector<float> npos((size_t)4 * n), nvel((size_t)4 * n);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < (int64_t)n; ++i) {
    const float* xi = pos + 4 * i;
    const float* vi = vel + 4 * i;
    const float rho_i = rho[i];
    double F[3] = {0, 0, 0}, B[3] = {0, 0, 0}, mag = 0.0;
    // S8: f_i = sum_j pair(i,j)
    candidates(g, n, xi, 1, brute, [&](uint32_t j) {
      float t[3];
      if (pair_term(p->mass, p->h, p->stiffness, p->rest_density, p->viscosity, xi, vi, rho_i, pos + 4 * (size_t)j,
                    vel + 4 * (size_t)j, rho[j], t)) {
        F[0] += (double)t[0];
        F[1] += (double)t[1];
        F[2] += (double)t[2];
        mag += sqrt((double)t[0] * t[0] + (double)t[1] * t[1] + (double)t[2] * t[2]);
      }
    });
    // S9: boid -> fluid push, D:C-COUPLE; touched counts the pairs Listing 3 gets past its early-out
    uint32_t tch = 0;
    if (n_boid > 0) {
      candidates(bg, n_boid, xi, 1, brute, [&](uint32_t b) {
        float t[3];
        if (pair_term(p->mass, bp->push_radius, p->stiffness, p->rest_density, p->viscosity, xi, vi, rho_i,
                      bpos + 4 * (size_t)b, bvel + 4 * (size_t)b, rho_b[b], t)) {
          ++tch;
          B[0] += (double)t[0];
          B[1] += (double)t[1];
          B[2] += (double)t[2];
          mag += fabs((double)bp->w_push) * sqrt((double)t[0] * t[0] + (double)t[1] * t[1] + (double)t[2] * t[2]);
        }
      });
    }
    const double wp = n_boid > 0 ? (double)bp->w_push : 0.0;
    float a[3];
    for (int c = 0; c < 3; ++c)  // D:A-RHO: a_i = f_i / rho_i + g  (Eq. 1)
      a[c] = (float)((F[c] + wp * B[c]) / (double)rho_i + (double)p->gravity[c]);
    if (accel) {
      accel[4 * i + 0] = a[0];
      accel[4 * i + 1] = a[1];
      accel[4 * i + 2] = a[2];
      accel[4 * i + 3] = 0.0f;
    }
    if (amag) {
      double gm = sqrt((double)p->gravity[0] * p->gravity[0] + (double)p->gravity[1] * p->gravity[1] +
                       (double)p->gravity[2] * p->gravity[2]);
      amag[i] = (float)(mag / (double)rho_i + gm);
    }
    if (touched) touched[i] = tch;
    // S10: Euler-Cromer (D:A-INTEG), then per-axis wall (D:A-WALL)
    for (int c = 0; c < 3; ++c) {
      float v = vi[c] + p->dt * a[c];
      float x = xi[c] + p->dt * v;
      if (x < p->box_min[c]) {
        x = p->box_min[c];
        v = -p->wall_damping * v;
      }
      if (x > p->box_max[c]) {
        x = p->box_max[c];
        v = -p->wall_damping * v;
      }
      npos[4 * i + c] = x;
      nvel[4 * i + c] = v;
    }
    npos[4 * i + 3] = xi[3];
    nvel[4 * i + 3] = vi[3];
  }
  if (density) memcpy(density, rho.data(), sizeof(float) * n);
  if (ncount) memcpy(ncount, cnt.data(), sizeof(uint32_t) * n);
  memcpy(pos, npos.data(), sizeof(float) * 4 * (size_t)n);
  memcpy(vel, nvel.data(), sizeof(float) * 4 * (size_t)n);
  return 0;
}

int ref_boid_step(const ref_sph_params* p, const ref_boid_params* bp, const float* pos, const float* vel,
                  const float* density, uint32_t n, float* bpos, float* bvel, uint32_t n_boid, int brute,
                  float* dv_parts) {
  if (n_boid == 0) return 0;
  Grid g, bg;
  make_particle_grid(p, g);
  boid_grid_init(bp, bg);
  if (!brute) {
    g.build(pos, n);
    bg.build(bpos, n_boid);
  }
  std::vector<float> rho_b(n_boid);
  boid_density(p, g, pos, n, bpos, n_boid, brute, rho_b.data());
  const float vis2 = bp->visible_range * bp->visible_range;
  const float prot2 = bp->protect_range * bp->protect_range;
  const int reach_p = reach_cells(bp->push_radius, p->h);
  std::vector<float> npos((size_t)4 * n_boid), nvel((size_t)4 * n_boid);
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t b = 0; b < (int64_t)n_boid; ++b) {
    const float* xb = bpos + 4 * b;
    const float* vb = bvel + 4 * b;
    // S11: separation / alignment / cohesion on step-start state (D:C-SEP, D:C-ALI, D:C-COH, D:C-JACOBI)
    double sep[3] = {0, 0, 0}, vs[3] = {0, 0, 0}, ps[3] = {0, 0, 0};
    uint32_t cnt = 0;
    candidates(bg, n_boid, xb, 1, brute, [&](uint32_t j) {
      const float* xj = bpos + 4 * (size_t)j;
      const float* vj = bvel + 4 * (size_t)j;
      float d[3] = {xb[0] - xj[0], xb[1] - xj[1], xb[2] - xj[2]};
      float r2 = r2f(d[0], d[1], d[2]);
      if (r2 < vis2) {
        for (int c = 0; c < 3; ++c) {
          vs[c] += (double)vj[c];
          ps[c] += (double)xj[c];
        }
        ++cnt;
      }
      if (r2 < prot2) {
        float s = 1.0f - sqrtf(r2) / bp->protect_range;
        if (s < 0.0f) s = 0.0f;
        if (s > 1.0f) s = 1.0f;
        for (int c = 0; c < 3; ++c) sep[c] += (double)(s * d[c]);
      }
    });
    // S12: fluid -> boid, A_b = (1/rho_b) sum_i pair_R(b,i)  (D:C-COUPLE)
    double A[3] = {0, 0, 0};
    candidates(g, n, xb, reach_p, brute, [&](uint32_t i) {
      float t[3];
      if (pair_term(p->mass, bp->push_radius, p->stiffness, p->rest_density, p->viscosity, xb, vb, rho_b[b],
                    pos + 4 * (size_t)i, vel + 4 * (size_t)i, density[i], t)) {
        A[0] += (double)t[0];
        A[1] += (double)t[1];
        A[2] += (double)t[2];
      }
    });
    float v[3], x[3];
    for (int c = 0; c < 3; ++c) {
      double d_sep = (double)bp->w_sep * sep[c];
      double d_ali = cnt > 0 ? (double)bp->w_ali * (vs[c] / (double)cnt - (double)vb[c]) : 0.0;
      double d_coh = cnt > 0 ? (double)bp->w_coh * (ps[c] / (double)cnt - (double)xb[c]) : 0.0;
      double d_fl = (double)bp->sph_factor * (double)p->dt * (A[c] / (double)rho_b[b]);
      double d_edge = 0.0;  // S13: D:C-EDGE
      if (xb[c] < bp->space_min[c]) d_edge += (double)bp->edge_turn;
      if (xb[c] > bp->space_max[c]) d_edge -= (double)bp->edge_turn;
      v[c] = (float)((double)vb[c] + d_sep + d_ali + d_coh + d_fl + d_edge);
      if (dv_parts) {
        dv_parts[16 * b + 0 + c] = (float)d_sep;
        dv_parts[16 * b + 4 + c] = (float)d_ali;
        dv_parts[16 * b + 8 + c] = (float)d_coh;
        dv_parts[16 * b + 12 + c] = (float)d_fl;
      }
    }
    // D:C-SPEED
    float speed = sqrtf(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    if (speed > bp->max_speed) {
      float s = bp->max_speed / speed;
      for (int c = 0; c < 3; ++c) v[c] *= s;
    } else if (speed > 0.0f && speed < bp->min_speed) {
      float s = bp->min_speed / speed;
      for (int c = 0; c < 3; ++c) v[c] *= s;
    }
    for (int c = 0; c < 3; ++c) x[c] = xb[c] + v[c] * p->dt;
    for (int c = 0; c < 3; ++c) {
      npos[4 * b + c] = x[c];
      nvel[4 * b + c] = v[c];
    }
    npos[4 * b + 3] = xb[3];
    nvel[4 * b + 3] = vb[3];
  }
  memcpy(bpos, npos.data(), sizeof(float) * 4 * (size_t)n_boid);
  memcpy(bvel, nvel.data(), sizeof(float) * 4 * (size_t)n_boid);
  return 0;
}

int ref_voxel_sdf(const ref_sph_params* p, const ref_mc_params* mp, const float* pos, uint32_t n, int brute,
                  float* phi) {
  Grid g;
  make_particle_grid(p, g);
  if (!brute) g.build(pos, n);
  const uint32_t G = mp->n_point_per_axis;
  const float R = mp->radius, R2 = R * R;
  const int reach = reach_cells(R, p->h);  // D:A-R
  const int64_t total = (int64_t)G * G * G;
#pragma omp parallel for schedule(dynamic, 1024)
  for (int64_t idx = 0; idx < total; ++idx) {
    uint32_t i = (uint32_t)(idx % G), j = (uint32_t)((idx / G) % G), k = (uint32_t)(idx / ((int64_t)G * G));
    // corner = (xmin,ymin,zmin) + id * grid_size
    float x[3] = {mp->origin[0] + (float)i * mp->spacing, mp->origin[1] + (float)j * mp->spacing,
                  mp->origin[2] + (float)k * mp->spacing};
    double S0 = 0.0, S1[3] = {0, 0, 0};
    candidates(g, n, x, reach, brute, [&](uint32_t q) {
      const float* pj = pos + 4 * (size_t)q;
      float d[3] = {pj[0] - x[0], pj[1] - x[1], pj[2] - x[2]};
      float r2 = r2f(d[0], d[1], d[2]);
      if (r2 < R2) {
        float u = 1.0f - r2 / R2;  // k(s) = (1 - s^2)^3, s = |x - x_j|/R
        float kj = u * u * u;
        S0 += (double)kj;
        for (int c = 0; c < 3; ++c) S1[c] += (double)(kj * d[c]);
      }
    });
    // D:A-PHI: phi = |sum k_j (x_j - x)| / sum k_j - rbar; D:A-PHI0 when no neighbour
    if (S0 > 0.0)
      phi[idx] = (float)(sqrt(S1[0] * S1[0] + S1[1] * S1[1] + S1[2] * S1[2]) / S0 - (double)mp->particle_radius);
    else
      phi[idx] = R - mp->particle_radius;
  }
  return 0;
}

double ref_w_poly6(double r, double h) {
  if (r < 0 || r > h) return 0.0;
  double t = h * h - r * r;
  return 315.0 / (64.0 * M_PI * pow(h, 9.0)) * t * t * t;
}

void ref_pair_term(float mass, float radius, float stiffness, float rest_density, float viscosity,
                   const float* pos_a, const float* vel_a, float rho_a, const float* pos_b, const float* vel_b,
                   float rho_b, float* out) {
  float t[3] = {0, 0, 0};
  if (!pair_term(mass, radius, stiffness, rest_density, viscosity, pos_a, vel_a, rho_a, pos_b, vel_b, rho_b, t))
    t[0] = t[1] = t[2] = 0.0f;
  out[0] = t[0];
  out[1] = t[1];
  out[2] = t[2];
}

// N4: obstacle avoidance (P:261, P:336 step 7; D:C-OBST).  Sums in binary64, rounded once, like the other boid rules.
int ref_boid_obstacles(const ref_obstacle_params* op, const float* normals, float protect_range, float visible_range,
                       const float* bpos, float* bvel, uint32_t n_boid, int brute) {
  if (!op || !normals || !(op->cell > 0.0f)) return -1;
  const int dx = (int)op->dims[0], dy = (int)op->dims[1], dz = (int)op->dims[2];
  const float vis2 = visible_range * visible_range, prot2 = protect_range * protect_range;
#pragma omp parallel for schedule(static)
  for (int64_t b = 0; b < (int64_t)n_boid; ++b) {
    const float* p = bpos + 4 * b;
    int lo[3] = {0, 0, 0}, hi[3] = {dx - 1, dy - 1, dz - 1};
    if (!brute) {
      const int dims[3] = {dx, dy, dz};
      for (int a = 0; a < 3; ++a) {  // cells whose centre can lie within the visible range
        const int c0 = (int)std::floor((p[a] - visible_range - op->origin[a]) / op->cell) - 1;
        const int c1 = (int)std::floor((p[a] + visible_range - op->origin[a]) / op->cell) + 1;
        lo[a] = std::max(c0, 0);
        hi[a] = std::min(c1, dims[a] - 1);
      }
    }
    double acc[3] = {0.0, 0.0, 0.0};
    for (int cz = lo[2]; cz <= hi[2]; ++cz)
      for (int cy = lo[1]; cy <= hi[1]; ++cy)
        for (int cx = lo[0]; cx <= hi[0]; ++cx) {
          const float* nc = normals + 4 * ((size_t)cx + (size_t)dx * ((size_t)cy + (size_t)dy * (size_t)cz));
          if (nc[0] == 0.0f && nc[1] == 0.0f && nc[2] == 0.0f) continue;
          const float ex = p[0] - (op->origin[0] + ((float)cx + 0.5f) * op->cell);
          const float ey = p[1] - (op->origin[1] + ((float)cy + 0.5f) * op->cell);
          const float ez = p[2] - (op->origin[2] + ((float)cz + 0.5f) * op->cell);
          const float d2 = std::fmaf(ez, ez, std::fmaf(ey, ey, ex * ex));
          if (!(d2 < vis2)) continue;
          const float g = d2 < prot2 ? op->heavy : 1.0f;
          acc[0] += (double)(g * nc[0]);
          acc[1] += (double)(g * nc[1]);
          acc[2] += (double)(g * nc[2]);
        }
    for (int a = 0; a < 3; ++a) bvel[4 * b + a] = (float)((double)bvel[4 * b + a] + (double)op->w_obs * acc[a]);
  }
  return 0;
}

}  // extern "C"
