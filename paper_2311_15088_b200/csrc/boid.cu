// boid.cu -- S11-S13: boid separation / alignment / cohesion, fluid force on the boid, edge rule, speed
// clamp, position update.  P:277-337 (boid update loop), P:377 (sph_factor), D:C-* readings.
#include "kernels.h"

namespace sphb {

namespace {

constexpr int kThreads = 128;

// One warp per cell-sorted boid.  Lanes stride over the candidates of each x-run; the partial sums
// (binary64) are joined by a fixed shuffle tree; lane 0 finishes the update.  All rules read step-start
// state (sorted copies) and write the caller's arrays, so the update is a Jacobi step (D:C-JACOBI).
__global__ void __launch_bounds__(kThreads)
k_boid_step(SphConst c, BoidConst bc, const float4* __restrict__ posS, const float4* __restrict__ velS,
            const float* __restrict__ rhoS, const uint32_t* __restrict__ start, const float4* __restrict__ bposS,
            const float4* __restrict__ bvelS, const float* __restrict__ rho_bS, const uint32_t* __restrict__ bstart,
            const uint32_t* __restrict__ bperm, uint32_t nb, float4* __restrict__ bpos, float4* __restrict__ bvel,
            float4* __restrict__ dv_parts) {
  const uint32_t b = (blockIdx.x * kThreads + threadIdx.x) >> 5;
  const uint32_t lane = threadIdx.x & 31u;
  if (b >= nb) return;
  const float4 pb = __ldg(bposS + b);
  const float4 vb = __ldg(bvelS + b);
  const float rho_b = __ldg(rho_bS + b);

  // S11: boid-boid rules over the 27 boid cells (cell >= visible range, D:C-BGRID)
  double sep[3] = {0, 0, 0}, vs[3] = {0, 0, 0}, ps[3] = {0, 0, 0};
  uint32_t cnt = 0;
  {
    const GridDesc& g = bc.grid;
    const int cx = cell_coord(pb.x, g.lo[0], g.cell, g.dim[0]);
    const int cy = cell_coord(pb.y, g.lo[1], g.cell, g.dim[1]);
    const int cz = cell_coord(pb.z, g.lo[2], g.cell, g.dim[2]);
    for (int z = max(cz - 1, 0); z <= min(cz + 1, g.dim[2] - 1); ++z)
      for (int y = max(cy - 1, 0); y <= min(cy + 1, g.dim[1] - 1); ++y) {
        const uint32_t base = (uint32_t)g.dim[0] * ((uint32_t)y + (uint32_t)g.dim[1] * (uint32_t)z);
        const uint32_t s0 = __ldg(bstart + base + max(cx - 1, 0));
        const uint32_t s1 = __ldg(bstart + base + min(cx + 1, g.dim[0] - 1) + 1);
        for (uint32_t s = s0 + lane; s < s1; s += 32) {
          const float4 pj = __ldg(bposS + s);
          const float dx = pb.x - pj.x, dy = pb.y - pj.y, dz = pb.z - pj.z;
          const float r2 = dist2(dx, dy, dz);
          if (r2 < bc.vis2) {  // P:307, P:326 (self included: D:C-ALI)
            const float4 vj = __ldg(bvelS + s);
            vs[0] += (double)vj.x, vs[1] += (double)vj.y, vs[2] += (double)vj.z;
            ps[0] += (double)pj.x, ps[1] += (double)pj.y, ps[2] += (double)pj.z;
            ++cnt;
          }
          if (r2 < bc.prot2) {  // P:285-291 with D:C-SEP
            float sgain = 1.0f - __fdiv_rn(__fsqrt_rn(r2), bc.protect);
            sgain = fminf(fmaxf(sgain, 0.0f), 1.0f);
            sep[0] += (double)__fmul_rn(sgain, dx);
            sep[1] += (double)__fmul_rn(sgain, dy);
            sep[2] += (double)__fmul_rn(sgain, dz);
          }
        }
      }
  }

  // S12: A_b = (1/rho_b) sum_i pair_R(b,i) over the (2 reach + 1)^3 particle cells (D:C-COUPLE)
  double A[3] = {0, 0, 0};
  {
    const GridDesc& g = c.grid;
    const int cx = cell_coord(pb.x, g.lo[0], g.cell, g.dim[0]);
    const int cy = cell_coord(pb.y, g.lo[1], g.cell, g.dim[1]);
    const int cz = cell_coord(pb.z, g.lo[2], g.cell, g.dim[2]);
    const int rc = bc.reach_push;
    const float pi_f = 3.14159265358979323846f;
    const float Rp = bc.push_radius, Rp2 = Rp * Rp, piRp4 = pi_f * (Rp2 * Rp2);
    const float k15 = 15.0f * c.stiffness, mu40 = 40.0f * c.viscosity, rho0x2 = 2.0f * c.rho0;
    for (int z = max(cz - rc, 0); z <= min(cz + rc, g.dim[2] - 1); ++z)
      for (int y = max(cy - rc, 0); y <= min(cy + rc, g.dim[1] - 1); ++y) {
        const uint32_t base = (uint32_t)g.dim[0] * ((uint32_t)y + (uint32_t)g.dim[1] * (uint32_t)z);
        const uint32_t s0 = __ldg(start + base + max(cx - rc, 0));
        const uint32_t s1 = __ldg(start + base + min(cx + rc, g.dim[0] - 1) + 1);
        for (uint32_t s = s0 + lane; s < s1; s += 32) {
          const float4 pj = __ldg(posS + s);
          const float dx = pb.x - pj.x, dy = pb.y - pj.y, dz = pb.z - pj.z;
          const float r2 = dist2(dx, dy, dz);
          if (r2 > Rp2 || r2 == 0.0f) continue;
          const float4 vj = __ldg(velS + s);
          const float rho_j = __ldg(rhoS + s);
          const float q = __fdiv_rn(__fsqrt_rn(r2), Rp);
          const float q2 = 1.0f - q;
          const float coef = __fdiv_rn(c.mass * q2, piRp4 * rho_j);
          const float pterm = __fdiv_rn(k15 * ((rho_b + rho_j) - rho0x2) * q2, q);
          A[0] += (double)(coef * (pterm * dx - mu40 * (vb.x - vj.x)));
          A[1] += (double)(coef * (pterm * dy - mu40 * (vb.y - vj.y)));
          A[2] += (double)(coef * (pterm * dz - mu40 * (vb.z - vj.z)));
        }
      }
  }

#pragma unroll
  for (int a = 0; a < 3; ++a) {
    sep[a] = warp_sum_f64(sep[a]);
    vs[a] = warp_sum_f64(vs[a]);
    ps[a] = warp_sum_f64(ps[a]);
    A[a] = warp_sum_f64(A[a]);
  }
  cnt = warp_sum_u32(cnt);
  if (lane != 0) return;

  const float pbv[3] = {pb.x, pb.y, pb.z}, vbv[3] = {vb.x, vb.y, vb.z};
  float v[3], part[4][3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double d_sep = (double)bc.w_sep * sep[a];
    const double d_ali = cnt > 0 ? (double)bc.w_ali * (vs[a] / (double)cnt - (double)vbv[a]) : 0.0;
    const double d_coh = cnt > 0 ? (double)bc.w_coh * (ps[a] / (double)cnt - (double)pbv[a]) : 0.0;
    const double d_fl = (double)bc.sph_factor * (double)c.dt * (A[a] / (double)rho_b);
    double d_edge = 0.0;  // S13 edge rule (D:C-EDGE)
    if (pbv[a] < bc.space_min[a]) d_edge += (double)bc.edge_turn;
    if (pbv[a] > bc.space_max[a]) d_edge -= (double)bc.edge_turn;
    v[a] = (float)((double)vbv[a] + d_sep + d_ali + d_coh + d_fl + d_edge);
    part[0][a] = (float)d_sep, part[1][a] = (float)d_ali, part[2][a] = (float)d_coh, part[3][a] = (float)d_fl;
  }
  // speed limits (D:C-SPEED)
  const float speed = __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(v[0], v[0]), __fmul_rn(v[1], v[1])), __fmul_rn(v[2], v[2])));
  if (speed > bc.max_speed) {
    const float sc = __fdiv_rn(bc.max_speed, speed);
    v[0] *= sc, v[1] *= sc, v[2] *= sc;
  } else if (speed > 0.0f && speed < bc.min_speed) {
    const float sc = __fdiv_rn(bc.min_speed, speed);
    v[0] *= sc, v[1] *= sc, v[2] *= sc;
  }
  const uint32_t id = __ldg(bperm + b);
  bpos[id] = make_float4(pb.x + v[0] * c.dt, pb.y + v[1] * c.dt, pb.z + v[2] * c.dt, pb.w);
  bvel[id] = make_float4(v[0], v[1], v[2], vb.w);
  if (dv_parts) {
#pragma unroll
    for (int r = 0; r < 4; ++r) dv_parts[4 * id + r] = make_float4(part[r][0], part[r][1], part[r][2], 0.0f);
  }
}

// N4 (P:261 Obstacle Grid, P:336 step 7; D:C-OBST): obstacle avoidance on the boids' state after the
// position update.  v_b += w_obs * sum over the Obstacle Grid cells whose centre x_c lies within the visual range of
// g * n_c, g = heavy inside the protection range.  One warp per boid, lanes stride over the cells of the range.
__global__ void __launch_bounds__(kThreads)
k_boid_obstacles(ObstacleConst oc, const float4* __restrict__ normals, float prot2, float vis2, float visible,
                 const float4* __restrict__ bpos, float4* __restrict__ bvel, uint32_t nb) {
  const uint32_t b = (blockIdx.x * kThreads + threadIdx.x) >> 5;
  const uint32_t lane = threadIdx.x & 31u;
  if (b >= nb) return;
  const float4 p = __ldg(bpos + b);
  const float pc[3] = {p.x, p.y, p.z};
  int lo[3], n[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {  // cells whose centre can lie within the visual range (one cell of slack each side)
    const int c0 = __float2int_rd(__fdiv_rn(pc[a] - visible - oc.origin[a], oc.cell)) - 1;
    const int c1 = __float2int_rd(__fdiv_rn(pc[a] + visible - oc.origin[a], oc.cell)) + 1;
    lo[a] = max(c0, 0);
    n[a] = max(min(c1, oc.dims[a] - 1) - lo[a] + 1, 0);
  }
  const uint32_t total = (uint32_t)n[0] * (uint32_t)n[1] * (uint32_t)n[2];
  double acc[3] = {0.0, 0.0, 0.0};
  for (uint32_t t = lane; t < total; t += 32) {
    const uint32_t tz = t / ((uint32_t)n[0] * (uint32_t)n[1]), r = t - tz * (uint32_t)n[0] * (uint32_t)n[1];
    const uint32_t ty = r / (uint32_t)n[0], tx = r - ty * (uint32_t)n[0];
    const int cx = lo[0] + (int)tx, cy = lo[1] + (int)ty, cz = lo[2] + (int)tz;
    const float4 nc = __ldg(normals + (size_t)cx + (size_t)oc.dims[0] * ((size_t)cy + (size_t)oc.dims[1] * (size_t)cz));
    if (nc.x == 0.0f && nc.y == 0.0f && nc.z == 0.0f) continue;
    const float ex = __fsub_rn(p.x, __fadd_rn(oc.origin[0], __fmul_rn((float)cx + 0.5f, oc.cell)));
    const float ey = __fsub_rn(p.y, __fadd_rn(oc.origin[1], __fmul_rn((float)cy + 0.5f, oc.cell)));
    const float ez = __fsub_rn(p.z, __fadd_rn(oc.origin[2], __fmul_rn((float)cz + 0.5f, oc.cell)));
    const float d2 = dist2(ex, ey, ez);
    if (!(d2 < vis2)) continue;
    const float g = d2 < prot2 ? oc.heavy : 1.0f;
    acc[0] += (double)__fmul_rn(g, nc.x);
    acc[1] += (double)__fmul_rn(g, nc.y);
    acc[2] += (double)__fmul_rn(g, nc.z);
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) acc[a] = warp_sum_f64(acc[a]);
  if (lane != 0) return;
  const float4 v = bvel[b];
  bvel[b] = make_float4((float)((double)v.x + (double)oc.w_obs * acc[0]), (float)((double)v.y + (double)oc.w_obs * acc[1]),
                        (float)((double)v.z + (double)oc.w_obs * acc[2]), v.w);
}

}  // namespace

void launch_boid_step(const SphConst& c, const BoidConst& bc, const GridBuf& pg, const GridBuf& bg, uint32_t n,
                      uint32_t nb, const float* rhoS, const float* rho_bS, float4* bpos, float4* bvel,
                      float4* dv_parts, cudaStream_t s, Prof* prof) {
  (void)n;
  if (nb == 0) return;
  const uint32_t warps_per_block = kThreads / 32;
  prof->begin(K_BOID_STEP, s);
  k_boid_step<<<(nb + warps_per_block - 1) / warps_per_block, kThreads, 0, s>>>(
      c, bc, pg.posS, pg.velS, rhoS, pg.start, bg.posS, bg.velS, rho_bS, bg.start, bg.perm, nb, bpos, bvel, dv_parts);
  prof->end(s);
}

void launch_boid_obstacles(const ObstacleConst& oc, const float4* normals, const BoidConst& bc, const float4* bpos,
                           float4* bvel, uint32_t nb, cudaStream_t s, Prof* prof) {
  if (nb == 0) return;
  const uint32_t warps_per_block = kThreads / 32;
  prof->begin(K_BOID_OBSTACLES, s);
  k_boid_obstacles<<<(nb + warps_per_block - 1) / warps_per_block, kThreads, 0, s>>>(oc, normals, bc.prot2, bc.vis2,
                                                                                     bc.visible, bpos, bvel, nb);
  prof->end(s);
}

}  // namespace sphb
