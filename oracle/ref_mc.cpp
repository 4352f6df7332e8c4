// oracle/ref_mc.cpp -- CPU ORACLE (test infrastructure, see ref.h): marching-cubes table generator and
// polygoniser.  The paper names edge_table / triangle_table but does not print them;
// the table is GENERATED here from the numbering the paper fixes (D:M-TABLE), not transcribed.
// "P:n" = PAPER.md line n; "D:X" = reading X in DESIGN.md section 3.
#include "ref.h"

#include <math.h>
#include <string.h>

#include <cmath>
#include <utility>
#include <vector>

namespace {

// Numbering of ref [48] as used in the paper's worked example: corner 3's edges are
// 2, 3 and 11.  Corners 0-3 run round the z = 0 face, 4-7 sit above them; edges 0-3 bottom ring,
// 4-7 top ring, 8-11 verticals.  (D:M-NUMBERING: the axis assignment is ours.)
const int kCorner[8][3] = {{0, 0, 0}, {1, 0, 0}, {1, 1, 0}, {0, 1, 0}, {0, 0, 1}, {1, 0, 1}, {1, 1, 1}, {0, 1, 1}};
const int kEdge[12][2] = {{0, 1}, {1, 2}, {2, 3}, {3, 0}, {4, 5}, {5, 6}, {6, 7}, {7, 4}, {0, 4}, {1, 5}, {2, 6}, {3, 7}};
// The six faces as corner cycles.
const int kFace[6][4] = {{0, 1, 2, 3}, {4, 5, 6, 7}, {0, 1, 5, 4}, {3, 2, 6, 7}, {0, 3, 7, 4}, {1, 2, 6, 5}};

struct Table {
  int8_t tri[256][16];
  uint8_t ntri[256];
  uint16_t edge_mask[256];
  bool ok;
};

int edge_between(int a, int b) {
  for (int e = 0; e < 12; ++e)
    if ((kEdge[e][0] == a && kEdge[e][1] == b) || (kEdge[e][0] == b && kEdge[e][1] == a)) return e;
  return -1;
}

bool share_face(int e1, int e2) {
  for (int f = 0; f < 6; ++f) {
    int hit = 0;
    for (int s = 0; s < 4; ++s) {
      int e = edge_between(kFace[f][s], kFace[f][(s + 1) & 3]);
      hit += (e == e1) + (e == e2);
    }
    if (hit == 2) return true;
  }
  return false;
}

// D:M-TABLE.  For one case (bit n set <=> corner n is below the isolevel):
//  1. on every face, join the crossed edges pairwise; on a face with four crossed edges (the two
//     "below" corners diagonal) each segment cuts off one "below" corner;
//  2. every crossed edge now has two partners, so the segments close into loops; loops are taken in
//     ascending order of their smallest edge and start at it;
//  3. a loop is oriented so that its normal points to the ">= iso" side, and fan-triangulated from the
//     first of its vertices (in loop order) whose fan diagonals never join two edges of one cube face.
void build_case(int cs, Table& T) {
  bool below[8];
  for (int n = 0; n < 8; ++n) below[n] = (cs >> n) & 1;
  int partner[12][2];
  int np[12];
  for (int e = 0; e < 12; ++e) np[e] = 0, partner[e][0] = partner[e][1] = -1;
  auto link = [&](int a, int b) {
    partner[a][np[a]++] = b;
    partner[b][np[b]++] = a;
  };
  for (int f = 0; f < 6; ++f) {
    const int* c = kFace[f];
    int E[4];
    bool crossed[4];
    int nc = 0;
    for (int s = 0; s < 4; ++s) {
      E[s] = edge_between(c[s], c[(s + 1) & 3]);
      crossed[s] = below[c[s]] != below[c[(s + 1) & 3]];
      nc += crossed[s];
    }
    if (nc == 2) {
      int a = -1, b = -1;
      for (int s = 0; s < 4; ++s)
        if (crossed[s]) (a < 0 ? a : b) = E[s];
      link(a, b);
    } else if (nc == 4) {
      if (below[c[0]]) {  // c0 and c2 below: cut off c0 with (E3,E0), c2 with (E1,E2)
        link(E[3], E[0]);
        link(E[1], E[2]);
      } else {  // c1 and c3 below
        link(E[0], E[1]);
        link(E[2], E[3]);
      }
    }
  }
  uint16_t mask = 0;
  int out = 0;
  bool seen[12] = {false};
  for (int e0 = 0; e0 < 12; ++e0) {
    bool cr = below[kEdge[e0][0]] != below[kEdge[e0][1]];
    if (!cr || seen[e0]) continue;
    if (np[e0] != 2) {
      T.ok = false;
      return;
    }
    int loop[12], len = 0;
    int prev = -1, cur = e0;
    do {
      seen[cur] = true;
      loop[len++] = cur;
      int nxt = partner[cur][0] != prev ? partner[cur][0] : partner[cur][1];
      if (len == 1) nxt = partner[cur][0];
      prev = cur;
      cur = nxt;
    } while (cur != e0 && len < 12);
    // orientation: Newell normal of the edge-midpoint polygon against the sum of below->above edge vectors
    double mid[12][3];
    double D[3] = {0, 0, 0};
    for (int i = 0; i < len; ++i) {
      int a = kEdge[loop[i]][0], b = kEdge[loop[i]][1];
      for (int c = 0; c < 3; ++c) mid[i][c] = 0.5 * (kCorner[a][c] + kCorner[b][c]);
      int lo = below[a] ? a : b, hi = below[a] ? b : a;
      for (int c = 0; c < 3; ++c) D[c] += kCorner[hi][c] - kCorner[lo][c];
    }
    double N[3] = {0, 0, 0};
    for (int i = 0; i < len; ++i) {
      const double* u = mid[i];
      const double* v = mid[(i + 1) % len];
      N[0] += u[1] * v[2] - u[2] * v[1];
      N[1] += u[2] * v[0] - u[0] * v[2];
      N[2] += u[0] * v[1] - u[1] * v[0];
    }
    // Newell's sum of cross products about the origin is only origin-free for a closed polygon: it is.
    double dot = N[0] * D[0] + N[1] * D[1] + N[2] * D[2];
    if (dot == 0.0) {
      T.ok = false;
      return;
    }
    if (dot < 0.0)
      for (int i = 1, j = len - 1; i < j; ++i, --j) {
        int t = loop[i];
        loop[i] = loop[j];
        loop[j] = t;
      }
    for (int i = 0; i < len; ++i) mask |= (uint16_t)(1u << loop[i]);
    // fan apex: the first loop vertex from which no fan diagonal joins two edges of one cube face
    // (such a diagonal would lie in the face, where the neighbouring cube may put the same diagonal)
    for (int r = 0; r < len; ++r) {
      bool clean = true;
      for (int i = 2; i + 1 < len && clean; ++i) clean = !share_face(loop[r], loop[(r + i) % len]);
      if (clean) {
        int rot[12];
        for (int i = 0; i < len; ++i) rot[i] = loop[(r + i) % len];
        for (int i = 0; i < len; ++i) loop[i] = rot[i];
        break;
      }
    }
    for (int i = 1; i + 1 < len; ++i) {
      if (out + 3 > 15) {
        T.ok = false;
        return;
      }
      T.tri[cs][out++] = (int8_t)loop[0];
      T.tri[cs][out++] = (int8_t)loop[i];
      T.tri[cs][out++] = (int8_t)loop[i + 1];
    }
  }
  T.ntri[cs] = (uint8_t)(out / 3);
  T.edge_mask[cs] = mask;
}

const Table& table() {
  static Table T;
  static bool built = false;
  if (!built) {
    memset(T.tri, -1, sizeof(T.tri));
    memset(T.ntri, 0, sizeof(T.ntri));
    memset(T.edge_mask, 0, sizeof(T.edge_mask));
    T.ok = true;
    for (int cs = 0; cs < 256; ++cs) build_case(cs, T);
    built = true;
  }
  return T;
}

}  // namespace

extern "C" {

void ref_mc_table(int8_t* tri, uint8_t* ntri, uint16_t* edge_table) {
  const Table& T = table();
  if (tri) memcpy(tri, T.tri, sizeof(T.tri));
  if (ntri) memcpy(ntri, T.ntri, sizeof(T.ntri));
  if (edge_table) memcpy(edge_table, T.edge_mask, sizeof(T.edge_mask));
}

void ref_mc_numbering(int* corner_offsets, int* edge_corners) {
  memcpy(corner_offsets, kCorner, sizeof(kCorner));
  memcpy(edge_corners, kEdge, sizeof(kEdge));
}

int ref_mc_polygonise(const ref_mc_params* mp, const float* phi, float* tris, uint32_t tri_capacity,
                      uint32_t* n_tris, uint8_t* case_of_cube) {
  const Table& T = table();
  if (!T.ok) return -2;
  const uint32_t G = mp->n_point_per_axis;
  if (G < 2) {
    if (n_tris) *n_tris = 0;
    return 0;
  }
  const uint32_t Q = G - 1;
  const float iso = mp->iso;
  uint64_t count = 0;
  // cube-major order, then table order (D:A-APPEND)
  for (uint32_t k = 0; k < Q; ++k)
    for (uint32_t j = 0; j < Q; ++j)
      for (uint32_t i = 0; i < Q; ++i) {
        uint64_t gidx[8];
        float val[8], cp[8][3];
        int cs = 0;
        for (int n = 0; n < 8; ++n) {
          uint32_t ci = i + kCorner[n][0], cj = j + kCorner[n][1], ck = k + kCorner[n][2];
          gidx[n] = ci + (uint64_t)G * (cj + (uint64_t)G * ck);
          val[n] = phi[gidx[n]];
          cp[n][0] = mp->origin[0] + (float)ci * mp->spacing;
          cp[n][1] = mp->origin[1] + (float)cj * mp->spacing;
          cp[n][2] = mp->origin[2] + (float)ck * mp->spacing;
          if (val[n] < iso) cs |= 1 << n;  // P:536-539 Listing 10
        }
        if (case_of_cube) case_of_cube[i + (uint64_t)Q * (j + (uint64_t)Q * k)] = (uint8_t)cs;
        for (int t = 0; T.tri[cs][t] != -1; t += 3) {  // P:556 Listing 11
          if (count < tri_capacity && tris) {
            for (int v = 0; v < 3; ++v) {
              int e = T.tri[cs][t + v];
              int a = kEdge[e][0], b = kEdge[e][1];
              if (gidx[b] < gidx[a]) {  // D:A-EDGE: p1 is the corner with the smaller global index
                int s = a;
                a = b;
                b = s;
              }
              float w = (iso - val[a]) / (val[b] - val[a]);  // P:546 Eq. 51
              float* o = tris + 9 * count + 3 * v;
              for (int c = 0; c < 3; ++c) o[c] = cp[a][c] + w * (cp[b][c] - cp[a][c]);
            }
          }
          ++count;
        }
      }
  if (n_tris) *n_tris = (uint32_t)count;
  return count > tri_capacity ? 1 : 0;
}

// N3: indexed mesh with per-vertex normals.  The paper only says that normals are computed for each
// vertex and reports connectivity of the triangles; reading D:A-NORMAL / D:A-WELD:
//  * one vertex per grid edge whose end corners lie on different sides of iso, numbered in ascending edge key
//    3 * (point index of the edge's lower corner) + axis (x = 0, y = 1, z = 2); its position is Eq. 51 with
//    p1 = the lower corner (D:A-EDGE), so it is bitwise the vertex ref_mc_polygonise emits for that edge;
//  * indices[3 t + v] = vertex id of triangle t, corner v, triangles in ref_mc_polygonise's order;
//  * normal = normalise(g_a + w (g_b - g_a)), g = grad phi at a corner by central differences (one-sided on the
//    border of the grid), w the weight of Eq. 51; phi grows outwards, so the normal points out of the fluid.
static void grad_phi(const ref_mc_params* mp, const float* phi, uint32_t i, uint32_t j, uint32_t k, float g[3]) {
  const uint32_t G = mp->n_point_per_axis;
  const uint32_t c[3] = {i, j, k};
  const uint64_t stride[3] = {1, G, (uint64_t)G * G};
  const uint64_t p = i + (uint64_t)G * (j + (uint64_t)G * k);
  for (int a = 0; a < 3; ++a) {
    const bool lo = c[a] > 0, hi = c[a] + 1 < G;
    const float fm = lo ? phi[p - stride[a]] : phi[p], fp = hi ? phi[p + stride[a]] : phi[p];
    const float span = (float)((lo ? 1 : 0) + (hi ? 1 : 0)) * mp->spacing;
    g[a] = span > 0.0f ? (fp - fm) / span : 0.0f;
  }
}

int ref_mc_indexed(const ref_mc_params* mp, const float* phi, float* verts, float* normals, uint32_t vert_capacity,
                   uint32_t* indices, uint32_t tri_capacity, uint32_t* n_verts, uint32_t* n_tris) {
  const Table& T = table();
  if (!T.ok) return -2;
  const uint32_t G = mp->n_point_per_axis;
  if (n_verts) *n_verts = 0;
  if (n_tris) *n_tris = 0;
  if (G < 2) return 0;
  const float iso = mp->iso;
  const uint64_t NP = (uint64_t)G * G * G;
  const uint64_t stride[3] = {1, G, (uint64_t)G * G};
  std::vector<uint32_t> vid(3 * NP, 0xffffffffu);
  uint64_t nv = 0;
  for (uint32_t k = 0; k < G; ++k)
    for (uint32_t j = 0; j < G; ++j)
      for (uint32_t i = 0; i < G; ++i) {
        const uint64_t p = i + (uint64_t)G * (j + (uint64_t)G * k);
        const uint32_t c[3] = {i, j, k};
        for (int a = 0; a < 3; ++a) {
          if (c[a] + 1 >= G) continue;
          const float va = phi[p], vb = phi[p + stride[a]];
          if ((va < iso) == (vb < iso)) continue;
          vid[3 * p + a] = (uint32_t)nv;
          if (nv < vert_capacity) {
            const float w = (iso - va) / (vb - va);  // P:546 Eq. 51, p1 = lower corner
            uint32_t cb[3] = {i, j, k};
            cb[a] += 1;
            float ga[3], gb[3], nrm[3];
            grad_phi(mp, phi, i, j, k, ga);
            grad_phi(mp, phi, cb[0], cb[1], cb[2], gb);
            for (int x = 0; x < 3; ++x) {
              const float pa = mp->origin[x] + (float)c[x] * mp->spacing;
              const float pb = mp->origin[x] + (float)cb[x] * mp->spacing;
              if (verts) verts[3 * nv + x] = pa + w * (pb - pa);
              nrm[x] = ga[x] + w * (gb[x] - ga[x]);
            }
            if (normals) {
              const float len = std::sqrt(nrm[0] * nrm[0] + nrm[1] * nrm[1] + nrm[2] * nrm[2]);
              for (int x = 0; x < 3; ++x) normals[3 * nv + x] = len > 0.0f ? nrm[x] / len : 0.0f;
            }
          }
          ++nv;
        }
      }
  const uint32_t Q = G - 1;
  uint64_t count = 0;
  for (uint32_t k = 0; k < Q; ++k)
    for (uint32_t j = 0; j < Q; ++j)
      for (uint32_t i = 0; i < Q; ++i) {
        uint64_t gidx[8];
        int cs = 0;
        for (int n = 0; n < 8; ++n) {
          gidx[n] = (i + kCorner[n][0]) + (uint64_t)G * ((j + kCorner[n][1]) + (uint64_t)G * (k + kCorner[n][2]));
          if (phi[gidx[n]] < iso) cs |= 1 << n;
        }
        for (int t = 0; T.tri[cs][t] != -1; t += 3) {
          if (count < tri_capacity && indices)
            for (int v = 0; v < 3; ++v) {
              const int e = T.tri[cs][t + v];
              uint64_t pa = gidx[kEdge[e][0]], pb = gidx[kEdge[e][1]];
              if (pb < pa) std::swap(pa, pb);
              const uint64_t d = pb - pa;
              const int axis = d == 1 ? 0 : (d == G ? 1 : 2);
              indices[3 * count + v] = vid[3 * pa + axis];
            }
          ++count;
        }
      }
  if (n_verts) *n_verts = (uint32_t)nv;
  if (n_tris) *n_tris = (uint32_t)count;
  return (nv > vert_capacity || count > tri_capacity) ? 1 : 0;
}

// N3, connectivity ("for the triangles to connect with each other", Table 2 last column P:595-602; reading
// D:A-CONNECT): triangles are connected when they share a welded vertex; a component is a maximal connected set.
// label[v] = the smallest vertex id of v's component; a vertex no triangle uses is a component of its own with no
// triangle.  Plain flood fill over the vertex -> triangle incidence lists, components discovered in ascending
// vertex id, so the seed of each fill is the component's smallest id.
int ref_mesh_components(const uint32_t* indices, uint32_t n_tris, uint32_t n_verts, uint32_t* label,
                        uint32_t* n_components, uint32_t* largest_tris) {
  if (n_components) *n_components = 0;
  if (largest_tris) *largest_tris = 0;
  for (uint64_t e = 0; e < 3ull * n_tris; ++e)
    if (indices[e] >= n_verts) return -1;
  std::vector<uint32_t> first(n_verts + 1ull, 0), inc(3ull * n_tris);
  for (uint64_t e = 0; e < 3ull * n_tris; ++e) ++first[indices[e] + 1ull];
  for (uint32_t v = 0; v < n_verts; ++v) first[v + 1ull] += first[v];
  std::vector<uint32_t> fill(first.begin(), first.end() - 1);
  for (uint32_t t = 0; t < n_tris; ++t)
    for (int c = 0; c < 3; ++c) inc[fill[indices[3ull * t + c]]++] = t;
  std::vector<uint32_t> lab(n_verts, 0xffffffffu), stack;
  std::vector<char> seen_tri(n_tris, 0);
  uint32_t comps = 0, largest = 0;
  for (uint32_t seed = 0; seed < n_verts; ++seed) {
    if (lab[seed] != 0xffffffffu) continue;
    ++comps;
    uint32_t tris_here = 0;
    lab[seed] = seed;
    stack.assign(1, seed);
    while (!stack.empty()) {
      const uint32_t v = stack.back();
      stack.pop_back();
      for (uint32_t q = first[v]; q < first[v + 1ull]; ++q) {
        const uint32_t t = inc[q];
        if (seen_tri[t]) continue;
        seen_tri[t] = 1;
        ++tris_here;
        for (int c = 0; c < 3; ++c) {
          const uint32_t w = indices[3ull * t + c];
          if (lab[w] == 0xffffffffu) {
            lab[w] = seed;
            stack.push_back(w);
          }
        }
      }
    }
    if (tris_here > largest) largest = tris_here;
  }
  if (label)
    for (uint32_t v = 0; v < n_verts; ++v) label[v] = lab[v];
  if (n_components) *n_components = comps;
  if (largest_tris) *largest_tris = largest;
  return 0;
}


}  // extern "C"
