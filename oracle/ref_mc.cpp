// oracle/ref_mc.cpp -- CPU ORACLE (test infrastructure, see ref.h): marching-cubes table generator and
// polygoniser.  The paper names edge_table / triangle_table but does not print them;
// the table is GENERATED here from the numbering the paper fixes (D:M-TABLE), not transcribed.
// "P:n" = PAPER.md line n; "D:X" = reading X in DESIGN.md section 3.
#include "ref.h"

#include <math.h>
#include <string.h>
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

}  // extern "C"
