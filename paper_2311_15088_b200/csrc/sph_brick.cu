// sph_brick.cu -- S6 with the neighbourhood of a BRICK of cells staged once per block in shared memory, and S8-S10 from
// the neighbour masks it stores.  P:440-471 (Listing 8 + section 9: neighbour search, stored neighbours), P:172 / P:182
// (density), P:351-375 (Listing 3).  Selected by sph_set_force_variant(ctx, 2); DESIGN.md section 10 has the A/B.
//
//   k_density_brick : a block owns a brick of BX x BY x BZ cells and copies the (BX+2)(BY+2)(BZ+2) cells around it --
//                     (BY+2)(BZ+2) contiguous x-runs of the cell-sorted positions -- into shared memory once.  A thread
//                     owns TWO targets of one cell (they share their nine runs) and tests two candidates per step on
//                     packed binary32.  The neighbour predicate bits of every chunk of 32 candidates are stored as they
//                     are (one mask word per target and chunk): the stored neighbour list of P:469-471 at 1 bit per
//                     candidate instead of an index per neighbour.
//   k_force_masks   : one thread per particle walks its mask words as one bit stream and gathers the neighbours.
// A brick whose neighbourhood does not fit the staging capacity is split in two along an axis, down to single cells;
// a single cell whose 27 cells still do not fit is processed straight from global memory.  Every target sees the same
// candidates in the same chunks whichever way its brick was split, so the masks do not depend on the split.
// Arithmetic: every predicate bit is decided by the operations of D:A-FP in their order (per half of a packed
// instruction); the density terms of a chunk are summed in binary32 and the chunk sums joined in binary64.
#include "kernels.h"
#include "sph_common.cuh"

namespace sphb {

namespace {

constexpr int BX = 4, BY = 4, BZ = 2;            // brick of cells per block
constexpr int kMaxRows = (BY + 2) * (BZ + 2);    // x-runs of the staged neighbourhood
constexpr int kBounds = BX + 3;                  // cell bounds per run: cells x0-1 .. x0+BX
constexpr int kMaxCells = BX * BY * BZ;
constexpr int kDThreads = 128;                   // k_density_brick: two targets per thread
constexpr int kTabCap = 16;                      // (mask word, chunk base) entries per thread of k_force_masks
constexpr uint32_t kFull = 0xffffffffu;
// Every barrier below follows loops whose trip counts differ between the lanes of a warp, and bar.sync is an ALIGNED
// barrier (every lane of a warp has to arrive together): __syncwarp() first makes that explicit.
__device__ __forceinline__ void block_sync() {
  __syncwarp();
  __syncthreads();
}

static_assert(kMaxRows <= 32 && kMaxCells <= 32, "one warp scans the rows / cells of a brick");

struct Box {
  int x0, y0, z0, sx, sy, sz;
};

struct BrickTab {
  uint32_t cs[kMaxRows][kBounds + 1];  // bounds of the cells of every staged run, in SLOT SPACE: index into the staged
                                       // arrays when the box is staged, cell-sorted global slot when it is not
  uint32_t g0[kMaxRows];               // global slot of the first particle of each run
  uint32_t off[kMaxRows + 1];          // staged index of the first particle of each run; off[rows] = T
  uint32_t pre[33];                    // density units before each cell of the box: all 32 lanes of warp 0 write their entry
                                       // (lanes past the box's cells repeat the total, which is what the search in
                                       // density_box relies on), entry 32 = the total; so 33 whatever the brick's size
  uint32_t T, ntarget;                 // particles in the neighbourhood, targets in the box
  Box stack[8];
  Box cur;
  int sp, action;
};

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, uint32_t lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(kFull, v, o);
    if (lane >= (uint32_t)o) v += t;
  }
  return v;
}

// Copy the runs into shared memory and turn the bounds into staged indices; ends with a barrier.  Positions are staged
// as three float arrays x[cap], y[cap], z[cap]: two candidates per 8-byte load, and the runs of x-adjacent cells start
// 32 bytes apart on the rest lattice, so the lanes of a warp hit different banks (with float4 records they start 128
// bytes apart -- the same banks -- and every candidate load was a two-way conflict).
__device__ __forceinline__ void brick_stage(BrickTab& tb, const Box& b, const float4* __restrict__ posS, float* sx,
                                            uint32_t cap) {
  const int tid = threadIdx.x, nthreads = blockDim.x;
  const int ny = b.sy + 2, nrows = ny * (b.sz + 2), nb = b.sx + 3;
  for (int idx = tid; idx < nrows * nb; idx += nthreads) {
    const int r = idx / nb, hx = idx - r * nb;
    tb.cs[r][hx] = tb.cs[r][hx] - tb.g0[r] + tb.off[r];
  }
  const int warp = tid >> 5, lane = tid & 31, nwarps = nthreads >> 5;
  for (int r = warp; r < nrows; r += nwarps) {
    const uint32_t o = tb.off[r], len = tb.off[r + 1] - o, gs = tb.g0[r];
    for (uint32_t k = lane; k < len; k += 32) {
      const float4 p = __ldg(posS + gs + k);
      sx[o + k] = p.x, sx[cap + o + k] = p.y, sx[2u * cap + o + k] = p.z;
    }
  }
  block_sync();
}

// The block's brick, clipped to the grid, goes on the stack.
__device__ __forceinline__ void brick_begin(BrickTab& tb, const GridDesc& g, const uint32_t* __restrict__ start) {
  if (threadIdx.x < 32) {
    const int nbx = (g.dim[0] + BX - 1) / BX, nby = (g.dim[1] + BY - 1) / BY;
    const int bx = (int)(blockIdx.x % (uint32_t)nbx), by = (int)((blockIdx.x / (uint32_t)nbx) % (uint32_t)nby),
              bz = (int)(blockIdx.x / ((uint32_t)nbx * (uint32_t)nby));
    Box b;
    b.x0 = bx * BX, b.y0 = by * BY, b.z0 = bz * BZ;
    b.sx = min(BX, g.dim[0] - b.x0), b.sy = min(BY, g.dim[1] - b.y0), b.sz = min(BZ, g.dim[2] - b.z0);
    // most bricks of a sparsely filled box are empty (the fluid of config 2 occupies 3 % of them): the brick's own rows
    // are looked at by one warp first, and an empty brick leaves after one barrier instead of a whole round
    const int lane = (int)threadIdx.x;
    uint32_t cnt = 0;
    if (lane < b.sy * b.sz) {
      const uint32_t row = (uint32_t)g.dim[0] * ((uint32_t)(b.y0 + lane % b.sy) + (uint32_t)g.dim[1] * (uint32_t)(b.z0 + lane / b.sy));
      cnt = __ldg(start + row + b.x0 + b.sx) - __ldg(start + row + b.x0);
    }
    const bool any = __any_sync(kFull, cnt != 0u);
    if (lane == 0) {
      tb.stack[0] = b;
      tb.sp = any ? 1 : 0;
    }
  }
  block_sync();
}

// One round of the box loop: thread 0 pops a box, the block loads the bounds of its runs (global slots; cells outside the
// grid are empty, D:A-BOUND: a run is clipped in x, a row outside in y or z has no particles), and warp 0 scans the run
// lengths, counts the targets, lays out the density pass's units (pairs of targets of one cell) and decides what happens
// to the box -- the decision is lane 0's and travels through shared memory, so every thread acts on the same one.  A box
// without targets is dropped; a box whose neighbourhood exceeds `cap` particles is split (z, then y, then x) unless it
// is one cell, which is then processed from global memory.  Three barriers per round.
enum { kActDone = 0, kActSkip = 1, kActStaged = 2, kActGlobal = 3 };

__device__ __forceinline__ int brick_round(BrickTab& tb, Box& b, const GridDesc& g, const uint32_t* __restrict__ start,
                                           uint32_t cap) {
  const int tid = threadIdx.x, nthreads = blockDim.x;
  if (tid == 0) {
    if (tb.sp == 0) {
      tb.action = kActDone;
    } else {
      tb.sp -= 1;
      tb.cur = tb.stack[tb.sp];
      tb.action = kActSkip;
    }
  }
  block_sync();
  if (tb.action == kActDone) return kActDone;
  b = tb.cur;
  const int ny = b.sy + 2, nrows = ny * (b.sz + 2), nb = b.sx + 3;
  for (int idx = tid; idx < nrows * nb; idx += nthreads) {
    const int r = idx / nb, hx = idx - r * nb;
    const int y = b.y0 - 1 + r % ny, z = b.z0 - 1 + r / ny;
    uint32_t v = 0;
    if (y >= 0 && y < g.dim[1] && z >= 0 && z < g.dim[2]) {
      const int x = min(max(b.x0 - 1 + hx, 0), g.dim[0]);
      v = __ldg(start + (uint32_t)g.dim[0] * ((uint32_t)y + (uint32_t)g.dim[1] * (uint32_t)z) + (uint32_t)x);
    }
    tb.cs[r][hx] = v;
  }
  block_sync();
  if (tid < 32) {
    const bool row = tid < nrows;
    const uint32_t a = row ? tb.cs[tid][0] : 0u, e = row ? tb.cs[tid][nb - 1] : 0u;
    const uint32_t len = e - a;
    const uint32_t inc = warp_incl_scan(len, (uint32_t)tid);
    if (row) {
      tb.g0[tid] = a;
      tb.off[tid] = inc - len;
    }
    if (tid == nrows - 1) tb.off[nrows] = inc;
    const uint32_t T = __shfl_sync(kFull, inc, 31);
    const int hy = tid % ny, hz = tid / ny;
    const bool inside = row && hy >= 1 && hy <= b.sy && hz >= 1 && hz <= b.sz;
    const uint32_t nt = warp_sum_u32(inside ? tb.cs[tid][b.sx + 1] - tb.cs[tid][1] : 0u);
    // units of the density pass before each cell of the box (cell = lane, x fastest); differences of bounds, so the
    // raw global slots serve
    uint32_t u = 0;
    if (tid < b.sx * b.sy * b.sz) {
      const int lx = tid % b.sx, ly = (tid / b.sx) % b.sy, lz = tid / (b.sx * b.sy);
      const int r = (ly + 1) + ny * (lz + 1);
      u = (tb.cs[r][lx + 2] - tb.cs[r][lx + 1] + 1u) >> 1;
    }
    const uint32_t uinc = warp_incl_scan(u, (uint32_t)tid);
    tb.pre[tid] = uinc - u;
    if (tid == 31) tb.pre[32] = uinc;
    if (tid == 0) {
      tb.T = T;
      tb.ntarget = nt;
      int act = kActSkip;
      if (nt != 0) {
        if (T <= cap) {
          act = kActStaged;
        } else if (b.sx * b.sy * b.sz == 1) {
          act = kActGlobal;
        } else {
          Box lo = b, hi = b;
          if (b.sz > 1) {
            lo.sz = b.sz / 2, hi.sz = b.sz - lo.sz, hi.z0 = b.z0 + lo.sz;
          } else if (b.sy > 1) {
            lo.sy = b.sy / 2, hi.sy = b.sy - lo.sy, hi.y0 = b.y0 + lo.sy;
          } else {
            lo.sx = b.sx / 2, hi.sx = b.sx - lo.sx, hi.x0 = b.x0 + lo.sx;
          }
          tb.stack[tb.sp] = hi;
          tb.stack[tb.sp + 1] = lo;
          tb.sp += 2;
        }
      }
      tb.action = act;
    }
  }
  block_sync();
  return tb.action;
}

// ---- S6 -------------------------------------------------------------------------------------------------------------
// rho_i = m C6 sum_{r^2 < h^2} (h^2 - r^2)^3, self included; ncount_i = #{r^2 < h^2}; the
// predicate bits of chunk k (32 candidates from the start of a run, runs in (dz, dy) order) of target i go to
// masks[w * stride + i], w counting the target's chunks; candidate j of the chunk is bit 31 - j.
//
// A thread owns two targets A, B of one cell.  Staged: two candidates per step, loaded as (x0,x1), (y0,y1), (z0,z1);
// per target three packed subtractions, dist2 and r^2 - h^2 on packed binary32 -- the scalar test's operations in its
// order per half, so every predicate bit is the scalar one (D:A-FP).  A chunk that starts or ends on an odd slot does
// that candidate alone, with the two TARGETS in the two halves.  The terms max(h^2 - r^2, 0)^3 of a chunk are summed in
// binary32 (<= 32 terms in four partial sums) and the chunk sums joined in binary64.
struct DensAcc {
  f32x2 accA, accB;  // sums over candidate pairs, per target
  f32x2 accAB;       // sums over single candidates: lo = target A, hi = target B
  uint32_t maskA, maskB;
};

__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}

// One target against two candidates.
__device__ __forceinline__ void test_two(f32x2 tx, f32x2 ty, f32x2 tz, f32x2 X, f32x2 Y, f32x2 Z, f32x2 neg_h2,
                                         uint32_t& mask, f32x2& acc) {
  const f32x2 dx = sub2(tx, X), dy = sub2(ty, Y), dz = sub2(tz, Z);
  const f32x2 t2 = add2(fma2(dz, dz, fma2(dy, dy, mul2(dx, dx))), neg_h2);
  float t0, t1;
  unpack2(t2, t0, t1);
  mask = __funnelshift_l(__float_as_uint(t0), mask, 1);
  mask = __funnelshift_l(__float_as_uint(t1), mask, 1);
  const f32x2 m = pack2(fmaxf(-t0, 0.0f), fmaxf(-t1, 0.0f));
  acc = fma2(mul2(m, m), m, acc);
}

template <bool SM>
__device__ __forceinline__ void density_box(const SphConst& c, BrickTab& tb, const Box& b, const float* sx, uint32_t cap,
                                            const float4* __restrict__ posS, const uint32_t* __restrict__ perm,
                                            float* __restrict__ rhoS, float4* __restrict__ velS,
                                            float* __restrict__ density_out, uint32_t* __restrict__ ncount_out,
                                            uint32_t* __restrict__ masks, uint32_t stride) {
  const int tid = threadIdx.x;
  const int ny = b.sy + 2;
  const float* sy = sx + cap;
  const float* sz = sx + 2u * cap;
  const uint32_t U = tb.pre[32];
  const f32x2 neg_h2 = pack2(-c.h2, -c.h2);
#pragma unroll 1
  for (uint32_t u = (uint32_t)tid; u < U; u += (uint32_t)kDThreads) {
    int ci = 0;
#pragma unroll
    for (int st = 16; st > 0; st >>= 1)
      if (tb.pre[ci + st] <= u) ci += st;
    const int lx = ci % b.sx, ly = (ci / b.sx) % b.sy, lz = ci / (b.sx * b.sy);
    const int r0 = (ly + 1) + ny * (lz + 1);
    const uint32_t a = tb.cs[r0][lx + 1] + 2u * (u - tb.pre[ci]);
    const bool hasB = a + 1u < tb.cs[r0][lx + 2];
    const uint32_t iA = SM ? a - tb.off[r0] + tb.g0[r0] : a;
    const uint32_t bslot = hasB ? a + 1u : a;
    float3 pA, pB;
    if (SM) {
      pA = make_float3(sx[a], sy[a], sz[a]);
      pB = make_float3(sx[bslot], sy[bslot], sz[bslot]);
    } else {
      const float4 qa = __ldg(posS + a), qb = __ldg(posS + bslot);
      pA = make_float3(qa.x, qa.y, qa.z);
      pB = make_float3(qb.x, qb.y, qb.z);
    }
    const f32x2 ax2 = pack2(pA.x, pA.x), ay2 = pack2(pA.y, pA.y), az2 = pack2(pA.z, pA.z);
    const f32x2 bx2 = pack2(pB.x, pB.x), by2 = pack2(pB.y, pB.y), bz2 = pack2(pB.z, pB.z);
    const f32x2 abx = pack2(pA.x, pB.x), aby = pack2(pA.y, pB.y), abz = pack2(pA.z, pB.z);
    double SA = 0.0, SB = 0.0;
    uint32_t cntA = 0, cntB = 0, w = 0;
    // word w of target i: masks[w * stride + i]; the lanes' targets are consecutive, so a warp's stores of one word
    // fall into a few 128-byte lines.  (Tiles of 256 particles, word-major inside a tile -- all words of a particle within
    // 32 KB -- measured no better at 4 M particles and 3 % worse here: it is not the TLB that the long stride costs.)
    uint32_t* mcol = masks + iA;
#pragma unroll 1
    for (int dz = 0; dz < 3; ++dz)
#pragma unroll 1
      for (int dy = 0; dy < 3; ++dy) {
        const int r = (ly + dy) + ny * (lz + dz);
        const uint32_t s0 = tb.cs[r][lx], s1 = tb.cs[r][lx + 3];
#pragma unroll 1
        for (uint32_t c0 = s0; c0 < s1; c0 += 32u) {
          const uint32_t ce = min(c0 + 32u, s1), nc = ce - c0;
          DensAcc d;
          d.accA = d.accB = d.accAB = pack2(0.0f, 0.0f);
          d.maskA = d.maskB = 0u;
          uint32_t s = c0;
#define SPHB_SINGLE(S)                                                                                      \
  {                                                                                                         \
    float qx, qy, qz;                                                                                       \
    if (SM) {                                                                                               \
      qx = sx[S], qy = sy[S], qz = sz[S];                                                                   \
    } else {                                                                                                \
      const float4 q4 = __ldg(posS + (S));                                                                  \
      qx = q4.x, qy = q4.y, qz = q4.z;                                                                      \
    }                                                                                                       \
    PairAcc pa;                                                                                             \
    pa.acc = d.accAB, pa.maskA = d.maskA, pa.maskB = d.maskB;                                               \
    pair_test(pa, sub2(abx, pack2(qx, qx)), sub2(aby, pack2(qy, qy)), sub2(abz, pack2(qz, qz)), neg_h2);    \
    d.accAB = pa.acc, d.maskA = pa.maskA, d.maskB = pa.maskB;                                               \
  }
#define SPHB_TWO(S)                                                                                         \
  {                                                                                                         \
    const f32x2 X = *reinterpret_cast<const f32x2*>(sx + (S)), Y = *reinterpret_cast<const f32x2*>(sy + (S)), \
                Z = *reinterpret_cast<const f32x2*>(sz + (S));                                              \
    test_two(ax2, ay2, az2, X, Y, Z, neg_h2, d.maskA, d.accA);                                              \
    test_two(bx2, by2, bz2, X, Y, Z, neg_h2, d.maskB, d.accB);                                              \
  }
          if (SM) {
            if (s & 1u) {  // 8-byte loads need an even slot
              SPHB_SINGLE(s);
              ++s;
            }
#pragma unroll 1
            for (; s + 4u <= ce; s += 4u) {
              SPHB_TWO(s);
              SPHB_TWO(s + 2u);
            }
            if (s + 2u <= ce) {
              SPHB_TWO(s);
              s += 2u;
            }
            if (s < ce) SPHB_SINGLE(s);
          } else {
#pragma unroll 1
            for (; s < ce; ++s) SPHB_SINGLE(s);
          }
#undef SPHB_SINGLE
#undef SPHB_TWO
          const uint32_t mA = d.maskA << (32u - nc), mB = d.maskB << (32u - nc);  // candidate j of the chunk -> bit 31 - j
          cntA += __popc(mA), cntB += __popc(mB);
          if (w < (uint32_t)kNbrMaskWords) {
            mcol[(size_t)w * stride] = mA;
            if (hasB) mcol[(size_t)w * stride + 1] = mB;
          }
          ++w;
          float a0, a1, b0, b1, e0, e1;
          unpack2(d.accA, a0, a1), unpack2(d.accB, b0, b1), unpack2(d.accAB, e0, e1);
          SA += (double)((a0 + a1) + e0);
          SB += (double)((b0 + b1) + e1);
        }
      }
    const float rhoA = (float)((double)c.mass_c6 * SA), rhoB = (float)((double)c.mass_c6 * SB);
    rhoS[iA] = rhoA;
    reinterpret_cast<float*>(velS + iA)[3] = 1.0f / rhoA;  // the force passes pick 1 / rho_j up with the neighbour's velocity
    if (hasB) {
      rhoS[iA + 1] = rhoB;
      reinterpret_cast<float*>(velS + iA + 1)[3] = 1.0f / rhoB;
    }
    if (density_out || ncount_out) {
      const uint32_t idA = __ldg(perm + iA);
      if (density_out) density_out[idA] = rhoA;
      if (ncount_out) ncount_out[idA] = cntA;
      if (hasB) {
        const uint32_t idB = __ldg(perm + iA + 1);
        if (density_out) density_out[idB] = rhoB;
        if (ncount_out) ncount_out[idB] = cntB;
      }
    }
  }
}

__global__ void __launch_bounds__(kDThreads, 8) k_density_brick(SphConst c, const float4* __restrict__ posS,
                                                             const uint32_t* __restrict__ start,
                                                             const uint32_t* __restrict__ perm,
                                                             float* __restrict__ rhoS, float4* __restrict__ velS,
                                                             float* __restrict__ density_out,
                                                             uint32_t* __restrict__ ncount_out,
                                                             uint32_t* __restrict__ masks, uint32_t stride,
                                                             uint32_t cap) {
  extern __shared__ __align__(16) unsigned char brick_dyn[];
  float* sx = reinterpret_cast<float*>(brick_dyn);
  __shared__ BrickTab tb;
  brick_begin(tb, c.grid, start);
  Box b;
  for (;;) {
    const int act = brick_round(tb, b, c.grid, start, cap);
    if (act == kActDone) break;
    if (act == kActStaged) {
      brick_stage(tb, b, posS, sx, cap);
      density_box<true>(c, tb, b, sx, cap, posS, perm, rhoS, velS, density_out, ncount_out, masks, stride);
    } else if (act == kActGlobal) {
      density_box<false>(c, tb, b, sx, cap, posS, perm, rhoS, velS, density_out, ncount_out, masks, stride);
    }
    block_sync();  // the staged arrays, the tables and the decision are reused by the next round
  }
}

// ---- S8-S10 ---------------------------------------------------------------------------------------------------------
// ---- S8-S10 from the mask words ------------------------------------------------------------------------------------
// One thread per cell-sorted particle.  Prologue: the non-empty mask words of the particle and the cell-sorted slot of
// the first candidate of their chunks (the chunks are those of k_density_brick: 32 candidates from the start of a run)
// go into the thread's column of a shared table of kTabCap entries; a full table is consumed before the walk goes on.
// Main loop: the thread walks the table's words as ONE bit stream -- next set bit -> slot -> two 16-byte gathers from
// global memory (L1 / L2) -- two neighbours per trip on packed binary32, so a lane's trips are half its neighbour count
// whatever the spread of the bits over the chunks, and no lane waits for another lane's chunk.  A particle with more
// chunks than mask words walks the grid instead.  (A brick-staged consumer, k_force_brick, with the neighbours'
// records gathered from shared memory was built and measured: 250 us against 192 us at config 4, 6.6 ms against
// 2.1 ms at config 5 where its bricks split down to a few cells; DESIGN.md section 10.  It is not kept.)
constexpr int kMThreads = 128;

__global__ void __launch_bounds__(kMThreads)
k_force_masks(SphConst c, BoidConst bc, bool has_boids, const float4* __restrict__ posS,
              const float4* __restrict__ velS, const uint32_t* __restrict__ start, const uint32_t* __restrict__ perm,
              uint32_t n, const float* __restrict__ rhoS, const uint32_t* __restrict__ masks, uint32_t stride,
              const float4* __restrict__ bposS, const float4* __restrict__ bvelS, const float* __restrict__ rho_bS,
              const uint32_t* __restrict__ bstart, float4* __restrict__ pos, float4* __restrict__ vel,
              float4* __restrict__ accel_out, uint32_t* __restrict__ touched_out) {
  __shared__ uint32_t s_tabm[kTabCap * kMThreads], s_tabb[kTabCap * kMThreads];
  uint32_t* tabm = s_tabm + threadIdx.x;
  uint32_t* tabb = s_tabb + threadIdx.x;
  const uint32_t i = blockIdx.x * kMThreads + threadIdx.x;
  if (i >= n) return;  // no barrier and no warp-wide operation below
  const float4 pi = __ldg(posS + i);
  float4 vi = __ldg(velS + i);
  vi.w = __ldg(rhoS + i);
  const CellOf wk = walk_init(c.grid, pi);
  const PairConst kf = make_pair_const(c, c.h);
  const PairConst2 kf2 = make_pair_const2(kf);
  const f32x2 rho_m = pack2(vi.w - 2.0f * c.rho0, vi.w - 2.0f * c.rho0);
  ForceAcc F = {0.0, 0.0, 0.0};
  uint32_t ne = 0;
  auto consume = [&]() {
    uint32_t e = 0, m = 0, base = 0;
    // next two set bits of the stream -> slots; false when the stream is exhausted.  An odd count leaves the second
    // half on the target itself: r^2 = 0, no force
    auto pop2 = [&](uint32_t& sl0, uint32_t& sl1) -> bool {
      sl0 = sl1 = i;
      if (m == 0u) {
        if (e == ne) return false;
        m = tabm[e * kMThreads], base = tabb[e * kMThreads], ++e;
      }
      uint32_t j = __clz(m);
      m ^= 0x80000000u >> j;
      sl0 = base + j;
      if (m == 0u && e != ne) m = tabm[e * kMThreads], base = tabb[e * kMThreads], ++e;
      if (m != 0u) {
        j = __clz(m);
        m ^= 0x80000000u >> j;
        sl1 = base + j;
      }
      return true;
    };
    uint32_t a0, a1;
    bool more = pop2(a0, a1);
#pragma unroll 1
    while (more) {
      // the gathers of this pair are issued, then the next pair's slots are popped while they are in flight
      const float4 p0 = __ldg(posS + a0), v0 = __ldg(velS + a0), p1 = __ldg(posS + a1), v1 = __ldg(velS + a1);
      more = pop2(a0, a1);
      eval_two(kf2, p0, v0, p1, v1, pi, vi, rho_m, F);
    }
    ne = 0;
  };
  // word w: mcol[w * stride], one coalesced load per warp; fetched four words ahead (the rows live in L2 / HBM)
  const uint32_t* mcol = masks + i;
  uint32_t q0 = __ldg(mcol), q1 = __ldg(mcol + stride), q2 = __ldg(mcol + 2u * (size_t)stride),
           q3 = __ldg(mcol + 3u * (size_t)stride);
  uint32_t w = 0;
  bool overflow = false;
#pragma unroll 1
  for (int r9 = 0; r9 < 9 && !overflow; ++r9) {
    uint32_t s0 = 0, s1 = 0;
    walk_row(c.grid, start, wk, r9 % 3 - 1, r9 / 3 - 1, s0, s1);
#pragma unroll 1
    for (uint32_t c0 = s0; c0 < s1; c0 += 32u) {
      if (w == (uint32_t)kNbrMaskWords) {  // more chunks than mask words
        overflow = true;
        break;
      }
      const uint32_t m = q0;
      q0 = q1, q1 = q2, q2 = q3;
      ++w;
      if (w + 3u < (uint32_t)kNbrMaskWords) q3 = __ldg(mcol + (size_t)(w + 3u) * stride);
      if (m != 0u) {
        tabm[ne * kMThreads] = m;
        tabb[ne * kMThreads] = c0;
        if (++ne == (uint32_t)kTabCap) consume();
      }
    }
  }
  consume();
  if (overflow) {  // start again on the grid
    const float4 pw = pi, vw = vi;
    ForceAcc Fw = {0.0, 0.0, 0.0};
    walk_force<true>(c, kf, posS, velS, start, pw, vw, wk, Fw);
    F = Fw;
  }
  push_integrate_store(c, bc, has_boids, true, i, pi, vi, F, perm, bposS, bvelS, rho_bS, bstart, pos, vel, accel_out,
                       touched_out);
}

uint32_t brick_blocks(const GridDesc& g) {
  return (uint32_t)(((g.dim[0] + BX - 1) / BX) * ((g.dim[1] + BY - 1) / BY) * ((g.dim[2] + BZ - 1) / BZ));
}

}  // namespace

// Staging capacity (particles of a box's neighbourhood).  A brick of config 4 holds 144 cells x 8 = 1152 particles; a
// box that exceeds the capacity is split, so the choice only moves where the split happens.
constexpr uint32_t kBrickCap = 2048;   // k_density_brick: 24 KB of x / y / z
void launch_density_brick(const SphConst& c, const GridBuf& b, uint32_t n, float* rhoS, float* density_out,
                          uint32_t* ncount_out, uint32_t* masks, uint32_t stride, cudaStream_t s, Prof* prof) {
  if (n == 0) return;
  const size_t smem = (size_t)kBrickCap * 12;
  prof->begin(K_DENSITY_BRICK, s);
  k_density_brick<<<brick_blocks(c.grid), kDThreads, smem, s>>>(c, b.posS, b.start, b.perm, rhoS, b.velS, density_out,
                                                                ncount_out, masks, stride, kBrickCap);
  prof->end(s);
}

void launch_force_masks(const SphConst& c, const BoidConst* bc, const GridBuf& pg, const GridBuf& bg, uint32_t n,
                        uint32_t nb, const float* rhoS, const float* rho_bS, float4* pos, float4* vel, float4* accel_out,
                        uint32_t* touched_out, const uint32_t* masks, uint32_t stride, cudaStream_t s, Prof* prof) {
  if (n == 0) return;
  BoidConst dummy = {};
  const bool has = nb > 0 && bc != nullptr;
  prof->begin(K_FORCE_MASKS, s);
  k_force_masks<<<(n + kMThreads - 1) / kMThreads, kMThreads, 0, s>>>(
      c, has ? *bc : dummy, has, pg.posS, pg.velS, pg.start, pg.perm, n, rhoS, masks, stride, bg.posS, bg.velS, rho_bS,
      bg.start, pos, vel, accel_out, touched_out);
  prof->end(s);
}

}  // namespace sphb
