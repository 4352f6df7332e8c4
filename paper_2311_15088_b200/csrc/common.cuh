// common.cuh -- shared device helpers of libsphboid (CUDA, sm_100a).
// "P:n" = PAPER.md line n (arXiv 2311.15088); "D:X" = reading X in DESIGN.md section 3.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace sphb {

// Uniform grid over [lo, lo + dim*cell): P:389-395 (Eq. 47 get_cell, hash), D:A-DIMS, D:A-CLAMPCELL.
struct GridDesc {
  float lo[3];
  float cell;
  int dim[3];
  uint32_t C;
};

// P:391 Eq. 47: c = floor((p - m)/d) with IEEE subtract and divide (D:A-FP), clamped to [0, dim-1].
__device__ __forceinline__ int cell_coord(float p, float lo, float cell, int dim) {
  float t = __fdiv_rn(__fsub_rn(p, lo), cell);
  int c = __float2int_rd(t);
  return min(max(c, 0), dim - 1);
}

// hash(cx,cy,cz) = cx + dimx*(cy + dimy*cz)
__device__ __forceinline__ uint32_t cell_hash(const GridDesc& g, int cx, int cy, int cz) {
  return (uint32_t)cx + (uint32_t)g.dim[0] * ((uint32_t)cy + (uint32_t)g.dim[1] * (uint32_t)cz);
}

// D:A-FP: r^2 = fma(dz,dz, fma(dy,dy, dx*dx)) -- the arithmetic every integer decision is taken in.
__device__ __forceinline__ float dist2(float dx, float dy, float dz) {
  return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// Order-preserving map binary32 -> uint32 (for atomicMin / atomicMax on floats).
__device__ __forceinline__ uint32_t encode_ordered(float f) {
  const uint32_t b = __float_as_uint(f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

__device__ __forceinline__ uint32_t warp_sum_u32(uint32_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__device__ __forceinline__ double warp_sum_f64(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---- single-pass device-wide exclusive scan: block-local scan + decoupled look-back -------------------
// One 64-bit status word per tile: high 32 bits = flag, low 32 bits = value.  Flags are tagged with the
// launch epoch (2*epoch+1 = tile aggregate ready, 2*epoch+2 = inclusive prefix ready), so words left by an
// earlier launch read as "not ready" and the array never needs clearing.  Tiles are handed out by a ticket
// counter, so a tile's predecessors are always already running: the spin below cannot deadlock.  Epoch and ticket
// live in device memory and are advanced / reset by the last block of a launch to retire (scan_end), so a launch
// carries no host-side state and the kernels can be replayed from a CUDA graph.
struct ScanState {
  unsigned long long* status;  // [max_tiles]
  uint32_t* ticket;            // next tile of the running launch; back to 0 when the launch's last block retires
  uint32_t* ctl;               // [2] = {launch epoch (> 0), blocks of the running launch that have retired}
  uint32_t epoch;              // the running launch's epoch: filled in on the device by scan_begin (0 on the host)
};

__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Called by the 32 threads of ONE warp of the block.  Returns the exclusive prefix of `tile`
// (sum of the aggregates of tiles 0..tile-1) and publishes this tile's inclusive prefix.
__device__ __forceinline__ uint32_t lookback_exclusive(const ScanState& st, uint32_t tile, uint32_t aggregate) {
  const uint32_t lane = threadIdx.x & 31u;
  const unsigned long long flagA = (unsigned long long)(2u * st.epoch + 1u) << 32;
  const unsigned long long flagP = (unsigned long long)(2u * st.epoch + 2u) << 32;
  if (tile == 0) {
    if (lane == 0) st_status(st.status, flagP | aggregate);
    return 0u;
  }
  if (lane == 0) st_status(st.status + tile, flagA | aggregate);
  uint32_t exclusive = 0;
  int base = (int)tile - 1;
  while (true) {
    const int idx = base - (int)lane;
    unsigned long long s;
    bool ready;
    do {
      s = idx >= 0 ? ld_status(st.status + idx) : flagP;
      const unsigned long long f = s & 0xffffffff00000000ull;
      ready = (f == flagA) || (f == flagP);
    } while (!__all_sync(0xffffffffu, ready));
    const bool is_p = (s & 0xffffffff00000000ull) == flagP;
    const uint32_t pmask = __ballot_sync(0xffffffffu, is_p);
    const int first_p = pmask ? (__ffs(pmask) - 1) : 32;
    uint32_t v = ((int)lane <= first_p) ? (uint32_t)s : 0u;
    exclusive += warp_sum_u32(v);
    if (pmask) break;
    base -= 32;
  }
  if (lane == 0) st_status(st.status + tile, flagP | (exclusive + aggregate));
  return exclusive;
}

// Thread 0 of a block: take a tile and read the launch's epoch (unchanged until every block has retired).
__device__ __forceinline__ uint32_t scan_begin(const ScanState& st, uint32_t* epoch_out) {
  const uint32_t tile = atomicAdd(st.ticket, 1u);
  uint32_t e;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(e) : "l"(st.ctl) : "memory");
  *epoch_out = e;
  return tile;
}
// Thread 0 of a block, once the block no longer reads or writes the status words: the last of the launch's n_tiles
// blocks re-arms the state for the next launch.
__device__ __forceinline__ void scan_end(const ScanState& st, uint32_t n_tiles) {
  __threadfence();
  if (atomicAdd(st.ctl + 1, 1u) == n_tiles - 1u) {
    *st.ticket = 0u;
    st.ctl[1] = 0u;
    st.ctl[0] = st.epoch + 1u;
    __threadfence();
  }
}

// Block-wide exclusive scan of one value per thread (blockDim.x <= 1024, multiple of 32).
// `smem` holds 33 uint32.  Returns the exclusive prefix; *total gets the block sum.
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* smem, uint32_t* total) {
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= (uint32_t)o) inc += t;
  }
  if (lane == 31) smem[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    const uint32_t nw = blockDim.x >> 5;
    uint32_t w = lane < nw ? smem[lane] : 0u;
    uint32_t winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= (uint32_t)o) winc += t;
    }
    smem[lane] = winc - w;  // exclusive prefix of each warp
    if (lane == 31) smem[32] = winc;
  }
  __syncthreads();
  const uint32_t r = smem[warp] + inc - v;
  *total = smem[32];
  __syncthreads();
  return r;
}

}  // namespace sphb
