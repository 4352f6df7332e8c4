// probes/fp32_pipes.cu -- microbenchmark behind DESIGN.md section 1 / 7: issue rate of FFMA, packed FFMA2
// (fma.rn.f32x2), FFMA + FMNMX mixes, FADD and DADD on sm_100a.  Not part of libsphboid; build and run by hand:
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o fp32_pipes paper_2311_15088_b200/csrc/probes/fp32_pipes.cu && ./fp32_pipes
// Result on this pool's B200: profiles/r01_fp32_pipes.txt.
// microbench: FFMA vs FFMA2 (fma.rn.f32x2) vs mixed pipes on sm_100a
#include <cstdio>
#include <cuda_runtime.h>
#define ITERS 4096
template <int MODE>
__global__ void k(float* out, float a, float b) {
  float x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 0.001f + i;
  for (int it = 0; it < ITERS; ++it) {
    if (MODE == 0) {
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
    } else if (MODE == 1) {
#pragma unroll
      for (int i = 0; i < 16; i += 2) {
        unsigned long long v, av, bv;
        asm("mov.b64 %0, {%1,%2};" : "=l"(v) : "f"(x[i]), "f"(x[i + 1]));
        asm("mov.b64 %0, {%1,%2};" : "=l"(av) : "f"(a), "f"(a));
        asm("mov.b64 %0, {%1,%2};" : "=l"(bv) : "f"(b), "f"(b));
        asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(v) : "l"(v), "l"(av), "l"(bv));
        asm("mov.b64 {%0,%1}, %2;" : "=f"(x[i]), "=f"(x[i + 1]) : "l"(v));
      }
    } else if (MODE == 2) {  // 8 ffma + 8 fmnmx
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = fmaf(x[i], a, b);
#pragma unroll
      for (int i = 8; i < 16; ++i) x[i] = fmaxf(x[i], x[i - 8]);
    } else if (MODE == 3) {  // 16 ffma + 8 fmnmx (are the fmnmx free?)
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
#pragma unroll
      for (int i = 8; i < 16; ++i) x[i] = fmaxf(x[i], a);
    } else if (MODE == 4) {  // 16 fadd
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = x[i] + a;
    } else if (MODE == 5) {  // 8 ffma2 (16 fma) + 8 fmnmx
#pragma unroll
      for (int i = 0; i < 16; i += 2) {
        unsigned long long v, av, bv;
        asm("mov.b64 %0, {%1,%2};" : "=l"(v) : "f"(x[i]), "f"(x[i + 1]));
        asm("mov.b64 %0, {%1,%2};" : "=l"(av) : "f"(a), "f"(a));
        asm("mov.b64 %0, {%1,%2};" : "=l"(bv) : "f"(b), "f"(b));
        asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(v) : "l"(v), "l"(av), "l"(bv));
        asm("mov.b64 {%0,%1}, %2;" : "=f"(x[i]), "=f"(x[i + 1]) : "l"(v));
      }
#pragma unroll
      for (int i = 8; i < 16; ++i) x[i] = fmaxf(x[i], a);
    } else if (MODE == 6) {  // 16 dadd-ish: fp64 add
      double* d = reinterpret_cast<double*>(x);
#pragma unroll
      for (int i = 0; i < 8; ++i) d[i] = d[i] + (double)a;
    }
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int MODE>
void run(const char* name, double ops_per_iter) {
  float* out;
  cudaMalloc(&out, 148 * 8 * 256 * 4);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0), cudaEventCreate(&e1);
  k<MODE><<<148 * 8, 256>>>(out, 1.0001f, 0.5f);
  cudaEventRecord(e0);
  for (int r = 0; r < 5; ++r) k<MODE><<<148 * 8, 256>>>(out, 1.0001f, 0.5f);
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms;
  cudaEventElapsedTime(&ms, e0, e1);
  ms /= 5;
  double lane_ops = (double)148 * 8 * 256 * ITERS * ops_per_iter;
  printf("%-28s %.3f ms  %.2f T lane-ops/s (ops counted as scalar results)\n", name, ms, lane_ops / ms / 1e9);
  cudaFree(out);
}
int main() {
  run<0>("16 FFMA", 16);
  run<1>("8 FFMA2 (=16 fma)", 16);
  run<2>("8 FFMA + 8 FMNMX", 16);
  run<3>("16 FFMA + 8 FMNMX", 24);
  run<4>("16 FADD", 16);
  run<5>("8 FFMA2 + 8 FMNMX", 24);
  run<6>("8 DADD", 8);
  return 0;
}
