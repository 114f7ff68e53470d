// microbenchmarks: throughput (many independent chains, full occupancy) and dependent latency of FFMA, DFMA, MUFU, F2F
#include <cstdio>
#include <cuda_runtime.h>
#define ITER 4096
template <int OP, int ILP> __global__ void k(float* out, float a, double da) {
  float x[ILP]; double d[ILP];
  for (int i = 0; i < ILP; ++i) { x[i] = a + threadIdx.x + i; d[i] = da + threadIdx.x + i; }
  for (int it = 0; it < ITER; ++it) {
#pragma unroll
    for (int i = 0; i < ILP; ++i) {
      if (OP == 0) x[i] = fmaf(x[i], a, 1.0f);
      if (OP == 1) d[i] = fma(d[i], da, 1.0);
      if (OP == 2) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
      if (OP == 3) { float t = (float)d[i]; d[i] = (double)t + 1e-30 * it; }   // F2F.F32.F64 + F2F.F64.F32 + DADD
      if (OP == 4) d[i] = d[i] + da;
      if (OP == 5) d[i] = d[i] * da;
      if (OP == 6) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
      if (OP == 7) { x[i] = fmaf(x[i], a, 1.0f); d[i] = fma(d[i], da, 1.0); }  // mixed 1:1
      if (OP == 8) { x[i] = fmaf(x[i], a, 1.0f); x[i] = fmaf(x[i], a, 2.0f); x[i] = fmaf(x[i], a, 3.0f); d[i] = fma(d[i], da, 1.0); }  // 3:1
      if (OP == 9) { d[i] = fma(d[i], da, 1.0); asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i])); }
    }
  }
  float s = 0; for (int i = 0; i < ILP; ++i) s += x[i] + (float)d[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int OP, int ILP> void run(const char* name, int blocks, int threads, int ops_per_iter) {
  float* out; cudaMalloc(&out, (size_t)blocks * threads * 4);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  k<OP, ILP><<<blocks, threads>>>(out, 0.999f, 0.999);
  cudaEventRecord(e0);
  k<OP, ILP><<<blocks, threads>>>(out, 0.999f, 0.999);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  double warp_inst = (double)blocks * threads / 32 * ITER * ILP * ops_per_iter;
  double cyc = ms * 1e-3 * 1.965e9;
  int sms = 148;
  printf("%-28s blocks %5d thr %4d ILP %d: %.3f ms, %.3f warp-inst/clk/SM (%.1f lanes/clk/SM), cycles per dependent step per warp %.1f\n",
         name, blocks, threads, ILP, ms, warp_inst / cyc / sms, warp_inst / cyc / sms * 32, cyc / ITER);
  cudaFree(out);
}
int main() {
  // throughput: 148*8 blocks x 256 threads, ILP 4
  run<0, 4>("FFMA throughput", 148 * 8, 256, 1);
  run<1, 4>("DFMA throughput", 148 * 8, 256, 1);
  run<4, 4>("DADD throughput", 148 * 8, 256, 1);
  run<5, 4>("DMUL throughput", 148 * 8, 256, 1);
  run<2, 4>("MUFU.EX2 throughput", 148 * 8, 256, 1);
  run<6, 4>("MUFU.RCP throughput", 148 * 8, 256, 1);
  run<3, 4>("F2F pair+DADD throughput", 148 * 8, 256, 3);
  run<7, 4>("FFMA+DFMA 1:1", 148 * 8, 256, 2);
  run<8, 4>("FFMA+DFMA 3:1", 148 * 8, 256, 4);
  run<9, 4>("DFMA+MUFU 1:1", 148 * 8, 256, 2);
  // latency: one warp per SM, ILP 1
  run<0, 1>("FFMA latency", 148, 32, 1);
  run<1, 1>("DFMA latency", 148, 32, 1);
  run<4, 1>("DADD latency", 148, 32, 1);
  run<2, 1>("MUFU.EX2 latency", 148, 32, 1);
  run<3, 1>("F2F pair+DADD latency", 148, 32, 3);
  // DFMA at limited occupancy: 4 warps per SMSP (512 thr/SM), ILP 1, 2, 4
  run<1, 1>("DFMA 16 warps/SM ILP1", 148, 512, 1);
  run<1, 2>("DFMA 16 warps/SM ILP2", 148, 512, 1);
  run<1, 4>("DFMA 16 warps/SM ILP4", 148, 512, 1);
  run<1, 8>("DFMA 16 warps/SM ILP8", 148, 512, 1);
  return 0;
}
