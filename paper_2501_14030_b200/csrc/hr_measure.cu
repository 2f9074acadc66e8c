// hr_measure.cu -- measurement hooks of include/hr.h that need no solver: the FP64 / FP32 FMA peak of the
// device (the secondary roof of SURVEY.md section 8(d)) and the launch-latency floor of a graph of n dependent
// launches (the floor under a step on L2-resident grids).  Product code; shares nothing with
// oracle/.
#include <cuda_runtime.h>

#include <cstdio>

#include "hr_internal.h"

namespace {

template <typename T, int CH>
__global__ void __launch_bounds__(1024) k_alu(T* out, int iters, T a, T b) {
  T x[CH];
#pragma unroll
  for (int c = 0; c < CH; ++c) x[c] = T(threadIdx.x + c) * T(1e-3);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int c = 0; c < CH; ++c) x[c] = x[c] * a + b;  // contracted to one FMA per chain
  }
  T s = T(0);
#pragma unroll
  for (int c = 0; c < CH; ++c) s += x[c];
  if (s == T(-1)) out[0] = s;  // never true; keeps the chains alive
}

template <int CH>
__global__ void __launch_bounds__(1024) k_alu_f32x2(float* out, int iters, float a, float b) {
  unsigned long long x[CH], aa, bb;
  asm("mov.b64 %0, {%1, %1};" : "=l"(aa) : "f"(a));
  asm("mov.b64 %0, {%1, %1};" : "=l"(bb) : "f"(b));
#pragma unroll
  for (int c = 0; c < CH; ++c) {
    const float v = (threadIdx.x + c) * 1e-3f;
    asm("mov.b64 %0, {%1, %1};" : "=l"(x[c]) : "f"(v));
  }
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int c = 0; c < CH; ++c) asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[c]) : "l"(aa), "l"(bb));
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < CH; ++c) {
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(x[c]));
    s += lo + hi;
  }
  if (s == -1.f) out[0] = s;
}

__global__ void k_empty() {}

}  // namespace

cudaError_t hrk_measure_alu(cudaStream_t st, int dtype, int packed, double* tflops) {
  constexpr int CH = 8, ITERS = 4096;
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
  void* out = nullptr;
  if ((e = cudaMalloc(&out, 64)) != cudaSuccess) return e;
  const int grid = sms * 8;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best_ms = 1e30;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    if (dtype == HR_F64)
      k_alu<double, CH><<<grid, 1024, 0, st>>>(static_cast<double*>(out), ITERS, 0.999999, 1e-7);
    else if (packed)
      k_alu_f32x2<CH><<<grid, 1024, 0, st>>>(static_cast<float*>(out), ITERS, 0.999999f, 1e-7f);
    else
      k_alu<float, CH><<<grid, 1024, 0, st>>>(static_cast<float*>(out), ITERS, 0.999999f, 1e-7f);
    cudaEventRecord(e1, st);
    if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best_ms) best_ms = ms;  // the first launch is the warm-up
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (e != cudaSuccess) return e;
  const double fmas = (double)grid * 1024.0 * ITERS * CH * ((dtype == HR_F32 && packed) ? 2.0 : 1.0);
  *tflops = 2.0 * fmas / (best_ms * 1e-3) / 1e12;
  return cudaGetLastError();
}

cudaError_t hrk_measure_launch_floor(cudaStream_t st, int nodes, int grid, int block, int reps,
                                     double* us_per_graph) {
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  cudaError_t e = cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal);
  if (e != cudaSuccess) return e;
  for (int i = 0; i < nodes; ++i) k_empty<<<grid, block, 0, st>>>();
  e = cudaStreamEndCapture(st, &graph);
  if (e != cudaSuccess) return e;
  e = cudaGraphInstantiate(&exec, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) return e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  for (int i = 0; i < 10; ++i) cudaGraphLaunch(exec, st);
  cudaEventRecord(e0, st);
  for (int i = 0; i < reps; ++i) cudaGraphLaunch(exec, st);
  cudaEventRecord(e1, st);
  e = cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaGraphExecDestroy(exec);
  if (e != cudaSuccess) return e;
  *us_per_graph = 1e3 * ms / reps;
  return cudaGetLastError();
}
