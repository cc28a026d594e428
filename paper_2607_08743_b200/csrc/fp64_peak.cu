// fp64_peak.cu -- FP64 pipe microbenchmark behind the roofline's ALU ceiling (BASELINE.md
// section 3): register-only chains of DFMA / DADD / DMUL on every SM, `ilp` independent chains per thread,
// `warps` warps per SM. Reports instructions per second; not part of the libsacra ABI.
#include <cuda_runtime.h>

template <int ILP, int OP>
__global__ void k_chain(double* out, int iters, double a, double b) {
  double x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) x[i] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = OP == 0 ? fma(x[i], a, b) : (OP == 1 ? x[i] + a : x[i] * a);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < ILP; ++i) s += x[i];
  if (s == 123.456) out[0] = s;   // never true: keeps the chains alive
}

template <int ILP, int OP>
static double run(int sms, int warps, int iters, double* out) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  k_chain<ILP, OP><<<sms, warps * 32>>>(out, 100, 1.0000001, 1e-9);
  cudaEventRecord(e0);
  k_chain<ILP, OP><<<sms, warps * 32>>>(out, iters, 1.0000001, 1e-9);
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return (double)sms * warps * 32 * (double)iters * ILP / (ms * 1e-3);
}

// op: 0 DFMA, 1 DADD, 2 DMUL; ilp in {1, 2, 4, 8}; returns thread-instructions per second (0 on error)
extern "C" double fp64_chain_rate(int op, int ilp, int warps_per_sm, int iters) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* out = nullptr;
  if (cudaMalloc(&out, 8) != cudaSuccess) return 0;
  double r = 0;
#define CASE(I, O) if (ilp == I && op == O) r = run<I, O>(sms, warps_per_sm, iters, out);
  CASE(1, 0) CASE(2, 0) CASE(4, 0) CASE(8, 0) CASE(1, 1) CASE(2, 1) CASE(4, 1) CASE(8, 1)
  CASE(1, 2) CASE(2, 2) CASE(4, 2) CASE(8, 2)
#undef CASE
  cudaFree(out);
  return cudaGetLastError() == cudaSuccess ? r : 0;
}
