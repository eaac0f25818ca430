// aluprobe.cu — ocn_alu_probe: register-resident FMA chains that MEASURE the denominator of the tendency kernels' roofline.
//
// The tendency kernels are bound by the FP64 (C0-C3) / FP32 (C4) pipe, and MEASURED_PEAKS.json holds no ALU peak
// (SURVEY 7 step 0, 8(d)).  bench.py times this probe with CUDA events and reports `roofline.peak` as measured: every thread runs
// n_iter iterations of 32 FMAs (8 independent chains x 4, both multiplicands in uniform registers); a warp instruction counts
// 2 flops per lane.  Results go to `sink` only if they are NaN (never), which keeps the chains alive.
// (Round 2 also carried exploration modes — integer / LDS instructions issued beside the FMAs, add- and multiply-only chains,
// register-operand variants; their table is kept in profiles/r2_alu_probe.md, the code left the product library in round 3.)
#include <cstdint>

#include "ocn_internal.h"

namespace {

__device__ __forceinline__ void fma_chain(double &a, double x, double y) { asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(a) : "d"(x), "d"(y)); }
__device__ __forceinline__ void fma_chain(float &a, float x, float y) { asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(a) : "f"(x), "f"(y)); }

template <class Real>
__global__ void __launch_bounds__(1024, 1) alu_probe_kernel(int n_iter, Real x, Real y, Real *sink) {
  Real a[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) a[c] = Real(c + threadIdx.x) * Real(1e-3);
  for (int it = 0; it < n_iter; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int c = 0; c < 8; ++c) fma_chain(a[c], x, y);
    }
  }
  Real s = Real(0);
#pragma unroll
  for (int c = 0; c < 8; ++c) s += a[c];
  if (s != s) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <class Real>
int launch_probe(int blocks, int threads, int n_iter, void *sink, cudaStream_t s) {
  alu_probe_kernel<Real><<<blocks, threads, 0, s>>>(n_iter, Real(0.999999), Real(1e-7), (Real *)sink);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "alu_probe_kernel launch");
}

}  // namespace

extern "C" int ocn_alu_probe(int dtype, int mode, int blocks, int threads_per_block, int n_iter, void *sink, double *flops_out,
                             void *stream) {
  if (dtype != OCN_F64 && dtype != OCN_F32) return ocn_fail(OCN_ERR_INVALID, "ocn_alu_probe: dtype must be OCN_F64 or OCN_F32");
  if (mode != 0) return ocn_fail(OCN_ERR_INVALID, "ocn_alu_probe: mode must be 0 (pure FMA chains; the exploration modes of round 2 are no longer part of the library)");
  if (blocks < 1 || threads_per_block < 32 || threads_per_block > 1024 || threads_per_block % 32 || n_iter < 1)
    return ocn_fail(OCN_ERR_INVALID, "ocn_alu_probe: need blocks >= 1, threads_per_block a multiple of 32 in [32, 1024], n_iter >= 1");
  if (!sink) return ocn_fail(OCN_ERR_INVALID, "ocn_alu_probe: sink is NULL");
  if (flops_out) *flops_out = 2.0 * 32.0 * (double)n_iter * (double)blocks * (double)threads_per_block;
  cudaStream_t s = (cudaStream_t)stream;
  return dtype == OCN_F64 ? launch_probe<double>(blocks, threads_per_block, n_iter, sink, s)
                          : launch_probe<float>(blocks, threads_per_block, n_iter, sink, s);
}
