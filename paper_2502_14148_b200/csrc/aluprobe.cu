// aluprobe.cu — ocn_alu_probe: register-resident FMA chains that MEASURE the denominator of the tendency kernels' roofline.
//
// The tendency kernels are bound by the FP64 (C0-C3) / FP32 (C4) pipe, and MEASURED_PEAKS.json holds no ALU peak
// (SURVEY 7 step 0, 8(d)).  bench.py times this probe with CUDA events and reports `roofline.peak` as measured:
//   mode 0  pure FMA: 8 independent chains per thread                     -> the pipe's issue peak
//   mode 1  one integer multiply-add per FMA, independent of the chains   -> do other pipes issue in the FMA's shadow?
//   mode 2  two integer multiply-adds per FMA
//   mode 3  one shared-memory load per FMA (immediate-offset LDS)
//   mode 4  pure add chains,   mode 5  pure multiply chains               -> is every FP64 opcode issued at the FMA rate?
//   mode 6  FMA with three distinct per-thread register operands (modes 0-5 take two operands from uniform registers)
//           -> does register-file bandwidth lower the rate of real code?   mode 7  the same with two register operands
// Every thread runs n_iter iterations of 32 FMAs (8 chains x 4); a warp instruction counts 2 flops per lane in modes
// 0-3, 1 in modes 4-5.  Results go to `sink` only if they are NaN (never), which keeps the chains alive.
#include <cstdint>

#include "ocn_internal.h"

namespace {

template <class Real> struct Fma;
template <> struct Fma<double> {
  static __device__ __forceinline__ void fma(double &a, double x, double y) { asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(a) : "d"(x), "d"(y)); }
  static __device__ __forceinline__ void add(double &a, double x) { asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(a) : "d"(x)); }
  static __device__ __forceinline__ void mul(double &a, double x) { asm volatile("mul.rn.f64 %0, %0, %1;" : "+d"(a) : "d"(x)); }
};
template <> struct Fma<float> {
  static __device__ __forceinline__ void fma(float &a, float x, float y) { asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(a) : "f"(x), "f"(y)); }
  static __device__ __forceinline__ void add(float &a, float x) { asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a) : "f"(x)); }
  static __device__ __forceinline__ void mul(float &a, float x) { asm volatile("mul.rn.f32 %0, %0, %1;" : "+f"(a) : "f"(x)); }
};
__device__ __forceinline__ void imad(unsigned &x, unsigned m, unsigned c) { asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x) : "r"(m), "r"(c)); }

template <class Real, int MODE>
__global__ void __launch_bounds__(1024, 1) alu_probe_kernel(int n_iter, Real x, Real y, Real *sink) {
  __shared__ Real sh[1024 + 64];
  sh[threadIdx.x] = Real(threadIdx.x) * Real(1e-9);
  if (threadIdx.x < 64) sh[1024 + threadIdx.x] = Real(0);
  __syncthreads();
  Real a[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) a[c] = Real(c + threadIdx.x) * Real(1e-3);
  Real b[8], d[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) { b[c] = Real(1) - Real(c + 1 + threadIdx.x) * Real(1e-9); d[c] = Real(c + 2 * threadIdx.x) * Real(1e-9); }
  unsigned iv[4] = {threadIdx.x, threadIdx.x + 1u, threadIdx.x + 2u, threadIdx.x + 3u};
  const unsigned mm = 1664525u + 2u * blockIdx.x, cc = 1013904223u;
  const Real *lp = sh + threadIdx.x;
  for (int it = 0; it < n_iter; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        if (MODE <= 3) Fma<Real>::fma(a[c], x, y);
        if (MODE == 6) Fma<Real>::fma(a[c], b[c], d[(c + 3) & 7]);
        if (MODE == 7) Fma<Real>::fma(a[c], b[c], y);
        if (MODE == 8 || MODE == 9 || MODE == 10 || MODE == 11) Fma<Real>::fma(a[c], b[c], y);      // 2 register operands
        if (MODE == 8) imad(iv[c & 3], mm, cc);                                                   // + IMAD (2 register operands)
        if (MODE == 9) asm volatile("add.u32 %0, %0, %1;" : "+r"(iv[c & 3]) : "r"(mm));         // + IADD (2 register operands)
        if (MODE == 10) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(iv[c & 3]) : "r"(mm), "r"(iv[(c + 1) & 3]));   // + LOP3 (3 regs)
        if (MODE == 11) {
          Real t;
          if (sizeof(Real) == 8) asm volatile("ld.shared.f64 %0, [%1];" : "=d"(*(double *)&t) : "r"((unsigned)__cvta_generic_to_shared(lp + ((r * 8 + c) & 63))));
          else asm volatile("ld.shared.f32 %0, [%1];" : "=f"(*(float *)&t) : "r"((unsigned)__cvta_generic_to_shared(lp + ((r * 8 + c) & 63))));
          (void)t;
        }
        if (MODE == 4) Fma<Real>::add(a[c], y);
        if (MODE == 5) Fma<Real>::mul(a[c], x);
        if (MODE == 1 || MODE == 2) imad(iv[c & 3], mm, cc);
        if (MODE == 2) imad(iv[(c + 2) & 3], mm, cc);
        if (MODE == 3) {
          Real t;
          if (sizeof(Real) == 8) asm volatile("ld.shared.f64 %0, [%1];" : "=d"(*(double *)&t) : "r"((unsigned)__cvta_generic_to_shared(lp + ((r * 8 + c) & 63))));
          else asm volatile("ld.shared.f32 %0, [%1];" : "=f"(*(float *)&t) : "r"((unsigned)__cvta_generic_to_shared(lp + ((r * 8 + c) & 63))));
          (void)t;   // volatile asm: the load is issued even though its value is dropped (an FP add per load would distort the count)
        }
      }
    }
  }
  Real s = Real(0);
#pragma unroll
  for (int c = 0; c < 8; ++c) s += a[c] + b[c] + d[c];
  s += Real(iv[0] ^ iv[1] ^ iv[2] ^ iv[3]) * Real(1e-30);
  if (s != s) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <class Real, int MODE>
int launch_probe(int blocks, int threads, int n_iter, void *sink, cudaStream_t s) {
  alu_probe_kernel<Real, MODE><<<blocks, threads, 0, s>>>(n_iter, Real(0.999999), Real(1e-7), (Real *)sink);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "alu_probe_kernel launch");
}

template <class Real>
int dispatch_probe(int mode, int blocks, int threads, int n_iter, void *sink, cudaStream_t s) {
  switch (mode) {
    case 0: return launch_probe<Real, 0>(blocks, threads, n_iter, sink, s);
    case 1: return launch_probe<Real, 1>(blocks, threads, n_iter, sink, s);
    case 2: return launch_probe<Real, 2>(blocks, threads, n_iter, sink, s);
    case 3: return launch_probe<Real, 3>(blocks, threads, n_iter, sink, s);
    case 4: return launch_probe<Real, 4>(blocks, threads, n_iter, sink, s);
    case 5: return launch_probe<Real, 5>(blocks, threads, n_iter, sink, s);
    case 6: return launch_probe<Real, 6>(blocks, threads, n_iter, sink, s);
    case 7: return launch_probe<Real, 7>(blocks, threads, n_iter, sink, s);
    case 8: return launch_probe<Real, 8>(blocks, threads, n_iter, sink, s);
    case 9: return launch_probe<Real, 9>(blocks, threads, n_iter, sink, s);
    case 10: return launch_probe<Real, 10>(blocks, threads, n_iter, sink, s);
    default: return launch_probe<Real, 11>(blocks, threads, n_iter, sink, s);
  }
}

}  // namespace

extern "C" int ocn_alu_probe(int dtype, int mode, int blocks, int threads_per_block, int n_iter, void *sink, double *flops_out,
                             void *stream) {
  if (dtype != OCN_F64 && dtype != OCN_F32) return ocn_fail(OCN_ERR_INVALID, "ocn_alu_probe: dtype must be OCN_F64 or OCN_F32");
  if (mode < 0 || mode > 11) return ocn_fail(OCN_ERR_INVALID, "ocn_alu_probe: mode must be 0..11");
  if (blocks < 1 || threads_per_block < 32 || threads_per_block > 1024 || threads_per_block % 32 || n_iter < 1)
    return ocn_fail(OCN_ERR_INVALID, "ocn_alu_probe: need blocks >= 1, threads_per_block a multiple of 32 in [32, 1024], n_iter >= 1");
  if (!sink) return ocn_fail(OCN_ERR_INVALID, "ocn_alu_probe: sink is NULL");
  if (flops_out) *flops_out = (mode <= 3 || mode >= 6 ? 2.0 : 1.0) * 32.0 * (double)n_iter * (double)blocks * (double)threads_per_block;
  cudaStream_t s = (cudaStream_t)stream;
  return dtype == OCN_F64 ? dispatch_probe<double>(mode, blocks, threads_per_block, n_iter, sink, s)
                          : dispatch_probe<float>(mode, blocks, threads_per_block, n_iter, sink, s);
}
