// Measures the chip's plain (non-tensor) FMA rate: the denominator of the "alu" roofline that the
// sweep kernel is reported against (MEASURED_PEAKS.json holds HBM and bf16 tensor figures only).
// Eight independent FMA chains per thread, 1024 threads per CTA, two CTAs per SM: every fp64
// (fp32) lane of every SM sub-partition has an instruction to issue every cycle.
#include <cuda_runtime.h>

#include "pt_b200.h"

namespace {

template <typename Real>
__global__ void __launch_bounds__(1024, 2) k_fma_chain(Real* out, const Real a, const Real b, const int iters)
{
  Real v0 = (Real)threadIdx.x, v1 = v0 + 1, v2 = v0 + 2, v3 = v0 + 3, v4 = v0 + 4, v5 = v0 + 5, v6 = v0 + 6,
       v7 = v0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      v0 = fma(v0, a, b); v1 = fma(v1, a, b); v2 = fma(v2, a, b); v3 = fma(v3, a, b);
      v4 = fma(v4, a, b); v5 = fma(v5, a, b); v6 = fma(v6, a, b); v7 = fma(v7, a, b);
    }
  }
  const Real s = ((v0 + v1) + (v2 + v3)) + ((v4 + v5) + (v6 + v7));
  if (s == (Real)123.456) out[0] = s;   // never true for the a, b used; keeps the chains alive
}

template <typename Real> cudaError_t measure(int iters, int reps, cudaStream_t st, double* tflops)
{
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  Real* out = nullptr;
  e = cudaMalloc(&out, sizeof(Real));
  if (e != cudaSuccess) return e;
  cudaEvent_t t0, t1;
  cudaEventCreate(&t0);
  cudaEventCreate(&t1);
  const int grid = 2 * sms;
  const Real a = (Real)0.999999, b = (Real)1e-6;
  k_fma_chain<Real><<<grid, 1024, 0, st>>>(out, a, b, iters / 8 + 1);   // warm-up
  double best = 0.0;
  for (int r = 0; r < reps && e == cudaSuccess; ++r) {
    cudaEventRecord(t0, st);
    k_fma_chain<Real><<<grid, 1024, 0, st>>>(out, a, b, iters);
    cudaEventRecord(t1, st);
    e = cudaEventSynchronize(t1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
    const double flops = 2.0 * 64.0 * (double)iters * 1024.0 * (double)grid;
    if (e == cudaSuccess && ms > 0.f && flops / (ms * 1e-3) * 1e-12 > best) best = flops / (ms * 1e-3) * 1e-12;
  }
  cudaEventDestroy(t0);
  cudaEventDestroy(t1);
  cudaFree(out);
  if (e == cudaSuccess) e = cudaGetLastError();
  *tflops = best;
  return e;
}

}  // namespace

extern "C" int pt_fma_peak(int precision, int iters, int reps, void* cuda_stream, double* tflops)
{
  if (!tflops || iters < 1 || reps < 1 || (precision != PT_F64 && precision != PT_F32)) return PT_EINVAL;
  *tflops = 0.0;
  const cudaError_t e = precision == PT_F32 ? measure<float>(iters, reps, (cudaStream_t)cuda_stream, tflops)
                                            : measure<double>(iters, reps, (cudaStream_t)cuda_stream, tflops);
  return e == cudaSuccess ? PT_OK : PT_ECUDA;
}
