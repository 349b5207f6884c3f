// pt_energy_noalloc: Eq. (4) for a batch of conformations WITHOUT any allocation -- for callers that
// cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// It is a variant of k_full_energy (pt_aux.cu; the existing path is pt_recompute_energy, whose scratch e_full / e_by_temp
// lives in the handle's cudaMalloc'ed workspace): every chain's pair sum is split over PT_NOALLOC_PARTS CTAs, their
// partial sums and a per-chain arrival counter are scratch, and the last CTA of a chain to finish adds the partials in a
// fixed order.  The scratch is the file-scope array below: every GPU that loads the library holds its 576 KiB until
// the process exits; it bounds the batch at PT_NOALLOC_MAX_CHAINS chains per call.
//
// The array's NAME is a host-side stand-in in host code, not a device address: the address is asked for once per
// device, with that device current (cudaGetSymbolAddress), and passed to the kernel.
// All calls share the array and it keeps the last call's contents: the arrival counters are cleared at the start of
// every call (cudaMemsetAsync on the caller's stream: no allocation), the partial sums are all written before they are
// read.  Two calls that overlap on the GPU (different streams, or different host threads) race on it: serialise them.
#include <math.h>
#include <stdint.h>

#include <mutex>
#include <string>

#include <cuda_runtime.h>

#include "pt_b200.h"

#define PT_NOALLOC_PARTS 8
#define PT_NOALLOC_PARTIALS ((size_t)PT_NOALLOC_MAX_CHAINS * PT_NOALLOC_PARTS)

namespace {

// [PT_NOALLOC_MAX_CHAINS][PARTS] partial sums, then PT_NOALLOC_MAX_CHAINS arrival counters (one per 8-byte word)
static __device__ __align__(256) double pt_noalloc_scratch[PT_NOALLOC_PARTIALS + PT_NOALLOC_MAX_CHAINS];

struct NaModel {
  int N;
  double sigma2, eps4, ljC, rc2, r0, R, feneC;
};

// CTA `part` of chain `chain`: rows i = part, part + PARTS, ... of the pair sum (lanes stride over j > i, warps over
// the rows), part 0 also the bonds; same arithmetic per term as k_full_energy (IEEE division, sqrt, log).
__global__ void __launch_bounds__(128) k_energy_noalloc(const NaModel m, const double* __restrict__ x, double* __restrict__ out,
                                                         double* __restrict__ partial, unsigned long long* __restrict__ count)
{
  __shared__ double s_w[4];
  __shared__ int s_last;
  const int chain = blockIdx.x / PT_NOALLOC_PARTS, part = blockIdx.x % PT_NOALLOC_PARTS;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int N = m.N;
  const double* c = x + (size_t)chain * 3 * N;   // AoS: x_j = c[3 j], y_j = c[3 j + 1], z_j = c[3 j + 2]
  double acc = 0.0;
  for (int i = part + PT_NOALLOC_PARTS * warp; i < N; i += PT_NOALLOC_PARTS * 4) {
    const double xi = c[3 * i], yi = c[3 * i + 1], zi = c[3 * i + 2];
    for (int j = i + 1 + lane; j < N; j += 32) {
      const double dx = xi - c[3 * j], dy = yi - c[3 * j + 1], dz = zi - c[3 * j + 2];
      const double r2 = dx * dx + dy * dy + dz * dz;
      if (r2 < m.rc2) {
        const double w = m.sigma2 / r2;
        const double s6 = w * w * w;
        acc += m.eps4 * (s6 * s6 - s6) - m.ljC;
      }
    }
  }
  if (part == 0) {
    for (int i = threadIdx.x; i + 1 < N; i += 128) {
      const double dx = c[3 * i] - c[3 * i + 3], dy = c[3 * i + 1] - c[3 * i + 4], dz = c[3 * i + 2] - c[3 * i + 5];
      const double r = sqrt(dx * dx + dy * dy + dz * dz);
      const double q = (r - m.r0) / m.R;
      const double g = 1.0 - q * q;
      acc += (q * q < 1.0) ? m.feneC * log(g) : __longlong_as_double(0x7ff0000000000000ll);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) s_w[warp] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    partial[(size_t)chain * PT_NOALLOC_PARTS + part] = (s_w[0] + s_w[1]) + (s_w[2] + s_w[3]);
    __threadfence();
    s_last = atomicAdd(&count[chain], 1ull) == (unsigned long long)(PT_NOALLOC_PARTS - 1);
  }
  __syncthreads();
  if (s_last && threadIdx.x == 0) {
    __threadfence();
    const volatile double* p = partial + (size_t)chain * PT_NOALLOC_PARTS;
    double e = 0.0;
    for (int q = 0; q < PT_NOALLOC_PARTS; ++q) e += p[q];   // fixed order: the result does not depend on who is last
    out[chain] = e;
  }
}

thread_local std::string g_err;

int fail(int code, const std::string& msg)
{
  g_err = msg;
  return code;
}

// device address of the scratch array, asked for once per device
constexpr int kMaxDevices = 64;
std::mutex g_mu;
double* g_scratch_of_device[kMaxDevices] = {};

}  // namespace

extern "C" {

int pt_energy_noalloc(const pt_params* p, const double* dev_conformations, double* dev_energies, int64_t n_chains,
                      void* stream)
{
  if (!p) return fail(PT_EINVAL, "params is NULL");
  if (p->N < 2) return fail(PT_EINVAL, "N must be >= 2");
  if (!(p->eps > 0.0) || !isfinite(p->eps) || !(p->r0 > 0.0) || !isfinite(p->r0) || !(p->R > 0.0) || !isfinite(p->R) ||
      !(p->K > 0.0) || !isfinite(p->K) || !(p->rc_over_sigma > 0.0) || !isfinite(p->rc_over_sigma))
    return fail(PT_EINVAL, "eps, r0, R, K and rc_over_sigma must be finite and > 0");
  if (n_chains < 0) return fail(PT_EINVAL, "n_chains must be >= 0");
  if (n_chains > PT_NOALLOC_MAX_CHAINS)
    return fail(PT_EINVAL, "pt_energy_noalloc: n_chains = " + std::to_string(n_chains) + " exceeds PT_NOALLOC_MAX_CHAINS = " +
                               std::to_string(PT_NOALLOC_MAX_CHAINS) + " (the static scratch array); split the batch");
  if (n_chains == 0) return PT_OK;
  if (!dev_conformations || !dev_energies) return fail(PT_EINVAL, "dev_conformations / dev_energies is NULL");

  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(PT_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices) return fail(PT_EINVAL, "device ordinal beyond 63");
  double* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_of_device[dev]) {
      // with device `dev` current: the symbol has one instance per device
      void* ptr = nullptr;
      e = cudaGetSymbolAddress(&ptr, pt_noalloc_scratch);
      if (e != cudaSuccess) return fail(PT_ECUDA, std::string("cudaGetSymbolAddress(pt_noalloc_scratch): ") + cudaGetErrorString(e));
      g_scratch_of_device[dev] = static_cast<double*>(ptr);
    }
    scratch = g_scratch_of_device[dev];
  }

  // model constants as pt_create derives them (sigma = 2^(-1/6) r0, r_c = rc_over_sigma sigma)
  NaModel m;
  const double sigma = p->r0 / pow(2.0, 1.0 / 6.0);
  const double rc = p->rc_over_sigma * sigma;
  m.N = p->N;
  m.sigma2 = sigma * sigma;
  const double wc = m.sigma2 / (rc * rc), s6c = wc * wc * wc;
  m.eps4 = 4.0 * p->eps;
  m.ljC = 4.0 * p->eps * (s6c * s6c - s6c);
  m.rc2 = rc * rc;
  m.r0 = p->r0;
  m.R = p->R;
  m.feneC = -0.5 * p->K * p->R * p->R;

  cudaStream_t st = static_cast<cudaStream_t>(stream);
  unsigned long long* count = reinterpret_cast<unsigned long long*>(scratch + PT_NOALLOC_PARTIALS);
  // the counters must start at zero whatever the last call left (an aborted launch, another batch size)
  e = cudaMemsetAsync(count, 0, (size_t)n_chains * sizeof(unsigned long long), st);
  if (e != cudaSuccess) return fail(PT_ECUDA, std::string("cudaMemsetAsync(counters): ") + cudaGetErrorString(e));
  k_energy_noalloc<<<(unsigned)(n_chains * PT_NOALLOC_PARTS), 128, 0, st>>>(m, dev_conformations, dev_energies, scratch, count);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(PT_ECUDA, std::string("k_energy_noalloc: ") + cudaGetErrorString(e));
  return PT_OK;
}

const char* pt_noalloc_last_error(void) { return g_err.c_str(); }

}  // extern "C"
