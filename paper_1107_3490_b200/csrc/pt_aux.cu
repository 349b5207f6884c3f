// Support kernels: state set-up, full energy (Eq. 4), replica exchange (Eq. 6), read-out gather.
#include <math.h>

#include "pt_device.cuh"

namespace {

// AoS fp64 conformations [C][N][3] (temperature order = slot order at init) -> SoA Real [C][3][Ng];
// identity labels; all statistics zero.
template <typename Real>
__global__ void k_scatter_init(const PtDev d, const double* __restrict__ src)
{
  const int s = blockIdx.x;
  Real* dst = reinterpret_cast<Real*>(d.coords) + (size_t)s * 3 * d.Ng;
  const double* a = src + (size_t)s * d.N * 3;
  for (int j = threadIdx.x; j < d.Ng; j += blockDim.x) {
    const bool in = j < d.N;
    dst[j] = in ? (Real)a[3 * j] : (Real)PT_FAR;
    dst[d.Ng + j] = in ? (Real)a[3 * j + 1] : (Real)PT_FAR;
    dst[2 * d.Ng + j] = in ? (Real)a[3 * j + 2] : (Real)PT_FAR;
  }
  if (threadIdx.x == 0) {
    d.temp_of_slot[s] = s % d.M;
    d.slot_of_temp[s] = s % d.M;
  }
}

__global__ void k_zero_stats(const PtDev d)
{
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const size_t nh = (size_t)d.C * (size_t)(d.nbins + 2);
  for (size_t q = tid; q < nh; q += stride) d.hist[q] = 0ull;
  for (size_t q = tid; q < (size_t)d.C * 3; q += stride) { d.mom[q] = 0.0; d.mcount[q] = 0ull; }
  for (size_t q = tid; q < (size_t)d.C * PT_NOBS; q += stride) d.obs[q] = 0.0;
  const size_t ns = (size_t)d.E * (size_t)(d.M > 1 ? d.M - 1 : 1) * 2;
  for (size_t q = tid; q < ns; q += stride) d.scount[q] = 0ull;
}

// Eq. (4): E(C) = 1/2 sum_{i != j} E_LJ^mod(r_ij) + sum_i E_FENE(r_{i,i+1}), one warp
// per chain, always accumulated in fp64 with IEEE division (this is init / invariant, not the loop).
template <typename Real>
__global__ void k_full_energy(const PtDev d, double* __restrict__ out)
{
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= d.C) return;
  const Real* x = reinterpret_cast<const Real*>(d.coords) + (size_t)warp * 3 * d.Ng;
  const Real* y = x + d.Ng;
  const Real* z = y + d.Ng;
  const int N = d.N;
  double acc = 0.0;
  for (int i = 0; i < N; ++i) {
    const double xi = (double)x[i], yi = (double)y[i], zi = (double)z[i];
    for (int j = i + 1 + lane; j < N; j += 32) {
      const double dx = xi - (double)x[j], dy = yi - (double)y[j], dz = zi - (double)z[j];
      const double r2 = dx * dx + dy * dy + dz * dz;
      if (r2 < d.rc2) {
        const double w = d.sigma2 / r2;
        const double s6 = w * w * w;
        acc += d.eps4 * (s6 * s6 - s6) - d.ljC;
      }
    }
  }
  for (int i = lane; i + 1 < N; i += 32) {
    const double dx = (double)x[i] - (double)x[i + 1], dy = (double)y[i] - (double)y[i + 1],
                 dz = (double)z[i] - (double)z[i + 1];
    const double r = sqrt(dx * dx + dy * dy + dz * dz);
    const double q = (r - d.r0) / d.R;
    const double g = 1.0 - q * q;
    acc += (q * q < 1.0) ? d.feneC * log(g) : __longlong_as_double(0x7ff0000000000000ll);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) out[warp] = acc;
}

// Section 3.3, Eq. (6): one thread per neighbour pair of this event's parity.
// The temperature labels of the two slots are swapped; coordinates stay where they are.
__global__ void k_exchange(const PtDev d, const uint32_t x)
{
  const int npairs = (d.M - (int)(x & 1u)) / 2;   // pairs (i, i+1), i = parity, parity+2, ..., i+1 <= M-1
  const int tid = blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= d.E * npairs) return;
  pt_exchange_pair(d, tid / npairs, (int)(x & 1u) + 2 * (tid % npairs), x);
}

// Read-out in temperature order: energies and AoS fp64 conformations.
template <typename Real>
__global__ void k_gather(const PtDev d, const double* __restrict__ slot_energy, double* __restrict__ out_e,
                         double* __restrict__ out_x)
{
  const int ti = blockIdx.x;
  const int e = ti / d.M, i = ti % d.M;
  const int s = e * d.M + d.slot_of_temp[ti];
  if (out_e && threadIdx.x == 0) out_e[ti] = slot_energy[s];
  if (out_x) {
    const Real* x = reinterpret_cast<const Real*>(d.coords) + (size_t)s * 3 * d.Ng;
    double* o = out_x + (size_t)ti * d.N * 3;
    for (int q = threadIdx.x; q < 3 * d.N; q += blockDim.x) {
      const int j = q / 3, a = q % 3;
      o[q] = (double)x[a * d.Ng + j];
    }
  }
  (void)i;
}

}  // namespace

cudaError_t pt_launch_scatter_init(const PtDev& d, int precision, const double* staging, cudaStream_t st)
{
  if (precision == PT_F32) k_scatter_init<float><<<d.C, 128, 0, st>>>(d, staging);
  else k_scatter_init<double><<<d.C, 128, 0, st>>>(d, staging);
  k_zero_stats<<<296, 256, 0, st>>>(d);
  return cudaGetLastError();
}

cudaError_t pt_launch_zero_stats(const PtDev& d, cudaStream_t st)
{
  k_zero_stats<<<296, 256, 0, st>>>(d);
  return cudaGetLastError();
}

cudaError_t pt_launch_full_energy(const PtDev& d, int precision, double* out, cudaStream_t st)
{
  const int threads = 128, wpb = threads / 32;
  const int grid = (d.C + wpb - 1) / wpb;
  if (precision == PT_F32) k_full_energy<float><<<grid, threads, 0, st>>>(d, out);
  else k_full_energy<double><<<grid, threads, 0, st>>>(d, out);
  return cudaGetLastError();
}

cudaError_t pt_launch_exchange(const PtDev& d, uint32_t x, cudaStream_t st)
{
  const int npairs = (d.M - (int)(x & 1u)) / 2;
  const int total = d.E * npairs;
  if (total <= 0) return cudaSuccess;
  k_exchange<<<(total + 127) / 128, 128, 0, st>>>(d, x);
  return cudaGetLastError();
}

cudaError_t pt_launch_gather(const PtDev& d, int precision, const double* slot_energy, double* out_e,
                             double* out_x, cudaStream_t st)
{
  if (precision == PT_F32) k_gather<float><<<d.C, 128, 0, st>>>(d, slot_energy, out_e, out_x);
  else k_gather<double><<<d.C, 128, 0, st>>>(d, slot_energy, out_e, out_x);
  return cudaGetLastError();
}
