// Metropolis sweep kernels for sm_100a.
//
// One chain's coordinates stay in shared memory for the whole launch (SoA x[], y[], z[]).
// Inside a chain the Markov chain is strictly serial; the parallelism is
//   (i)  over partner monomers j of the moved monomer m: L lanes stride over j and each adds
//        E_LJ^mod(|x' - x_j|) - E_LJ^mod(|x_m - x_j|) for its partners (Eq. 1, 2, 5), and
//   (ii) over chains: 32/L chains per warp, so that the serial part of a step (Philox, the FENE
//        sqrt/log, the Metropolis exp) is one instruction stream shared by 32/L chains.
// The paper's kernel (Listing 2) maps one replica to one block of 64 threads and
// recomputes the whole energy; that is prior art, kept only as the CTA-per-replica variant for
// long chains, and with the local Delta-E of Eq. (5) instead of the full sum.
#include <math.h>

#include "pt_device.cuh"

namespace {

template <typename Real> struct Fene;
template <> struct Fene<double> {
  // Eq. (3): -(K/2) R^2 log[1 - ((r - r0)/R)^2]; +inf outside (r0-R, r0+R)
  static __device__ __forceinline__ double eval(const PtDev& d, double r2, bool* inside)
  {
    const double r = sqrt(r2);
    const double q = (r - d.r0) * d.invR;
    const double g = fma(-q, q, 1.0);
    *inside = (g > 0.0);
    return *inside ? d.feneC * log(g) : __longlong_as_double(0x7ff0000000000000ll);
  }
  static __device__ __forceinline__ bool metropolis(double u, double beta, double dE)
  {
    return u < exp(-beta * dE);
  }
};
template <> struct Fene<float> {
  static __device__ __forceinline__ float eval(const PtDev& d, float r2, bool* inside)
  {
    const float r = sqrtf(r2);
    const float q = (r - (float)d.r0) * (float)d.invR;
    const float g = fmaf(-q, q, 1.0f);
    *inside = (g > 0.0f);
    return *inside ? (float)d.feneC * logf(g) : __int_as_float(0x7f800000);
  }
  static __device__ __forceinline__ bool metropolis(float u, double beta, float dE)
  {
    return u < expf(-(float)beta * dE);
  }
};

template <typename Real, int L> __device__ __forceinline__ Real group_sum(Real v)
{
#pragma unroll
  for (int o = L / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Everything a chain carries through a launch besides its coordinates.
struct ChainCtx {
  int s, e, i, ti;
  bool active;
  double beta;
  uint2 key;
  double erun, mom1, mom2;
  double ob0, ob1, ob2, ob3;
  unsigned acc, brej;
};

__device__ __forceinline__ void ctx_load(const PtDev& d, int s, ChainCtx& c)
{
  c.active = s < d.C;
  c.s = c.active ? s : d.C - 1;
  c.e = c.s / d.M;
  c.i = d.temp_of_slot[c.s];
  c.ti = c.e * d.M + c.i;
  c.beta = d.beta[c.i];
  c.key = d.keys[c.e];
  c.erun = d.erun[c.s];
  c.mom1 = d.mom[3 * c.ti + 1];
  c.mom2 = d.mom[3 * c.ti + 2];
  c.ob0 = d.obs[4 * c.ti + 0];
  c.ob1 = d.obs[4 * c.ti + 1];
  c.ob2 = d.obs[4 * c.ti + 2];
  c.ob3 = d.obs[4 * c.ti + 3];
  c.acc = 0;
  c.brej = 0;
}

// once per sweep, by one thread of the chain (A8): histogram, moments, energy trace
__device__ __forceinline__ void measure_energy(const PtDev& d, ChainCtx& c, uint32_t t)
{
  const double E = c.erun;
  if (d.nbins > 0) {
    const double b = floor((E - d.hist_emin) * d.hist_scale);
    int idx;
    if (b >= 0.0 && b < (double)d.nbins) idx = (int)b;
    else if (b < 0.0) idx = d.nbins;       // underflow
    else idx = d.nbins + 1;                // overflow (and NaN)
    atomicAdd(d.hist + (size_t)c.ti * (size_t)(d.nbins + 2) + idx, 1ull);
  }
  c.mom1 = __dadd_rn(c.mom1, E);
  c.mom2 = __dadd_rn(c.mom2, __dmul_rn(E, E));
  if (d.tr_e && (long long)t < d.cap_sweeps) d.tr_e[(size_t)c.ti * d.cap_sweeps + t] = E;
}

__device__ __forceinline__ void ctx_store(const PtDev& d, const ChainCtx& c, int n_sweeps)
{
  d.erun[c.s] = c.erun;
  d.mom[3 * c.ti + 0] += (double)n_sweeps;
  d.mom[3 * c.ti + 1] = c.mom1;
  d.mom[3 * c.ti + 2] = c.mom2;
  if (d.observables) {
    d.obs[4 * c.ti + 0] = c.ob0;
    d.obs[4 * c.ti + 1] = c.ob1;
    d.obs[4 * c.ti + 2] = c.ob2;
    d.obs[4 * c.ti + 3] = c.ob3;
  }
  d.mcount[3 * c.ti + 0] += (unsigned long long)n_sweeps * (unsigned long long)d.N;
  d.mcount[3 * c.ti + 1] += c.acc;
  d.mcount[3 * c.ti + 2] += c.brej;
}

// ------------------------------------------------------------------------------------------
// Warp-group kernel: L lanes per chain, 32/L chains per warp.
// ------------------------------------------------------------------------------------------
template <typename Real, int L>
__global__ void __launch_bounds__(128) k_sweep_group(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                     const int n_sweeps)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int G = 32 / L;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane / L, lig = lane % L;
  const int cl = warp * G + g;
  const int N = d.N, Ns = pl.Ns;
  const Real FAR = (Real)PT_FAR;

  ChainCtx c;
  ctx_load(d, blockIdx.x * pl.chains_per_cta + cl, c);
  const Real width = (Real)d.width[c.i];
  const PtLJ<Real> lj(d);

  Real* xs = reinterpret_cast<Real*>(smem_raw) + (size_t)cl * pl.sstride;
  Real* ys = xs + Ns;
  Real* zs = ys + Ns;

  // A1: HBM -> shared memory, padding entries far away
  Real* gx = reinterpret_cast<Real*>(d.coords) + (size_t)c.s * 3 * d.Ng;
  for (int j = lig; j < Ns; j += L) {
    const bool in = j < N;
    xs[j] = in ? gx[j] : FAR;
    ys[j] = in ? gx[d.Ng + j] : FAR;
    zs[j] = in ? gx[2 * d.Ng + j] : FAR;
  }
  __syncwarp();

  const bool pick = d.select_mode == PT_RANDOM_PICK;
  const bool leader = (lig == 0) && c.active;
  const unsigned bond_lanes = 3u << (g * L);   // lanes 0,1 of the group: the new bonds

  for (int sw = 0; sw < n_sweeps; ++sw) {
    const uint32_t t = t0 + (uint32_t)sw;
    for (int k = 0; k < N; ++k) {
      // A2: proposal
      int m = k;
      if (pick) {
        const uint4 wp = pt_draw(c.key, (uint32_t)k, t, (uint32_t)c.e, PT_TAG_PICK, (uint32_t)c.i);
        m = (int)__umulhi(wp.x, (uint32_t)N);
      }
      const uint4 w = pt_draw(c.key, (uint32_t)k, t, (uint32_t)c.e, PT_TAG_MOVE, (uint32_t)c.i);
      const Real xo = xs[m], yo = ys[m], zo = zs[m];
      const Real xn = PtNum<Real>::propose(xo, width, PtNum<Real>::sym(w.x));
      const Real yn = PtNum<Real>::propose(yo, width, PtNum<Real>::sym(w.y));
      const Real zn = PtNum<Real>::propose(zo, width, PtNum<Real>::sym(w.z));
      const Real u = PtNum<Real>::u01(w.w);
      __syncwarp();
      // hide monomer m from its own sum: its slot looks like a padding entry during the loop
      if (lig == 0) { xs[m] = FAR; ys[m] = FAR; zs[m] = FAR; }
      __syncwarp();

      // A3: Delta E_LJ, lanes stride over partners (Eq. 1, 2)
      Real en = (Real)0, eo = (Real)0;
#pragma unroll 2
      for (int j = lig; j < Ns; j += L) {
        const Real xj = xs[j], yj = ys[j], zj = zs[j];
        const Real ax = xn - xj, ay = yn - yj, az = zn - zj;
        const Real bx = xo - xj, by = yo - yj, bz = zo - zj;
        const Real r2n = fma(az, az, fma(ay, ay, ax * ax));
        const Real r2o = fma(bz, bz, fma(by, by, bx * bx));
        const Real tn = lj.inside(r2n);
        const Real to = lj.inside(r2o);
        if (r2n < lj.rc2) en += tn;
        if (r2o < lj.rc2) eo += to;
      }
      Real part = en - eo;

      // A5: the <= 2 bonds of m, new and old, one bond per lane (Eq. 3)
      bool broke = false;
      if (lig < 4) {
        const int nb = (lig & 1) ? m + 1 : m - 1;
        if (nb >= 0 && nb < N) {
          const bool isnew = lig < 2;
          const Real dx = (isnew ? xn : xo) - xs[nb];
          const Real dy = (isnew ? yn : yo) - ys[nb];
          const Real dz = (isnew ? zn : zo) - zs[nb];
          bool inside;
          const Real f = Fene<Real>::eval(d, fma(dz, dz, fma(dy, dy, dx * dx)), &inside);
          if (isnew) { part += f; broke = !inside; }
          else part -= f;
        }
      }
      const bool bond_broken = (__ballot_sync(0xffffffffu, broke) & bond_lanes) != 0u;

      // A4: reduce; every lane of the group gets the same Delta E
      const Real dE = group_sum<Real, L>(part);

      // A6: Metropolis, Eq. (5)
      bool accept;
      if (bond_broken) accept = false;
      else if (dE <= (Real)0) accept = true;
      else accept = Fene<Real>::metropolis(u, c.beta, dE);   // NaN compares false: reject

      // A7: commit (or restore)
      if (lig == 0) {
        xs[m] = accept ? xn : xo;
        ys[m] = accept ? yn : yo;
        zs[m] = accept ? zn : zo;
        if (d.tr_move && c.active && (long long)t < d.cap_sweeps)
          d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
      }
      if (accept) { c.erun += (double)dE; c.acc++; }
      c.brej += bond_broken ? 1u : 0u;
      __syncwarp();
    }

    // A8: measurement once per sweep
    if (d.observables) {
      // Eq. (8): r_gyr^2 = (1/N) sum_k (r_k - r_mean)^2; R_ee^2 = |r_N - r_1|^2
      double sx = 0.0, sy = 0.0, sz = 0.0;
      for (int j = lig; j < N; j += L) { sx += (double)xs[j]; sy += (double)ys[j]; sz += (double)zs[j]; }
      sx = group_sum<double, L>(sx) / (double)N;
      sy = group_sum<double, L>(sy) / (double)N;
      sz = group_sum<double, L>(sz) / (double)N;
      double q = 0.0;
      for (int j = lig; j < N; j += L) {
        const double dx = (double)xs[j] - sx, dy = (double)ys[j] - sy, dz = (double)zs[j] - sz;
        q += dx * dx + dy * dy + dz * dz;
      }
      const double rg2 = group_sum<double, L>(q) / (double)N;
      const double ex = (double)xs[N - 1] - (double)xs[0], ey = (double)ys[N - 1] - (double)ys[0],
                   ez = (double)zs[N - 1] - (double)zs[0];
      const double ree2 = ex * ex + ey * ey + ez * ez;
      c.ob0 += ree2; c.ob1 += rg2; c.ob2 += rg2 * rg2; c.ob3 += ree2 * ree2;
    }
    if (leader) measure_energy(d, c, t);
  }

  // A9: shared memory -> HBM
  __syncwarp();
  if (c.active) {
    for (int j = lig; j < N; j += L) { gx[j] = xs[j]; gx[d.Ng + j] = ys[j]; gx[2 * d.Ng + j] = zs[j]; }
    if (lig == 0) ctx_store(d, c, n_sweeps);
  }
}

// ------------------------------------------------------------------------------------------
// CTA-per-replica kernel: blockDim.x threads share one chain (long chains, few replicas).
// ------------------------------------------------------------------------------------------
template <typename Real>
__global__ void __launch_bounds__(256) k_sweep_cta(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                   const int n_sweeps)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[2][8];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int T = blockDim.x, NW = T >> 5;
  const int N = d.N, Ns = pl.Ns;
  const Real FAR = (Real)PT_FAR;

  ChainCtx c;
  ctx_load(d, blockIdx.x, c);
  const Real width = (Real)d.width[c.i];
  const PtLJ<Real> lj(d);

  Real* xs = reinterpret_cast<Real*>(smem_raw);
  Real* ys = xs + Ns;
  Real* zs = ys + Ns;
  Real* gx = reinterpret_cast<Real*>(d.coords) + (size_t)c.s * 3 * d.Ng;
  for (int j = tid; j < Ns; j += T) {
    const bool in = j < N;
    xs[j] = in ? gx[j] : FAR;
    ys[j] = in ? gx[d.Ng + j] : FAR;
    zs[j] = in ? gx[2 * d.Ng + j] : FAR;
  }
  __syncthreads();

  const bool pick = d.select_mode == PT_RANDOM_PICK;
  for (int sw = 0; sw < n_sweeps; ++sw) {
    const uint32_t t = t0 + (uint32_t)sw;
    for (int k = 0; k < N; ++k) {
      int m = k;
      if (pick) {
        const uint4 wp = pt_draw(c.key, (uint32_t)k, t, (uint32_t)c.e, PT_TAG_PICK, (uint32_t)c.i);
        m = (int)__umulhi(wp.x, (uint32_t)N);
      }
      const uint4 w = pt_draw(c.key, (uint32_t)k, t, (uint32_t)c.e, PT_TAG_MOVE, (uint32_t)c.i);
      const Real xo = xs[m], yo = ys[m], zo = zs[m];
      const Real xn = PtNum<Real>::propose(xo, width, PtNum<Real>::sym(w.x));
      const Real yn = PtNum<Real>::propose(yo, width, PtNum<Real>::sym(w.y));
      const Real zn = PtNum<Real>::propose(zo, width, PtNum<Real>::sym(w.z));
      const Real u = PtNum<Real>::u01(w.w);

      Real en = (Real)0, eo = (Real)0;
#pragma unroll 2
      for (int j = tid; j < Ns; j += T) {
        const Real xj = xs[j], yj = ys[j], zj = zs[j];
        const Real ax = xn - xj, ay = yn - yj, az = zn - zj;
        const Real bx = xo - xj, by = yo - yj, bz = zo - zj;
        const Real r2n = fma(az, az, fma(ay, ay, ax * ax));
        const Real r2o = fma(bz, bz, fma(by, by, bx * bx));
        const Real tn = lj.inside(r2n);
        const Real to = lj.inside(r2o);
        const bool other = j != m;
        if (other && r2n < lj.rc2) en += tn;
        if (other && r2o < lj.rc2) eo += to;
      }
      Real part = en - eo;
      bool broke = false;
      if (tid < 4) {
        const int nb = (tid & 1) ? m + 1 : m - 1;
        if (nb >= 0 && nb < N) {
          const bool isnew = tid < 2;
          const Real dx = (isnew ? xn : xo) - xs[nb];
          const Real dy = (isnew ? yn : yo) - ys[nb];
          const Real dz = (isnew ? zn : zo) - zs[nb];
          bool inside;
          const Real f = Fene<Real>::eval(d, fma(dz, dz, fma(dy, dy, dx * dx)), &inside);
          if (isnew) { part += f; broke = !inside; }
          else part -= f;
        }
      }
      const Real wsum = group_sum<Real, 32>(part);
      if (lane == 0) red[k & 1][warp] = (double)wsum;
      const bool bond_broken = __syncthreads_or(broke ? 1 : 0) != 0;
      double dEd = red[k & 1][0];
      for (int q = 1; q < NW; ++q) dEd += red[k & 1][q];
      const Real dE = (Real)dEd;

      bool accept;
      if (bond_broken) accept = false;
      else if (dE <= (Real)0) accept = true;
      else accept = Fene<Real>::metropolis(u, c.beta, dE);

      if (tid == 0) {
        if (accept) { xs[m] = xn; ys[m] = yn; zs[m] = zn; }
        if (d.tr_move && (long long)t < d.cap_sweeps)
          d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
      }
      if (accept) { c.erun += (double)dE; c.acc++; }
      c.brej += bond_broken ? 1u : 0u;
      __syncthreads();
    }

    if (d.observables && warp == 0) {
      double sx = 0.0, sy = 0.0, sz = 0.0;
      for (int j = lane; j < N; j += 32) { sx += (double)xs[j]; sy += (double)ys[j]; sz += (double)zs[j]; }
      sx = group_sum<double, 32>(sx) / (double)N;
      sy = group_sum<double, 32>(sy) / (double)N;
      sz = group_sum<double, 32>(sz) / (double)N;
      double q = 0.0;
      for (int j = lane; j < N; j += 32) {
        const double dx = (double)xs[j] - sx, dy = (double)ys[j] - sy, dz = (double)zs[j] - sz;
        q += dx * dx + dy * dy + dz * dz;
      }
      const double rg2 = group_sum<double, 32>(q) / (double)N;
      const double ex = (double)xs[N - 1] - (double)xs[0], ey = (double)ys[N - 1] - (double)ys[0],
                   ez = (double)zs[N - 1] - (double)zs[0];
      const double ree2 = ex * ex + ey * ey + ez * ez;
      c.ob0 += ree2; c.ob1 += rg2; c.ob2 += rg2 * rg2; c.ob3 += ree2 * ree2;
    }
    if (tid == 0) measure_energy(d, c, t);
  }

  __syncthreads();
  for (int j = tid; j < N; j += T) { gx[j] = xs[j]; gx[d.Ng + j] = ys[j]; gx[2 * d.Ng + j] = zs[j]; }
  if (tid == 0) ctx_store(d, c, n_sweeps);
}

int round_up(int a, int b) { return (a + b - 1) / b * b; }

template <typename Real> cudaError_t launch_t(const PtDev& d, const PtLaunch& pl, uint32_t t0, int n,
                                              cudaStream_t st)
{
  const dim3 grid(pl.grid), block(pl.threads);
  switch (pl.lanes) {
    case 4: k_sweep_group<Real, 4><<<grid, block, pl.smem_bytes, st>>>(d, pl, t0, n); break;
    case 8: k_sweep_group<Real, 8><<<grid, block, pl.smem_bytes, st>>>(d, pl, t0, n); break;
    case 16: k_sweep_group<Real, 16><<<grid, block, pl.smem_bytes, st>>>(d, pl, t0, n); break;
    case 32: k_sweep_group<Real, 32><<<grid, block, pl.smem_bytes, st>>>(d, pl, t0, n); break;
    default: k_sweep_cta<Real><<<grid, block, pl.smem_bytes, st>>>(d, pl, t0, n); break;
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t pt_plan_sweep(const PtDev& d, int precision, int lanes_requested, PtLaunch* plan)
{
  const int real_bytes = precision == PT_F32 ? 4 : 8;
  int L = lanes_requested;
  if (L == 0) {
    // Few long chains: one CTA per replica.  Otherwise as few lanes per chain as still give every
    // SM sub-partition a warp (the serial part of a step is shared by the 32/L chains of a warp).
    const long long smsp = 148ll * 4;
    if (d.N >= 192 && (long long)d.C * 4 <= 2 * smsp) L = 128;
    else {
      L = 32;
      while (L > 8 && (long long)d.C * (L / 2) / 32 >= 2 * smsp && d.N > L / 2) L /= 2;
      while (L > 4 && L / 2 >= d.N) L /= 2;
    }
  }
  PtLaunch pl{};
  pl.lanes = L;
  if (L <= 32) {
    const int G = 32 / L;
    pl.Ns = round_up(d.N, L);
    // chains of one warp must start in different banks: stride = L (mod Q) words, where Q words
    // span all 32 banks (fp64: a warp's 8-byte loads go in two phases of 16 lanes, Q = 16)
    const int Q = 128 / real_bytes;
    int ss = 3 * pl.Ns;
    while (ss % Q != L % Q) ++ss;
    pl.sstride = ss;
    const long long warps = ((long long)d.C + G - 1) / G;
    const int wpc = warps <= 148ll * 24 ? 1 : 4;
    pl.threads = 32 * wpc;
    pl.chains_per_cta = G * wpc;
    pl.grid = (int)((d.C + pl.chains_per_cta - 1) / pl.chains_per_cta);
    pl.smem_bytes = pl.chains_per_cta * pl.sstride * real_bytes;
  } else {
    pl.Ns = round_up(d.N, L);
    pl.sstride = 3 * pl.Ns;
    pl.threads = L;
    pl.chains_per_cta = 1;
    pl.grid = d.C;
    pl.smem_bytes = pl.sstride * real_bytes;
  }
  if (pl.smem_bytes > 200 * 1024) return cudaErrorInvalidValue;
  *plan = pl;
  return cudaSuccess;
}

cudaError_t pt_launch_sweep(const PtDev& d, int precision, const PtLaunch& pl, uint32_t t0, int n_sweeps,
                            cudaStream_t stream)
{
  static bool attr_done = false;
  if (!attr_done) {
    const int big = 200 * 1024;
    cudaFuncSetAttribute(k_sweep_group<double, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_group<double, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_group<double, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_group<double, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_cta<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_group<float, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_group<float, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_group<float, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_group<float, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sweep_cta<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  return precision == PT_F32 ? launch_t<float>(d, pl, t0, n_sweeps, stream)
                             : launch_t<double>(d, pl, t0, n_sweeps, stream);
}
