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
#include <stdlib.h>
#include <string.h>

#include "pt_sweep_common.cuh"

namespace {

// ------------------------------------------------------------------------------------------
// Warp-group kernel: L lanes per chain, 32/L chains per warp (L >= 8: roles 0..4 need 5 lanes).
// ------------------------------------------------------------------------------------------
// NI > 0: the partner loop has exactly NI iterations (Ns = NI * L) and is unrolled completely, so
// that the serial stream of a step (bond sqrt / log, log u) sits in the same basic block as the
// pair terms and the scheduler overlaps the two.  NI = 0: run-time trip count Ns / L.
template <typename Real, int L, int NI>
__global__ void __launch_bounds__(256, 1) k_sweep_group(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                     const int n_sweeps)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  static_assert(L >= 8 && L <= 32, "lanes per chain");
  constexpr int G = 32 / L;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane / L, lig = lane % L;
  const int cl = warp * G + g;
  const int N = d.N, Ns = pl.Ns;

  ChainCtx c;
  ctx_load(d, blockIdx.x * pl.chains_per_cta + cl, c);
  const Real width = (Real)d.width[c.i];
  const PtLJ<Real> lj(d);

  const PtCoords<Real> X(reinterpret_cast<Real*>(smem_raw) + (size_t)cl * pl.sstride, Ns);

  // A1: HBM -> shared memory; padding entries lie far outside every cutoff
  Real* gx = reinterpret_cast<Real*>(d.coords) + (size_t)c.s * 3 * d.Ng;
  for (int j = lig; j < Ns; j += L) {
    const bool in = j < N;
    X.set(j, in ? gx[j] : (Real)PT_FAR, in ? gx[d.Ng + j] : (Real)PT_FAR, in ? gx[2 * d.Ng + j] : (Real)PT_FAR);
  }
  __syncwarp();

  const bool pick = d.select_mode == PT_RANDOM_PICK;
  const bool leader = (lig == 0) && c.active;
  const unsigned bond_lanes = 3u << (g * L);   // roles 0, 1 of this group: the new bonds
  const double nbeta = -c.beta;

  Proposal<Real> nx = draw_proposal<Real>(c, pick, N, 0u, t0);
  for (int sw = 0; sw < n_sweeps; ++sw) {
    const uint32_t t = t0 + (uint32_t)sw;
    for (int k = 0; k < N; ++k) {
      // A2: this step's proposal was drawn one step ahead; draw the next one now so that the
      // integer work overlaps the fp64 work below
      const Proposal<Real> p = nx;
      {
        const bool last = k + 1 == N;
        nx = draw_proposal<Real>(c, pick, N, last ? 0u : (uint32_t)(k + 1), last ? t + 1u : t);
      }
      const int m = p.m;
      Real xo, yo, zo;
      X.get(m, xo, yo, zo);
      const Real xn = PtNum<Real>::propose(xo, width, p.sx);
      const Real yn = PtNum<Real>::propose(yo, width, p.sy);
      const Real zn = PtNum<Real>::propose(zo, width, p.sz);
      const Real ex = xn - xo, ey = yn - yo, ez = zn - zo;
      const Real dd = fma(ez, ez, fma(ey, ey, ex * ex));
      const Real tdx = ex + ex, tdy = ey + ey, tdz = ez + ez;

      // A5: bonds, and log u of A6
      Real lg;
      bool broke;
      const Real bond = bonds_and_logu<Real>(d, lig, m, N, X, xo, yo, zo, xn, yn, zn, p.u, &lg, &broke);

      // A3: Delta E_LJ, lanes stride over partners (Eq. 1, 2)
      Real en = (Real)0, eo = (Real)0;
      int cnt = 0;
      if (NI > 0) {
#pragma unroll
        for (int it = 0; it < NI; ++it) {
          const int j = lig + it * L;
          pair_terms<Real>(lj, j != m, X, j, xo, yo, zo, tdx, tdy, tdz, dd, en, eo, cnt);
        }
      } else {
#pragma unroll 2
        for (int j = lig; j < Ns; j += L)
          pair_terms<Real>(lj, j != m, X, j, xo, yo, zo, tdx, tdy, tdz, dd, en, eo, cnt);
      }
      const Real part = fma(-lj.C, (Real)cnt, en - eo) + bond;
      const bool bond_broken = (__ballot_sync(0xffffffffu, broke) & bond_lanes) != 0u;
      const Real logu = __shfl_sync(0xffffffffu, lg, g * L + 4);

      // A4: reduce; every lane of the group gets the same Delta E
      const Real dE = group_sum<Real, L>(part);

      // A6: Metropolis, Eq. (5): accept iff dE <= 0 or u < exp(-beta dE); NaN compares false
      const bool accept = !bond_broken && (dE <= (Real)0 || (double)logu < nbeta * (double)dE);

      // A7: commit
      if (lig == 0) {
        if (accept) X.set(m, xn, yn, zn);
        if (d.tr_move && c.active && (long long)t < d.cap_sweeps)
          d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
      }
      if (accept) { c.erun += (double)dE; c.acc++; }
      c.brej += bond_broken ? 1u : 0u;
      __syncwarp();
    }

    // A8: measurement once per sweep
    if (d.observables) measure_shape<Real, L>(c, N, lig, X);
    if (leader) measure_energy(d, c, t);
  }

  // A9: shared memory -> HBM
  __syncwarp();
  if (c.active) {
    for (int j = lig; j < N; j += L) X.get(j, gx[j], gx[d.Ng + j], gx[2 * d.Ng + j]);
    if (lig == 0) ctx_store(d, c, n_sweeps);
  }
}

// ------------------------------------------------------------------------------------------
// CTA-per-replica kernel: blockDim.x threads share one chain (long chains, few replicas).
// ------------------------------------------------------------------------------------------
template <typename Real>
__global__ void __launch_bounds__(256, 1) k_sweep_cta(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                   const int n_sweeps)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[2][8];
  __shared__ double s_logu[2];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int T = blockDim.x, NW = T >> 5;
  const int N = d.N, Ns = pl.Ns;

  ChainCtx c;
  ctx_load(d, blockIdx.x, c);
  const Real width = (Real)d.width[c.i];
  const PtLJ<Real> lj(d);

  const PtCoords<Real> X(reinterpret_cast<Real*>(smem_raw), Ns);
  Real* gx = reinterpret_cast<Real*>(d.coords) + (size_t)c.s * 3 * d.Ng;
  for (int j = tid; j < Ns; j += T) {
    const bool in = j < N;
    X.set(j, in ? gx[j] : (Real)PT_FAR, in ? gx[d.Ng + j] : (Real)PT_FAR, in ? gx[2 * d.Ng + j] : (Real)PT_FAR);
  }
  __syncthreads();

  const bool pick = d.select_mode == PT_RANDOM_PICK;
  const double nbeta = -c.beta;
  Proposal<Real> nx = draw_proposal<Real>(c, pick, N, 0u, t0);
  for (int sw = 0; sw < n_sweeps; ++sw) {
    const uint32_t t = t0 + (uint32_t)sw;
    for (int k = 0; k < N; ++k) {
      const Proposal<Real> p = nx;
      {
        const bool last = k + 1 == N;
        nx = draw_proposal<Real>(c, pick, N, last ? 0u : (uint32_t)(k + 1), last ? t + 1u : t);
      }
      const int m = p.m;
      Real xo, yo, zo;
      X.get(m, xo, yo, zo);
      const Real xn = PtNum<Real>::propose(xo, width, p.sx);
      const Real yn = PtNum<Real>::propose(yo, width, p.sy);
      const Real zn = PtNum<Real>::propose(zo, width, p.sz);
      const Real ex = xn - xo, ey = yn - yo, ez = zn - zo;
      const Real dd = fma(ez, ez, fma(ey, ey, ex * ex));
      const Real tdx = ex + ex, tdy = ey + ey, tdz = ez + ez;

      Real en = (Real)0, eo = (Real)0;
      int cnt = 0;
#pragma unroll 2
      for (int j = tid; j < Ns; j += T)
        pair_terms<Real>(lj, j != m, X, j, xo, yo, zo, tdx, tdy, tdz, dd, en, eo, cnt);
      Real part = fma(-lj.C, (Real)cnt, en - eo);

      // bonds and log u: roles 0..4 are threads 0..4 of warp 0; the other warps skip the stream
      bool broke = false;
      if (warp == 0) {
        Real lg;
        part += bonds_and_logu<Real>(d, lane, m, N, X, xo, yo, zo, xn, yn, zn, p.u, &lg, &broke);
        if (lane == 4) s_logu[k & 1] = (double)lg;
      }
      const Real wsum = group_sum<Real, 32>(part);
      if (lane == 0) red[k & 1][warp] = (double)wsum;
      const bool bond_broken = __syncthreads_or(broke ? 1 : 0) != 0;
      double dEd = red[k & 1][0];
      for (int q = 1; q < NW; ++q) dEd += red[k & 1][q];
      const Real dE = (Real)dEd;
      const double logu = s_logu[k & 1];

      const bool accept = !bond_broken && (dE <= (Real)0 || logu < nbeta * (double)dE);

      if (tid == 0) {
        if (accept) X.set(m, xn, yn, zn);
        if (d.tr_move && (long long)t < d.cap_sweeps)
          d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
      }
      if (accept) { c.erun += (double)dE; c.acc++; }
      c.brej += bond_broken ? 1u : 0u;
      __syncthreads();
    }

    if (d.observables && warp == 0) measure_shape<Real, 32>(c, N, lane, X);
    if (tid == 0) measure_energy(d, c, t);
  }

  __syncthreads();
  for (int j = tid; j < N; j += T) X.get(j, gx[j], gx[d.Ng + j], gx[2 * d.Ng + j]);
  if (tid == 0) ctx_store(d, c, n_sweeps);
}

int round_up(int a, int b) { return (a + b - 1) / b * b; }

typedef PtSweepFn SweepFn;

struct SweepVariant {
  int L, NI;
  SweepFn f64, f32;
};

#define PT_VARIANT(L, NI) { L, NI, k_sweep_group<double, L, NI>, k_sweep_group<float, L, NI> }
// Unrolled instantiations (NI = partner-loop iterations); NI = 0 is the run-time loop of the same
// lane count and must come last within its L.
const SweepVariant kVariants[] = {
    PT_VARIANT(8, 2),  PT_VARIANT(8, 4),  PT_VARIANT(8, 7),  PT_VARIANT(8, 10), PT_VARIANT(8, 13),
    PT_VARIANT(8, 0),
    PT_VARIANT(16, 1), PT_VARIANT(16, 2), PT_VARIANT(16, 4), PT_VARIANT(16, 7), PT_VARIANT(16, 0),
    PT_VARIANT(32, 1), PT_VARIANT(32, 2), PT_VARIANT(32, 4), PT_VARIANT(32, 0),
};

const SweepVariant* find_variant(int L, int ni_needed)
{
  for (const SweepVariant& v : kVariants)
    if (v.L == L && (v.NI == 0 || v.NI >= ni_needed)) return &v;
  return nullptr;
}

SweepFn kernel_of(const PtLaunch& pl, int precision, bool trace)
{
  if (pl.kind == PT_K_CTA) return precision == PT_F32 ? (SweepFn)k_sweep_cta<float> : (SweepFn)k_sweep_cta<double>;
  if (pl.kind == PT_K_SPEC)
    return precision == PT_F32 ? pt_spec_kernel_f32(pl.lanes, pl.ni, trace) : pt_spec_kernel_f64(pl.lanes, pl.ni, trace);
  for (const SweepVariant& v : kVariants)
    if (v.L == pl.lanes && v.NI == pl.ni) return precision == PT_F32 ? v.f32 : v.f64;
  return nullptr;
}

}  // namespace

cudaError_t pt_plan_sweep(const PtDev& d, int precision, int lanes_requested, PtLaunch* plan)
{
  const int real_bytes = precision == PT_F32 ? 4 : 8;
  int sms = 148;
  {
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) {
      int v = 0;
      if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) sms = v;
    }
    cudaGetLastError();
  }
  const long long smsp = 4ll * sms;
  int L = lanes_requested;
  if (L == 0) {
    // Few long chains: one CTA per replica.  Otherwise the fewest lanes per chain that still give
    // every SM sub-partition a warp: the serial part of a step (proposal, bonds, log u, decision)
    // is one instruction stream shared by the 32/L chains of a warp.
    if (d.N >= 192 && (long long)d.C <= smsp) L = 128;
    else {
      L = 32;
      while (L > 8 && ((long long)d.C * (L / 2) + 31) / 32 >= smsp && d.N > L / 2) L /= 2;
      while (L > 8 && L / 2 >= d.N) L /= 2;
    }
  }
  PtLaunch pl{};
  pl.lanes = L;
  if (L <= 32) {
    const int G = 32 / L;
    // The speculative schedule needs the sequential monomer order, N >= 4 and two padding slots.
    // PT_B200_SWEEP=serial forces the serial-schedule kernel (A/B measurements and tests).
    const char* forced = getenv("PT_B200_SWEEP");
    const bool serial_forced = forced && strcmp(forced, "serial") == 0;
    int ni = -1;
    if (d.select_mode == PT_SEQUENTIAL && d.N >= 4 && !serial_forced)
      ni = precision == PT_F32 ? pt_spec_find_f32(L, (d.N + 2 + L - 1) / L) : pt_spec_find_f64(L, (d.N + 2 + L - 1) / L);
    if (ni >= 0) {
      pl.kind = PT_K_SPEC;
      pl.ni = ni;
      pl.Ns = ni > 0 ? ni * L : round_up(d.N + 2, L);
    } else {
      const SweepVariant* v = find_variant(L, (d.N + L - 1) / L);
      if (!v) return cudaErrorInvalidValue;
      pl.kind = PT_K_GROUP;
      pl.ni = v->NI;
      pl.Ns = v->NI > 0 ? v->NI * L : round_up(d.N, L);
    }
    // chains of one warp must start in different banks: stride = L (mod Q) words, where Q words
    // span all 32 banks (fp64: a warp's 8-byte loads go in two phases of 16 lanes, Q = 16)
    const int Q = 128 / real_bytes;
    int ss = 3 * pl.Ns;
    while (ss % Q != L % Q) ++ss;
    pl.sstride = ss;
    // one CTA per SM when there are enough warps (its warps are dealt round-robin to the four
    // sub-partitions, so they are balanced by construction); single-warp CTAs otherwise
    const long long warps = ((long long)d.C + G - 1) / G;
    int wpc = 1;
    if (warps > sms) {
      wpc = (int)((warps + sms - 1) / sms);
      if (wpc > 8) wpc = 8;
    }
    pl.threads = 32 * wpc;
    pl.chains_per_cta = G * wpc;
    pl.grid = (int)((d.C + pl.chains_per_cta - 1) / pl.chains_per_cta);
    pl.smem_bytes = pl.chains_per_cta * pl.sstride * real_bytes;
  } else {
    pl.kind = PT_K_CTA;
    pl.ni = 0;
    pl.Ns = round_up(d.N, L);
    pl.sstride = 3 * pl.Ns;
    pl.threads = L;
    pl.chains_per_cta = 1;
    pl.grid = d.C;
    pl.smem_bytes = pl.sstride * real_bytes;
  }
  if (pl.smem_bytes > 200 * 1024) return cudaErrorInvalidValue;
  for (int trace = 0; trace < 2; ++trace) {
    SweepFn fn = kernel_of(pl, precision, trace != 0);
    if (!fn) return cudaErrorInvalidValue;
    if (pl.smem_bytes > 48 * 1024) {
      cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem_bytes);
      if (e != cudaSuccess) return e;
    }
  }
  *plan = pl;
  return cudaSuccess;
}

cudaError_t pt_launch_sweep(const PtDev& d, int precision, const PtLaunch& pl, uint32_t t0, int n_sweeps,
                            cudaStream_t stream)
{
  SweepFn fn = kernel_of(pl, precision, d.tr_move != nullptr);
  if (!fn) return cudaErrorInvalidValue;
  fn<<<dim3(pl.grid), dim3(pl.threads), pl.smem_bytes, stream>>>(d, pl, t0, n_sweeps);
  return cudaGetLastError();
}
