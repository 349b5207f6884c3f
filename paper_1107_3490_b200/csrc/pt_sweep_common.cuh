// Pieces shared by the sweep kernels of pt_sweep.cu: per-chain context, proposal,
// once-per-sweep measurement.  Everything is static to its translation unit.
#pragma once
#include <math.h>

#include "pt_device.cuh"

namespace {

// Sum over the L lanes of a chain's group, returned to all of them.  lig = lane in group, gbase = first
// lane of the group.  L a power of two: butterfly.  Otherwise (L = 10: three chains per warp, lanes
// 30, 31 are ghosts that duplicate lane 29 and are never read): a tree padded to the next power of
// two, then a broadcast from the group's first lane.
template <typename Real, int L> __device__ __forceinline__ Real group_sum(Real v, int lig, int gbase)
{
  if ((L & (L - 1)) == 0) {
#pragma unroll
    for (int o = L / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
  }
  int active = L;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    if (o < L) {
      const Real w = __shfl_down_sync(0xffffffffu, v, o);
      v += (lig < o && lig + o < active) ? w : (Real)0;
      active = o < active ? o : active;
    }
  }
  return __shfl_sync(0xffffffffu, v, gbase);
}

// Everything a chain carries through a launch besides its coordinates.
struct ChainCtx {
  int s, e, i, ti;
  bool active;
  double beta;
  uint2 key;
  double erun;
  double mom1, mom2;
  unsigned acc, brej;
};

// `end`: first chain this warp (or CTA) must NOT touch; chains at or beyond it are inactive clones of chain C-1
__device__ __forceinline__ void ctx_load(const PtDev& d, int s, int end, ChainCtx& c)
{
  c.active = s < end;   // callers pass end <= d.C
  c.s = c.active ? s : d.C - 1;
  c.e = c.s / d.M;
  c.i = d.temp_of_slot[c.s];
  c.ti = c.e * d.M + c.i;
  c.beta = d.beta[c.i];
  c.key = d.keys[c.e];
  c.erun = d.erun[c.s];
  c.mom1 = d.mom[3 * c.ti + 1];
  c.mom2 = d.mom[3 * c.ti + 2];
  c.acc = 0;
  c.brej = 0;
}

// once per sweep, by one thread of the chain (A8): histogram, moments, energy trace.  A temperature index
// is owned by exactly one chain during a launch, so no atomics are needed.  (The two energy sums stay in
// registers: moving them to global memory changed ptxas' schedule of the step loop for the worse, +2 %.)
__device__ __forceinline__ void measure_energy(const PtDev& d, ChainCtx& c, uint32_t t)
{
  const double E = c.erun;
  if (d.nbins > 0) {
    const double b = floor((E - d.hist_emin) * d.hist_scale);
    int idx;
    if (b >= 0.0 && b < (double)d.nbins) idx = (int)b;
    else if (b < 0.0) idx = d.nbins;       // underflow
    else idx = d.nbins + 1;                // overflow (and NaN)
    // temperature index ti is owned by exactly one chain during a launch: no atomic needed
    d.hist[(size_t)c.ti * (size_t)(d.nbins + 2) + idx] += 1ull;
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
  d.mcount[3 * c.ti + 0] += (unsigned long long)n_sweeps * (unsigned long long)d.N;
  d.mcount[3 * c.ti + 1] += c.acc;
  d.mcount[3 * c.ti + 2] += c.brej;
}

// The proposal of one step (A2): which monomer, where to, and the acceptance uniform.
template <typename Real> struct Proposal {
  int m;
  Real sx, sy, sz, u;
};

template <typename Real>
__device__ __forceinline__ Proposal<Real> draw_proposal(const ChainCtx& c, bool pick, int N, uint32_t k, uint32_t t)
{
  Proposal<Real> p;
  p.m = (int)k;
  if (pick) {   // "a random monomer of the chain is picked"
    const uint4 wp = pt_draw(c.key, k, t, (uint32_t)c.e, PT_TAG_PICK, (uint32_t)c.i);
    p.m = (int)__umulhi(wp.x, (uint32_t)N);
  }
  const uint4 w = pt_draw(c.key, k, t, (uint32_t)c.e, PT_TAG_MOVE, (uint32_t)c.i);
  p.sx = PtNum<Real>::sym(w.x);
  p.sy = PtNum<Real>::sym(w.y);
  p.sz = PtNum<Real>::sym(w.z);
  p.u = PtNum<Real>::u01(w.w);
  return p;
}

// A3 for one partner j (other = "j is not the moved monomer"): adds u (A u - B) of the new and of
// the old distance to en / eo when inside the cutoff and counts the inside pairs (cnt = #new - #old)
// for the shift -C.  The new squared distance follows from the old one:
// |b + delta|^2 = |b|^2 + 2 delta.b + |delta|^2 with b = x_m - x_j.  Branch-free: the moved monomer
// itself is pushed to a huge distance, pairs outside the cutoff contribute u = 0.
template <typename Real>
__device__ __forceinline__ void pair_terms(const PtLJ<Real>& lj, bool other, const PtCoords<Real>& X, int j, Real xo,
                                           Real yo, Real zo, Real tdx, Real tdy, Real tdz, Real dd, Real& en,
                                           Real& eo, int& cnt)
{
  Real xj, yj, zj;
  X.get(j, xj, yj, zj);
  const Real bx = xo - xj, by = yo - yj, bz = zo - zj;
  const Real r2o = PtNum<Real>::keep_or_far(fma(bz, bz, fma(by, by, bx * bx)), other);
  const Real r2n = fma(tdx, bx, fma(tdy, by, fma(tdz, bz, r2o + dd)));
  cnt -= lj.add(r2o, eo) ? 1 : 0;
  cnt += lj.add(r2n, en) ? 1 : 0;
}

// A5 + the logarithm of A6, one instruction stream for a whole warp: threads with role 0..3 take
// the bonds (new m-1, new m+1, old m-1, old m+1) of Eq. (3), role 4 takes log(u) for the
// Metropolis test  u < exp(-beta dE)  <=>  log u < -beta dE  (Eq. 5).  Returns this thread's
// addend to Delta E; *lg is log(arg) of the role; *broke says a new bond left (r0-R, r0+R).
template <typename Real>
__device__ __forceinline__ Real bonds_and_logu(const PtDev& d, int role, int m, int N, const PtCoords<Real>& X,
                                               Real xo, Real yo, Real zo, Real xn, Real yn, Real zn, Real u,
                                               Real* lg, bool* broke)
{
  const int nb = (role & 1) ? m + 1 : m - 1;
  const bool isbond = role < 4 && nb >= 0 && nb < N;
  const bool isnew = role < 2;
  const int nbc = isbond ? nb : m;
  Real xb, yb, zb;
  X.get(nbc, xb, yb, zb);
  const Real dx = (isnew ? xn : xo) - xb;
  const Real dy = (isnew ? yn : yo) - yb;
  const Real dz = (isnew ? zn : zo) - zb;
  const Real r2 = isbond ? fma(dz, dz, fma(dy, dy, dx * dx)) : (Real)(d.r0 * d.r0);
  const Real r = PtNum<Real>::sqrt_(r2);
  const Real q = (r - (Real)d.r0) * (Real)d.invR;
  const Real g = fma(-q, q, (Real)1);              // 1 - ((r - r0)/R)^2
  const bool in_range = g > (Real)0;               // false for NaN as well
  *broke = isbond && isnew && !in_range;
  const Real arg = role == 4 ? u : ((isbond && in_range) ? g : (Real)1);
  *lg = PtNum<Real>::log_(arg);
  const Real fc = isnew ? (Real)d.feneC : (Real)-d.feneC;   // -(K/2) R^2
  return role < 4 ? fc * *lg : (Real)0;
}

// Eq. (8), and R_ee once per sweep; all lanes of the group take part.
template <typename Real, int L>
__device__ __forceinline__ void measure_shape(const PtDev& d, const ChainCtx& c, int N, int lig, int gbase,
                                              const PtCoords<Real>& X)
{
  double sx = 0.0, sy = 0.0, sz = 0.0;
  for (int j = lig; j < N; j += L) {
    Real x, y, z;
    X.get(j, x, y, z);
    sx += (double)x; sy += (double)y; sz += (double)z;
  }
  sx = group_sum<double, L>(sx, lig, gbase) / (double)N;
  sy = group_sum<double, L>(sy, lig, gbase) / (double)N;
  sz = group_sum<double, L>(sz, lig, gbase) / (double)N;
  double q = 0.0;
  for (int j = lig; j < N; j += L) {
    Real x, y, z;
    X.get(j, x, y, z);
    const double dx = (double)x - sx, dy = (double)y - sy, dz = (double)z - sz;
    q += dx * dx + dy * dy + dz * dz;
  }
  const double rg2 = group_sum<double, L>(q, lig, gbase) / (double)N;
  Real x0, y0, z0, x1, y1, z1;
  X.get(0, x0, y0, z0);
  X.get(N - 1, x1, y1, z1);
  const double ex = (double)x1 - (double)x0, ey = (double)y1 - (double)y0, ez = (double)z1 - (double)z0;
  const double ree2 = ex * ex + ey * ey + ez * ez;
  if (lig == 0 && c.active) {
    double* ob = d.obs + PT_NOBS * (size_t)c.ti;
    ob[0] += ree2; ob[1] += rg2; ob[2] += rg2 * rg2; ob[3] += ree2 * ree2;
    ob[4] += c.erun * rg2;   // the cross moment of d<r_gyr^2>/dT = beta^2 (<E r_gyr^2> - <E><r_gyr^2>)
  }
}

}  // namespace
