// Device code of the sweep kernels: included by the translation units that
// instantiate them (pt_sweep_group.cu, pt_sweep_comp*.cu).  Everything is internal to its translation unit.
//
// One chain's coordinates stay in shared memory for the whole launch (SoA x[], y[], z[]).
// Inside a chain the Markov chain is strictly serial; the parallelism is
//   (i)  over partner monomers j of the moved monomer m: L lanes stride over j and each adds
//        E_LJ^mod(|x' - x_j|) - E_LJ^mod(|x_m - x_j|) for its partners (Eq. 1, 2, 5), and
//   (ii) over chains: 32/L chains per warp, so that the serial part of a step (Philox, the FENE
//        sqrt/log, the Metropolis exp) is one instruction stream shared by 32/L chains.
// The paper's kernel (Listing 2) maps one replica to one block of 64 threads and
// recomputes the whole energy; that is prior art, kept only as the CTA-per-replica variant for
// very long chains (N > 480), and with the local Delta-E of Eq. (5) instead of the full sum.
//
// Kernels: k_sweep_group (L = 8, 16, 32 lanes per chain, partner loop unrolled in stage-major groups
// with the bond stream interleaved), k_sweep_comp (warps of 8, 10, 16 and 32 lanes per chain side by side in
// one CTA, against wave quantisation), k_sweep_cta.  pt_plan_sweep (pt_sweep.cu) chooses; DESIGN.md section 7
// has the measurements.
#pragma once
#include <math.h>
#include <stdio.h>

#include "pt_sweep_common.cuh"

namespace {

// A2 for eight steps at once.  All lanes of a chain would draw the same Philox block; instead lane l
// (mod 8) draws the block of step g0 + l, converts it to the displacement (width * s, one rounding,
// DESIGN.md R7) and the acceptance uniform, and every step fetches its four numbers with shuffles:
// 1/8 of the integer work per step.  Steps are numbered g = sweep * N + k within the launch.
template <typename Real> struct DrawBlock {
  Real dx, dy, dz, u;
  int m;
};

template <typename Real>
__device__ __forceinline__ DrawBlock<Real> draw_block(const ChainCtx& c, bool pick, int N, Real width, uint32_t t0,
                                                      int g0, int lig)
{
  const int gl = g0 + (lig & 7);
  const uint32_t k = (uint32_t)(gl % N), t = t0 + (uint32_t)(gl / N);
  DrawBlock<Real> b;
  b.m = (int)k;
  if (pick) {   // "a random monomer of the chain is picked"
    const uint4 wp = pt_draw(c.key, k, t, (uint32_t)c.e, PT_TAG_PICK, (uint32_t)c.i);
    b.m = (int)__umulhi(wp.x, (uint32_t)N);
  }
  const uint4 w = pt_draw(c.key, k, t, (uint32_t)c.e, PT_TAG_MOVE, (uint32_t)c.i);
  b.dx = PtNum<Real>::scale(width, PtNum<Real>::sym(w.x));
  b.dy = PtNum<Real>::scale(width, PtNum<Real>::sym(w.y));
  b.dz = PtNum<Real>::scale(width, PtNum<Real>::sym(w.z));
  b.u = PtNum<Real>::u01(w.w);
  return b;
}

template <typename Real>
__device__ __forceinline__ DrawBlock<Real> draw_fetch(const DrawBlock<Real>& b, int g, unsigned gsh)
{
  const int src = (int)gsh + (g & 7);
  DrawBlock<Real> r;
  r.dx = __shfl_sync(0xffffffffu, b.dx, src);
  r.dy = __shfl_sync(0xffffffffu, b.dy, src);
  r.dz = __shfl_sync(0xffffffffu, b.dz, src);
  r.u = __shfl_sync(0xffffffffu, b.u, src);
  r.m = __shfl_sync(0xffffffffu, b.m, src);
  return r;
}

// A5 + the logarithm of A6 (same roles and arithmetic as bonds_and_logu) cut into LEVELS of mutually
// independent instructions.  A warp issues in order: as one block of code these ~30 dependent fp64
// levels run back to back at the full 8-cycle DFMA latency (the S of DESIGN.md section 7, about 40 %
// of a one-warp step).  The pair groups call run<P, NPTS>() after each of their stages instead: one
// dependent level per ~10 independent pair instructions.  The logarithm's series is evaluated by
// Estrin's scheme (depth 4 instead of 10).
template <typename Real> struct BondChain {
  static constexpr int NLEV = 31;
  const PtDev& d;
  const PtCoords<Real>& X;
  int role, m, N;
  Real xo, yo, zo, xn, yn, zn, u;
  // results
  Real bond, lg;
  bool broke;
  // intermediates
  Real xb, yb, zb, dx, dy, dz, r2, r, q, gq;
  Real y, g, h, rr, tt;
  Real f, mp, x, e, sv, s2, z, z2, z4, z8, p01, p23, p45, p67, p89, q0, q1, pz, de;
  bool isbond, isnew, in_range;

  static constexpr bool kShortChain = false;   // pair groups in the throughput form (see pair_group)
  __device__ __forceinline__ BondChain(const PtDev& dev, const PtCoords<Real>& coords) : d(dev), X(coords) {}

  template <int K> __device__ __forceinline__ void level()
  {
    if (K == 0) {
      const int nb = (role & 1) ? m + 1 : m - 1;
      isbond = role < 4 && nb >= 0 && nb < N;
      isnew = role < 2;
      X.get(isbond ? nb : m, xb, yb, zb);
    }
    if (K == 1) {
      dx = (isnew ? xn : xo) - xb;
      dy = (isnew ? yn : yo) - yb;
      dz = (isnew ? zn : zo) - zb;
    }
    if (K == 2) r2 = dx * dx;
    if (K == 3) r2 = fma(dy, dy, r2);
    if (K == 4) { r2 = fma(dz, dz, r2); r2 = isbond ? r2 : (Real)(d.r0 * d.r0); }
    if constexpr (sizeof(Real) == 8) {
      // sqrt: MUFU.RSQ64H seed y, g = a y, r = (1 - a y^2)/2, sqrt a = g (1 + r + 3/2 r^2)
      if (K == 5) asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(r2));
      if (K == 6) { g = r2 * y; h = 0.5 * y; }
      if (K == 7) rr = fma(-h, g, 0.5);
      if (K == 8) tt = 1.5 * rr;
      if (K == 9) tt = fma(tt, rr, rr);
      if (K == 10) r = fma(g, tt, g);
    } else {
      if (K == 5) r = sqrtf(r2);
    }
    if (K == 11) q = r - (Real)d.r0;
    if (K == 12) q = q * (Real)d.invR;
    if (K == 13) gq = fma(-q, q, (Real)1);               // 1 - ((r - r0)/R)^2, Eq. (3)
    if (K == 14) {
      in_range = gq > (Real)0;                           // false for NaN as well
      broke = isbond && isnew && !in_range;
      gq = role == 4 ? u : ((isbond && in_range) ? gq : (Real)1);   // argument of the logarithm
    }
    if constexpr (sizeof(Real) == 8) {
      // log v, v = 2^e m, m in [sqrt(1/2), sqrt(2)): log m = 2 atanh(s), s = (m-1)/(m+1) (PtNum<double>::log_)
      if (K == 15) {
        const int hi = __double2hiint(gq);
        const int ex = (hi - 0x3fe6a09e) >> 20;
        const double mm = __hiloint2double(hi - (ex << 20), __double2loint(gq));
        de = (double)ex;
        f = mm - 1.0;
        mp = mm + 1.0;
      }
      if (K == 16) x = PtNum<double>::rcp_seed(mp);
      if (K == 17) e = fma(-mp, x, 1.0);
      if (K == 18) e = fma(e, e, e);
      if (K == 19) x = fma(x, e, x);
      if (K == 20) sv = f * x;
      if (K == 21) { z = sv * sv; s2 = sv + sv; }
      if (K == 22) {
        p01 = fma(kPtLogC[1], z, kPtLogC[0]);
        p23 = fma(kPtLogC[3], z, kPtLogC[2]);
        p45 = fma(kPtLogC[5], z, kPtLogC[4]);
        p67 = fma(kPtLogC[7], z, kPtLogC[6]);
        p89 = fma(kPtLogC[9], z, kPtLogC[8]);
        z2 = z * z;
      }
      if (K == 23) { q0 = fma(p23, z2, p01); q1 = fma(p67, z2, p45); z4 = z2 * z2; }
      if (K == 24) { q0 = fma(q1, z4, q0); z8 = z4 * z4; }
      if (K == 25) q0 = fma(p89, z8, q0);
      if (K == 26) pz = q0 * z;
      if (K == 27) lg = fma(sv, pz, s2);
      if (K == 28) lg = fma(de, 0x1.abc9e3b39803fp-56, lg);
      if (K == 29) lg = fma(de, 0x1.62e42fefa39efp-1, lg);
    } else {
      if (K == 15) lg = __logf(gq);
    }
    if (K == 30) bond = role < 4 ? (isnew ? (Real)d.feneC : (Real)-d.feneC) * lg : (Real)0;
  }
  template <int A, int B> __device__ __forceinline__ void range()
  {
    if constexpr (A < B) {
      level<A>();
      range<A + 1, B>();
    }
  }
  // stage point P of NPTS
  // stage point P of NPTS; LEVG = levels handed out over the stage points (the rest runs after the pair groups)
  template <int P, int NPTS, int LEVG> __device__ __forceinline__ void run()
  {
    range<(P * LEVG) / NPTS, ((P + 1) * LEVG) / NPTS>();
  }
  __device__ __forceinline__ void run_all() { range<0, NLEV>(); }
};

constexpr int kGroupPoints = 14;   // stage points per pair group

// A3 for CNT partner iterations at once (iterations BEGIN .. BEGIN+CNT-1 of this lane), written stage
// by stage across the partners: every stage holds CNT or 2 CNT independent fp64 instructions, so that
// a dependent instruction is not issued within the 8-cycle DFMA latency of its producer (written
// partner by partner, ptxas kept one or two chains in flight).
//
// Arithmetic (Eq. 1-2).  With u = 1/r^6 and c = B/A, E_LJ^mod = A u (u - c) - C inside the cutoff.
// Per evaluation v = u - c/2 (one DFMA from x^2 and x = 1/r^2); per partner
//   u_n (u_n - c) - u_o (u_o - c) = (v_n - v_o)(v_n + v_o):   DADD, DADD, DFMA.
// A pair outside the cutoff, and the moved monomer itself, get a zero reciprocal seed (one FSEL), which stays
// zero through the Newton step: u = 0, v = -c/2, and the partner adds exactly nothing unless it crosses the
// cutoff.  The cutoff test is one DSETP (fp64 pipe) with the "not myself" mask as its predicate input, the
// shift C needs the count of inside pairs (one predicated add); A and C are applied once per step by the
// caller.  The new squared distance follows from the old one:
// |b + delta|^2 = |b|^2 + 2 delta.b + |delta|^2, b = x_m - x_j.
template <typename Real, int L, int NI, int BEGIN, int CNT, int PBASE, int NPTS, int LEVG, class Side>
__device__ __forceinline__ void pair_group(const PtLJ<Real>& lj, const PtCoords<Real>& X, int s0, int sm,
                                           Real xo, Real yo, Real zo, Real tdx, Real tdy, Real tdz, Real dd,
                                           Real (&acc)[4], int& cnt, Side& side)
{
#define PT_SIDE(n) side.template run<PBASE + (n), NPTS, LEVG>()
  Real bx[CNT], by[CNT], bz[CNT], ro[CNT], rn[CNT];
#pragma unroll
  for (int u = 0; u < CNT; ++u) X.get(s0 + (BEGIN + u) * L, bx[u], by[u], bz[u]);
#pragma unroll
  for (int u = 0; u < CNT; ++u) { bx[u] = xo - bx[u]; by[u] = yo - by[u]; bz[u] = zo - bz[u]; }
  if constexpr (Side::kShortChain) {
    // a lone warp (k_sweep_ws): the same instructions as below, as two chains of depth 3 side by side and one
    // addition -- r_n^2 = r_o^2 + (|delta|^2 + 2 delta.b) -- instead of one chain of depth 7
#pragma unroll
    for (int u = 0; u < CNT; ++u) { ro[u] = bx[u] * bx[u]; rn[u] = fma(tdz, bz[u], dd); }
#pragma unroll
    for (int u = 0; u < CNT; ++u) { ro[u] = fma(by[u], by[u], ro[u]); rn[u] = fma(tdy, by[u], rn[u]); }
#pragma unroll
    for (int u = 0; u < CNT; ++u) { ro[u] = fma(bz[u], bz[u], ro[u]); rn[u] = fma(tdx, bx[u], rn[u]); }
#pragma unroll
    for (int u = 0; u < CNT; ++u) rn[u] = ro[u] + rn[u];
  } else {
    PT_SIDE(0);
#pragma unroll
    for (int u = 0; u < CNT; ++u) ro[u] = bx[u] * bx[u];
    PT_SIDE(1);
#pragma unroll
    for (int u = 0; u < CNT; ++u) ro[u] = fma(by[u], by[u], ro[u]);
    PT_SIDE(2);
#pragma unroll
    for (int u = 0; u < CNT; ++u) ro[u] = fma(bz[u], bz[u], ro[u]);
    PT_SIDE(3);
#pragma unroll
    for (int u = 0; u < CNT; ++u) rn[u] = ro[u] + dd;
    PT_SIDE(4);
#pragma unroll
    for (int u = 0; u < CNT; ++u) rn[u] = fma(tdz, bz[u], rn[u]);
    PT_SIDE(5);
#pragma unroll
    for (int u = 0; u < CNT; ++u) rn[u] = fma(tdy, by[u], rn[u]);
    PT_SIDE(6);
#pragma unroll
    for (int u = 0; u < CNT; ++u) rn[u] = fma(tdx, bx[u], rn[u]);
    PT_SIDE(7);
  }
  Real dv[2 * CNT], xv[2 * CNT], ev[2 * CNT];
#pragma unroll
  for (int u = 0; u < CNT; ++u) {
    const int j = s0 + (BEGIN + u) * L;
    dv[2 * u] = ro[u];
    dv[2 * u + 1] = rn[u];
    xv[2 * u] = PtNum<Real>::template seed_if_inside<-1>(ro[u], lj.rc2, j, sm, cnt);
    xv[2 * u + 1] = PtNum<Real>::template seed_if_inside<1>(rn[u], lj.rc2, j, sm, cnt);
  }
  PT_SIDE(8);
  if (PtNum<Real>::kNewton) {
#pragma unroll
    for (int v = 0; v < 2 * CNT; ++v) ev[v] = fma(-dv[v], xv[v], (Real)1);
    PT_SIDE(9);
#pragma unroll
    for (int v = 0; v < 2 * CNT; ++v) ev[v] = fma(ev[v], ev[v], ev[v]);
    PT_SIDE(10);
#pragma unroll
    for (int v = 0; v < 2 * CNT; ++v) xv[v] = fma(xv[v], ev[v], xv[v]);
  } else {   // fp32: the MUFU reciprocal is final; the serial stream still gets its two turns
    PT_SIDE(9);
    PT_SIDE(10);
  }
#pragma unroll
  for (int v = 0; v < 2 * CNT; ++v) ev[v] = xv[v] * xv[v];
  PT_SIDE(11);
#pragma unroll
  for (int v = 0; v < 2 * CNT; ++v) xv[v] = fma(ev[v], xv[v], lj.mhc);          // v = 1/r^6 - c/2
  PT_SIDE(12);
#pragma unroll
  for (int u = 0; u < CNT; ++u) {
    ev[2 * u] = xv[2 * u + 1] - xv[2 * u];
    ev[2 * u + 1] = xv[2 * u + 1] + xv[2 * u];
  }
  PT_SIDE(13);
#pragma unroll
  for (int u = 0; u < CNT; ++u) acc[(BEGIN + u) & 3] = fma(ev[2 * u], ev[2 * u + 1], acc[(BEGIN + u) & 3]);
#undef PT_SIDE
}

// How the NI partner iterations of a lane are cut into groups (each group is one stage-major block of
// pair_group).  Balanced groups of at most kMaxGroup partners: 13 -> 5 + 4 + 4, 10 -> 5 + 5, <= 5 -> one group.
// Measured on B200 (config 5): 5 + 4 + 4 / 5 + 5 is 3 % faster than 4 + 4 + 5 / 4 + 6.
#ifndef PT_MAXGROUP
#define PT_MAXGROUP 5
#endif
constexpr int kMaxGroup = PT_MAXGROUP;
#ifndef PT_MAXGROUP_F2
#define PT_MAXGROUP_F2 5
#endif
constexpr int kMaxGroupF2 = PT_MAXGROUP_F2;   // fp32: pairs of partners per group
__host__ __device__ constexpr int n_groups(int NI, int mg = kMaxGroup) { return NI <= 0 ? 0 : (NI + mg - 1) / mg; }
// size and first iteration of group g: the first (NI mod n) groups get one more
__host__ __device__ constexpr int group_size(int NI, int g, int mg = kMaxGroup)
{
  return NI / n_groups(NI, mg) + (g < NI % n_groups(NI, mg) ? 1 : 0);
}
__host__ __device__ constexpr int group_begin(int NI, int g, int mg = kMaxGroup)
{
  return g == 0 ? 0 : group_begin(NI, g - 1, mg) + group_size(NI, g - 1, mg);
}

// The whole partner loop of NI > 0 iterations: returns this lane's share of Delta E_LJ.
// s0 = this lane's first partner, sm = the moved monomer (its own slot is masked out).
template <typename Real, int L, int NI, int LEVG, class Side>
__device__ __forceinline__ Real pair_groups(const PtLJ<Real>& lj, const PtCoords<Real>& X, int s0, int sm,
                                            Real xo, Real yo, Real zo, Real tdx, Real tdy, Real tdz, Real dd,
                                            Side& side)
{
  constexpr int P = kGroupPoints;
  constexpr int NG = n_groups(NI);
  static_assert(NG >= 1 && NG <= 4, "add a group");
  Real acc[4] = {(Real)0, (Real)0, (Real)0, (Real)0};
  int cnt = 0;
#define PT_PG(g)                                                                                             \
  if (NG > g)                                                                                                \
    pair_group<Real, L, NI, group_begin(NI, g < NG ? g : 0), group_size(NI, g < NG ? g : 0), g * P, NG * P, LEVG>( \
        lj, X, s0, sm, xo, yo, zo, tdx, tdy, tdz, dd, acc, cnt, side)
  PT_PG(0);
  PT_PG(1);
  PT_PG(2);
  PT_PG(3);
#undef PT_PG
  return fma(lj.A, (acc[0] + acc[1]) + (acc[2] + acc[3]), -lj.C * (Real)cnt);
}

#ifndef PT_F32_ONE_RCP
#define PT_F32_ONE_RCP 1
#endif
// ---- fp32: two adjacent partners per lane and iteration, packed arithmetic --------------------------------
// The fp32 kernels are bound by issue slots, not by a pipe (ncu: 70 % of the issue slots, 40 % of the FMA pipe), so
// they do the arithmetic of the partners 2p and 2p+1 with one FADD2 / FMUL2 / FFMA2 each: iteration `it` of lane `lig`
// takes the pair p = lig + L it (three 64-bit loads from the x[], y[], z[] arrays).  The cutoff is applied as Eq. (1)
// prints it, E_LJ(min(r, r_c)) - E_LJ(r_c): r^2 is clamped to r_c^2 (one FMNMX), a pair beyond the cutoff then has
// u = u_c in the old and in the new position and (v_n - v_o)(v_n + v_o) is exactly 0 -- no mask, no count of inside
// pairs, and C drops out.  The moved monomer itself gets r^2 = r_c^2 in both positions.  (The fp64 path cannot clamp:
// it has no single-instruction 64-bit minimum.)  The fp32 path is checked statistically (tests/test_gpu_fp32_stat.py).
template <int L, int BEGIN, int CNT, int PBASE, int NPTS, int LEVG, class Side>
__device__ __forceinline__ void pair_group_f2(const PtLJ<float>& lj, const PtCoords<float>& X, int p0, int m, PtF2 xo2,
                                              PtF2 yo2, PtF2 zo2, PtF2 tdx2, PtF2 tdy2, PtF2 tdz2, PtF2 dd2, PtF2 mhc2,
                                              PtF2 (&acc)[2], Side& side)
{
#define PT_SIDE(n) side.template run<PBASE + (n), NPTS, LEVG>()
  PtF2 bx[CNT], by[CNT], bz[CNT], ro[CNT], rn[CNT];
#pragma unroll
  for (int u = 0; u < CNT; ++u) X.get2(p0 + (BEGIN + u) * L, bx[u], by[u], bz[u]);
#pragma unroll
  for (int u = 0; u < CNT; ++u) { bx[u] = pt_sub2(xo2, bx[u]); by[u] = pt_sub2(yo2, by[u]); bz[u] = pt_sub2(zo2, bz[u]); }
  PT_SIDE(0);
#pragma unroll
  for (int u = 0; u < CNT; ++u) ro[u] = pt_mul2(bx[u], bx[u]);
  PT_SIDE(1);
#pragma unroll
  for (int u = 0; u < CNT; ++u) ro[u] = pt_fma2(by[u], by[u], ro[u]);
  PT_SIDE(2);
#pragma unroll
  for (int u = 0; u < CNT; ++u) ro[u] = pt_fma2(bz[u], bz[u], ro[u]);
  PT_SIDE(3);
#pragma unroll
  for (int u = 0; u < CNT; ++u) rn[u] = pt_add2(ro[u], dd2);
  PT_SIDE(4);
#pragma unroll
  for (int u = 0; u < CNT; ++u) rn[u] = pt_fma2(tdz2, bz[u], rn[u]);
  PT_SIDE(5);
#pragma unroll
  for (int u = 0; u < CNT; ++u) rn[u] = pt_fma2(tdy2, by[u], rn[u]);
  PT_SIDE(6);
#pragma unroll
  for (int u = 0; u < CNT; ++u) rn[u] = pt_fma2(tdx2, bx[u], rn[u]);
  PT_SIDE(7);
  PtF2 xo_[CNT], xn_[CNT];
#pragma unroll
  for (int u = 0; u < CNT; ++u) {
    const int j = 2 * (p0 + (BEGIN + u) * L);
    float oa, ob, na, nb;
    pt_f2_split(ro[u], oa, ob);
    pt_f2_split(rn[u], na, nb);
    const bool sa = j == m, sb = j + 1 == m;
    oa = sa ? lj.rc2 : fminf(oa, lj.rc2); na = sa ? lj.rc2 : fminf(na, lj.rc2);
    ob = sb ? lj.rc2 : fminf(ob, lj.rc2); nb = sb ? lj.rc2 : fminf(nb, lj.rc2);
#if PT_F32_ONE_RCP
    // one reciprocal for the old and the new distance of a partner: 1/r_o^2 = r_n^2 / (r_o^2 r_n^2)
    const PtF2 co = pt_f2(oa, ob), cn = pt_f2(na, nb);
    float pa, pb;
    pt_f2_split(pt_mul2(co, cn), pa, pb);
    const PtF2 ip = pt_f2(PtNum<float>::rcp(pa), PtNum<float>::rcp(pb));
    xo_[u] = pt_mul2(ip, cn);
    xn_[u] = pt_mul2(ip, co);
#else
    xo_[u] = pt_f2(PtNum<float>::rcp(oa), PtNum<float>::rcp(ob));
    xn_[u] = pt_f2(PtNum<float>::rcp(na), PtNum<float>::rcp(nb));
#endif
  }
  PT_SIDE(8);
  PT_SIDE(9);
  PT_SIDE(10);
  PtF2 eo[CNT], en[CNT];
#pragma unroll
  for (int u = 0; u < CNT; ++u) { eo[u] = pt_mul2(xo_[u], xo_[u]); en[u] = pt_mul2(xn_[u], xn_[u]); }
  PT_SIDE(11);
#pragma unroll
  for (int u = 0; u < CNT; ++u) { xo_[u] = pt_fma2(eo[u], xo_[u], mhc2); xn_[u] = pt_fma2(en[u], xn_[u], mhc2); }   // v = 1/r^6 - c/2
  PT_SIDE(12);
#pragma unroll
  for (int u = 0; u < CNT; ++u) { eo[u] = pt_sub2(xn_[u], xo_[u]); en[u] = pt_add2(xn_[u], xo_[u]); }
  PT_SIDE(13);
#pragma unroll
  for (int u = 0; u < CNT; ++u) acc[(BEGIN + u) & 1] = pt_fma2(eo[u], en[u], acc[(BEGIN + u) & 1]);
#undef PT_SIDE
}

// NI2 iterations of two partners each (2 L NI2 table slots); returns this lane's share of Delta E_LJ
template <int L, int NI2, int LEVG, class Side>
__device__ __forceinline__ float pair_groups_f2(const PtLJ<float>& lj, const PtCoords<float>& X, int lig, int m, float xo,
                                                float yo, float zo, float tdx, float tdy, float tdz, float dd,
                                                Side& side)
{
  constexpr int P = kGroupPoints;
  constexpr int NG = n_groups(NI2, kMaxGroupF2);
  static_assert(NG >= 1 && NG <= 4, "add a group");
  PtF2 acc[2] = {pt_f2(0.0f, 0.0f), pt_f2(0.0f, 0.0f)};
  const PtF2 xo2 = pt_f2(xo, xo), yo2 = pt_f2(yo, yo), zo2 = pt_f2(zo, zo), tdx2 = pt_f2(tdx, tdx), tdy2 = pt_f2(tdy, tdy),
             tdz2 = pt_f2(tdz, tdz), dd2 = pt_f2(dd, dd), mhc2 = pt_f2(lj.mhc, lj.mhc);
#define PT_PG(g)                                                                                              \
  if (NG > g)                                                                                                 \
    pair_group_f2<L, group_begin(NI2, g < NG ? g : 0, kMaxGroupF2), group_size(NI2, g < NG ? g : 0, kMaxGroupF2), g * P, NG * P, LEVG>(   \
        lj, X, lig, m, xo2, yo2, zo2, tdx2, tdy2, tdz2, dd2, mhc2, acc, side)
  PT_PG(0);
  PT_PG(1);
  PT_PG(2);
  PT_PG(3);
#undef PT_PG
  float a0, a1, b0, b1;
  pt_f2_split(acc[0], a0, a1);
  pt_f2_split(acc[1], b0, b1);
  return lj.A * ((a0 + a1) + (b0 + b1));
}

// ------------------------------------------------------------------------------------------
// Warp-group kernel: L lanes per chain, 32/L chains per warp (L >= 8: roles 0..4 need 5 lanes).
// ------------------------------------------------------------------------------------------
// NI > 0: the partner loop has exactly NI iterations (Ns = NI * L) and is unrolled completely, so
// that the serial stream of a step (bond sqrt / log, log u) sits in the same basic block as the
// pair terms and the scheduler overlaps the two.  NI = 0: run-time trip count Ns / L.
// One warp's share of a sweep launch: up to G = 32 / L chains, slots `chain0` .. `chain_end` - 1, coordinates at
// `smem0` (stride `sstride` Reals between chains, Ns slots per coordinate array).  `delay`: cycles to
// wait before the first step (phase stagger).
template <typename Real, int L, int NI, bool TRACE>
__device__ __forceinline__ void sweep_warp(const PtDev& d, Real* smem0, int sstride, int Ns_runtime, int chain0,
                                           int chain_end, int delay, const uint32_t t0, const int n_sweeps)
{
  static_assert(L >= 8 && L <= 32, "lanes per chain");
  constexpr int G = 32 / L;
  // Short partner loops have fewer stage points than the bond stream has levels: one level per point,
  // the rest of the stream runs behind the reduction of the pair sums (latency-bound shapes).
  constexpr bool F2 = sizeof(Real) == 4 && NI > 0;      // fp32: two partners per lane and iteration (pair_group_f2)
  constexpr int NI2 = (NI + 1) / 2;
  constexpr int NPTS = (F2 ? n_groups(NI2, kMaxGroupF2) : n_groups(NI)) * kGroupPoints;
  // table slots per coordinate array: unrolled kernels know them at compile time (fp32: an even number of iterations)
  const int Ns = NI > 0 ? (F2 ? 2 * L * NI2 : L * NI) : Ns_runtime;
  constexpr bool TAIL = NI > 0 && (L & (L - 1)) == 0 && NPTS < BondChain<Real>::NLEV;
  constexpr int LEVG = TAIL ? NPTS : BondChain<Real>::NLEV;
  // lanes beyond G L (L = 10: lanes 30, 31) are ghosts: they repeat the last real lane and nobody reads them
  const int lane = min((int)(threadIdx.x & 31), G * L - 1);
  const int g = lane / L, lig = lane % L;
  const int gbase = g * L;
  const int N = d.N;

  ChainCtx c;
  ctx_load(d, chain0 + g, chain_end, c);
  const Real width = (Real)d.width[c.i];
  const PtLJ<Real> lj(d);

  const PtCoords<Real> X(smem0 + (size_t)g * sstride, Ns);

  // A1: HBM -> shared memory; padding entries lie far outside every cutoff
  Real* gx = reinterpret_cast<Real*>(d.coords) + (size_t)c.s * 3 * d.Ng;
  for (int j = lig; j < Ns; j += L) {
    const bool in = j < N;
    X.set(j, in ? gx[j] : (Real)PT_FAR, in ? gx[d.Ng + j] : (Real)PT_FAR, in ? gx[2 * d.Ng + j] : (Real)PT_FAR);
  }
  __syncwarp();

  if (delay > 0) {
    const long long until = clock64() + (long long)delay;
    while (clock64() < until) { }
  }

  const bool pick = d.select_mode == PT_RANDOM_PICK;
  const bool leader = (lig == 0) && c.active;
  const unsigned bond_lanes = 3u << gbase;   // roles 0, 1 of this group: the new bonds
  const double nbeta = -c.beta;

  const unsigned gsh = (unsigned)gbase;
  DrawBlock<Real> blk = draw_block<Real>(c, pick, N, width, t0, 0, lig);
  DrawBlock<Real> nx = draw_fetch<Real>(blk, 0, gsh);
  int gstep = 0;   // step number within the launch
  for (int sw = 0; sw < n_sweeps; ++sw) {
    const uint32_t t = t0 + (uint32_t)sw;
    for (int k = 0; k < N; ++k) {
      // A2: this step's numbers were fetched one step ahead; fetch the next ones now (and draw the
      // next eight blocks when they are used up) so that the shuffles overlap the fp64 work below
      const DrawBlock<Real> p = nx;
      ++gstep;
      if ((gstep & 7) == 0) blk = draw_block<Real>(c, pick, N, width, t0, gstep, lig);
      nx = draw_fetch<Real>(blk, gstep, gsh);
      const int m = p.m;
      Real xo, yo, zo;
      X.get(m, xo, yo, zo);
      const Real xn = PtNum<Real>::shift(xo, p.dx);
      const Real yn = PtNum<Real>::shift(yo, p.dy);
      const Real zn = PtNum<Real>::shift(zo, p.dz);
      const Real ex = xn - xo, ey = yn - yo, ez = zn - zo;
      const Real dd = fma(ez, ez, fma(ey, ey, ex * ex));
      const Real tdx = ex + ex, tdy = ey + ey, tdz = ez + ez;

      // A5 (bonds, and log u of A6) rides along with A3 (Delta E_LJ, lanes stride over partners, Eq. 1, 2)
      BondChain<Real> bc(d, X);
      bc.role = lig; bc.m = m; bc.N = N;
      bc.xo = xo; bc.yo = yo; bc.zo = zo; bc.xn = xn; bc.yn = yn; bc.zn = zn; bc.u = p.u;
      Real part;
      if (NI > 0) {
        if constexpr (F2) part = pair_groups_f2<L, NI2, LEVG>(lj, X, lig, m, xo, yo, zo, tdx, tdy, tdz, dd, bc);
        else part = pair_groups<Real, L, (NI > 0 ? NI : 1), LEVG>(lj, X, lig, m, xo, yo, zo, tdx, tdy, tdz, dd, bc);
      } else {
        bc.run_all();
        Real en = (Real)0, eo = (Real)0;
        int cnt = 0;
#pragma unroll 2
        for (int j = lig; j < Ns; j += L)
          pair_terms<Real>(lj, j != m, X, j, xo, yo, zo, tdx, tdy, tdz, dd, en, eo, cnt);
        part = fma(-lj.C, (Real)cnt, en - eo);
      }
      Real dE, logu;
      bool bond_broken;
      if (TAIL) {
        // A4 in two parts: the pair sums are reduced while the bond stream finishes (its last levels ride
        // on the shuffle latencies); the bond terms sit in lanes 0..3 of the group and need two levels
        Real v = part;
        constexpr int REM = BondChain<Real>::NLEV - LEVG;
        constexpr int NSH = L == 32 ? 5 : (L == 16 ? 4 : 3);
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        bc.template range<LEVG, LEVG + REM / NSH>();
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        bc.template range<LEVG + REM / NSH, LEVG + 2 * REM / NSH>();
        v += __shfl_xor_sync(0xffffffffu, v, 4);
        bc.template range<LEVG + 2 * REM / NSH, LEVG + 3 * REM / NSH>();
        if (L >= 16) {
          v += __shfl_xor_sync(0xffffffffu, v, 8);
          bc.template range<LEVG + 3 * REM / NSH, LEVG + 4 * REM / NSH>();
        }
        if (L == 32) {
          v += __shfl_xor_sync(0xffffffffu, v, 16);
          bc.template range<LEVG + 4 * REM / NSH, LEVG + REM>();
        }
        Real b = bc.bond;
        b += __shfl_xor_sync(0xffffffffu, b, 1);
        b += __shfl_xor_sync(0xffffffffu, b, 2);
        bond_broken = (__ballot_sync(0xffffffffu, bc.broke) & bond_lanes) != 0u;
        logu = __shfl_sync(0xffffffffu, bc.lg, gbase + 4);
        dE = v + __shfl_sync(0xffffffffu, b, gbase);
      } else {
        bond_broken = (__ballot_sync(0xffffffffu, bc.broke) & bond_lanes) != 0u;
        logu = __shfl_sync(0xffffffffu, bc.lg, gbase + 4);
        // A4: reduce; every lane of the group gets the same Delta E
        dE = group_sum<Real, L>(part + bc.bond, lig, gbase);
      }

      // A6: Metropolis, Eq. (5): accept iff dE <= 0 or u < exp(-beta dE); NaN compares false
      const bool accept = !bond_broken && (dE <= (Real)0 || (double)logu < nbeta * (double)dE);

      // A7: commit (branch-free: predicated stores, selects for the bookkeeping)
      if (accept && lig == 0) X.set(m, xn, yn, zn);
      if (TRACE) {   // test support (pt_set_trace): a separate instantiation, the timed one has no branch here
        if (lig == 0 && d.tr_move && c.active && (long long)t < d.cap_sweeps)
          d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
      }
      c.erun += accept ? (double)dE : 0.0;
      c.acc += accept ? 1u : 0u;
      c.brej += bond_broken ? 1u : 0u;
      __syncwarp();
    }

    // A8: measurement once per sweep
    if (d.observables) measure_shape<Real, L>(d, c, N, lig, gbase, X);
    if (leader) measure_energy(d, c, t);
  }

  // A9: shared memory -> HBM
  __syncwarp();
  if (c.active) {
    for (int j = lig; j < N; j += L) X.get(j, gx[j], gx[d.Ng + j], gx[2 * d.Ng + j]);
    if (lig == 0) ctx_store(d, c, n_sweeps);
  }
}

// Warps w and w + 4 of a CTA share an SM sub-partition and run the same code: started together they
// stay in phase, both in the fp64-bound pair loop, then both in the latency-bound serial part of
// the step (period 2P + S).  The second one therefore starts `stagger` cycles (about one partner
// loop) late, so that its serial part can hide under the pair loop of the first.
template <typename Real, int L, int NI, bool TRACE>
__global__ void __launch_bounds__(256, 1) k_sweep_group(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                     const int n_sweeps)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int G = 32 / L;
  const int warp = threadIdx.x >> 5;
  sweep_warp<Real, L, NI, TRACE>(d, reinterpret_cast<Real*>(smem_raw) + (size_t)(warp * G) * pl.sstride, pl.sstride, pl.Ns,
                                 blockIdx.x * pl.chains_per_cta + warp * G, d.C, pl.stagger * (warp >> 2), t0, n_sweeps);
}

// Composed CTA against wave quantisation (the paper's staircase).  With uniform warps a
// sub-partition jumps from one warp to two as soon as the chains per SM pass a multiple of 4, 8 or 16, and the
// most loaded sub-partition sets the time.  Here the chains are spread evenly over the SMs (q = ceil(C / #SM) per
// CTA, one CTA per SM and wave), and every sub-partition gets one or two warps whose kinds are chosen for its load:
//   1 chain: 32 lanes   2: 2 x 16   3: 3 of 4 x 8   4: 4 x 8   5: 4 x 8 + 1 x 32   6: 4 x 8 + 2 x 16
//   7: 4 x 8 + 3 of 4 x 8   8: 4 x 8 + 4 x 8
// ("3 of 4 x 8": an 8-lane warp with one chain slot left idle).  Warp w of a CTA runs on sub-partition w mod 4; its
// kind, first chain, number of chains and shared-memory offset come from the launch descriptor.  N8, N16, N32 =
// partner iterations of the three kinds of warp (L x NI slots >= N).
template <typename Real, int N8, int N16, int N32, bool TRACE>
__global__ void __launch_bounds__(256, 1) k_sweep_comp(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                    const int n_sweeps)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5;
  const int kind = pl.wkind[warp];
  const int chain0 = blockIdx.x * pl.chains_per_cta + pl.wfirst[warp];
  const int chain_end = min(chain0 + pl.wcount[warp], (int)min((long long)d.C, (long long)(blockIdx.x + 1) * pl.chains_per_cta));
  if (chain0 >= chain_end) return;           // no chain for this warp (a partly filled last CTA, an unused warp slot)
  Real* base = reinterpret_cast<Real*>(smem_raw) + pl.woff[warp];
  const int delay = pl.wdelay[warp];
  if (kind == 0) sweep_warp<Real, 8, N8, TRACE>(d, base, pl.kstride[0], 8 * N8, chain0, chain_end, delay, t0, n_sweeps);
  else if (kind == 1) sweep_warp<Real, 16, N16, TRACE>(d, base, pl.kstride[1], 16 * N16, chain0, chain_end, delay, t0, n_sweeps);
  else sweep_warp<Real, 32, N32, TRACE>(d, base, pl.kstride[2], 32 * N32, chain0, chain_end, delay, t0, n_sweeps);
}

// Seven chains per sub-partition as 4 x 8 lanes + 3 x 10 lanes (lanes 30, 31 of a 10-lane warp idle): the mapping of
// the throughput batch (4096 chains on 148 SMs, N = 100: 13 and 10 partner iterations, 104 and 100 slots).  A
// 10-lane warp pays where 10 ceil(N/10) is much closer to N than 8 ceil(N/8) (measured: N = 100 2077 against 2440
// cycles per step of 4 x 8 + 4 x 8; N = 55 and 64 no gain).  Warps 0..3 are the 8-lane warps, 4..7 the 10-lane ones;
// the chain counts per warp come from the launch descriptor (6 chains on a sub-partition: 4 + 2).
// The start delay of the 10-lane warps is passed as a run-time value (always 0): with a literal 0 the wait loop
// disappears from the code and the schedule ptxas then finds for the step loop is 6 % slower (measured twice).
// FULL: every sub-partition holds exactly 7 chains (28 per CTA) and the layout is fixed at compile time; otherwise
// first chain, number of chains and shared-memory offset of every warp come from the launch descriptor.  Same
// arithmetic; the fixed form is the one ptxas schedules best (measured, config 5: 2108 against 2232 cycles per step).
template <typename Real, int N8, int N10, bool TRACE, bool FULL>
__global__ void __launch_bounds__(256, 1) k_sweep_seven(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                     const int n_sweeps)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Real* base = reinterpret_cast<Real*>(smem_raw);
  const int warp = threadIdx.x >> 5;
  if (FULL) {
    const int cta0 = blockIdx.x * 28;
    if (warp < 4)
      sweep_warp<Real, 8, N8, TRACE>(d, base + (size_t)(warp * 4) * pl.kstride[0], pl.kstride[0], 8 * N8, cta0 + warp * 4,
                                     d.C, 0, t0, n_sweeps);
    else
      sweep_warp<Real, 10, N10, TRACE>(d, base + (size_t)16 * pl.kstride[0] + (size_t)((warp - 4) * 3) * pl.kstride[3],
                                       pl.kstride[3], 10 * N10, cta0 + 16 + (warp - 4) * 3, d.C, pl.stagger, t0, n_sweeps);
  } else {
    const int chain0 = blockIdx.x * pl.chains_per_cta + pl.wfirst[warp];
    const int chain_end = min(chain0 + pl.wcount[warp], (int)min((long long)d.C, (long long)(blockIdx.x + 1) * pl.chains_per_cta));
    if (chain0 >= chain_end) return;           // no chain for this warp
    if (warp < 4)
      sweep_warp<Real, 8, N8, TRACE>(d, base + pl.woff[warp], pl.kstride[0], 8 * N8, chain0, chain_end, 0, t0, n_sweeps);
    else
      sweep_warp<Real, 10, N10, TRACE>(d, base + pl.woff[warp], pl.kstride[3], 10 * N10, chain0, chain_end, pl.stagger, t0,
                                       n_sweeps);
  }
}

// ------------------------------------------------------------------------------------------
// CTA-per-replica kernel: blockDim.x threads share one chain (long chains, few replicas).
// ------------------------------------------------------------------------------------------
template <typename Real, bool TRACE>
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
  ctx_load(d, blockIdx.x, d.C, c);
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
      const Real wsum = group_sum<Real, 32>(part, lane, 0);
      if (lane == 0) red[k & 1][warp] = (double)wsum;
      const bool bond_broken = __syncthreads_or(broke ? 1 : 0) != 0;
      double dEd = red[k & 1][0];
      for (int q = 1; q < NW; ++q) dEd += red[k & 1][q];
      const Real dE = (Real)dEd;
      const double logu = s_logu[k & 1];

      const bool accept = !bond_broken && (dE <= (Real)0 || logu < nbeta * (double)dE);

      if (tid == 0) {
        if (accept) X.set(m, xn, yn, zn);
        if (TRACE) {   // test support (pt_set_trace): a separate instantiation
          if (d.tr_move && (long long)t < d.cap_sweeps)
            d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
        }
      }
      if (accept) { c.erun += (double)dE; c.acc++; }
      c.brej += bond_broken ? 1u : 0u;
      __syncthreads();
    }

    if (d.observables && warp == 0) measure_shape<Real, 32>(d, c, N, lane, 0, X);
    if (tid == 0) measure_energy(d, c, t);
  }

  __syncthreads();
  for (int j = tid; j < N; j += T) X.get(j, gx[j], gx[d.Ng + j], gx[2 * d.Ng + j]);
  if (tid == 0) ctx_store(d, c, n_sweeps);
}

}  // namespace
