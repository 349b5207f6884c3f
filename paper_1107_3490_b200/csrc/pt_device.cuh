// Device-side arithmetic of the method: random stream, proposal maps, potentials.
// Written from the paper's equations; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pt_internal.h"

#define PT_TAG_MOVE 0u
#define PT_TAG_PICK 1u
#define PT_TAG_SWAP 2u

// ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 10 rounds of two 32x32->64 multiplies
// and a key schedule by Weyl constants.  Replaces the paper's host-made pool of uniforms, which
// the authors call the sub-optimal part of their design.
__device__ __forceinline__ uint4 pt_philox4x32_10(uint4 c, uint2 k)
{
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u;
    k.y += 0xBB67AE85u;
  }
  return c;
}

__device__ __forceinline__ uint4 pt_draw(uint2 key, uint32_t a, uint32_t b, uint32_t e, uint32_t tag,
                                         uint32_t i)
{
  return pt_philox4x32_10(make_uint4(a, b, e, (tag << 24) | i), key);
}

// 2/(2k+3), k = 0..9: the odd series of log m = 2 atanh(s) after factoring out 2 s (PtNum<double>::log_)
__constant__ double kPtLogC[10] = {2.0 / 3.0,  2.0 / 5.0,  2.0 / 7.0,  2.0 / 9.0,  2.0 / 11.0,
                                   2.0 / 13.0, 2.0 / 15.0, 2.0 / 17.0, 2.0 / 19.0, 2.0 / 21.0};

// ---- word -> number, proposal, reciprocal, cutoff test, per precision.
// Every random value is exactly representable, so the proposal is bit-reproducible.
template <typename Real> struct PtNum;

template <> struct PtNum<double> {
  // (2w + 1 - 2^32) / 2^32: odd numerators, symmetric about 0, never 0
  static __device__ __forceinline__ double sym(uint32_t w)
  {
    return (double)(2ll * (long long)w + 1ll - 4294967296ll) * (1.0 / 4294967296.0);
  }
  // (w + 1/2) / 2^32 in (0,1)
  static __device__ __forceinline__ double u01(uint32_t w)
  {
    return ((double)w + 0.5) * (1.0 / 4294967296.0);
  }
  // x' = x + d*s as two separately rounded operations (no FMA contraction)
  static __device__ __forceinline__ double propose(double x, double d, double s)
  {
    return __dadd_rn(x, __dmul_rn(d, s));
  }
  // the same in two calls: delta = scale(d, s), x' = shift(x, delta)
  static __device__ __forceinline__ double scale(double d, double s) { return __dmul_rn(d, s); }
  static __device__ __forceinline__ double shift(double x, double delta) { return __dadd_rn(x, delta); }
  // 1/d for finite d > 0: MUFU.RCP64H seed (relative error < 2^-19.9 measured on B200) and one
  // cubic Newton step x (1 + e + e^2), e = 1 - d x  ->  relative error e^3 < 2^-59 before the
  // final rounding; measured worst case 2 ulp.  3 fp64-pipe instructions instead of the ~9 of an
  // IEEE division.  d = 0 gives +inf, d = inf gives NaN (callers mask such pairs out).
  static __device__ __forceinline__ double rcp(double d)
  {
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
    const double e = fma(-d, x, 1.0);
    return fma(x, fma(e, e, e), x);
  }
  // the seed of rcp() alone, and whether it needs the Newton step
  static constexpr bool kNewton = true;
  static __device__ __forceinline__ double rcp_seed(double d)
  {
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
    return x;
  }
  // Reciprocal seed of r2 if (j != m and r2 < rc2), else +0; cnt += DELTA in the first case.  One
  // predicate from a DSETP (fp64 pipe; "j != m" is its predicate input) masks the seed and drives a
  // predicated add.  Written in PTX to keep that shape: ptxas emits MUFU.RCP64H + one FSEL on the seed's
  // high word (the low word of a seed is zero anyway), where C++ source gave two ISETP, SEL and a move.
  template <int DELTA>
  static __device__ __forceinline__ double seed_if_inside(double r2, double rc2, int j, int m, int& cnt)
  {
    double x;
    asm("{\n\t.reg .pred q, p;\n\t"
        "setp.ne.s32 q, %4, %5;\n\t"
        "setp.lt.and.f64 p, %2, %3, q;\n\t"
        "mov.f64 %0, 0d0000000000000000;\n\t"
        "@p rcp.approx.ftz.f64 %0, %2;\n\t"
        "@p add.s32 %1, %1, %6;\n\t}"
        : "=&d"(x), "+r"(cnt)
        : "d"(r2), "d"(rc2), "r"(j), "r"(m), "n"(DELTA));
    return x;
  }
  // r2 < rc2 for r2 >= 0 (or NaN), decided on the integer pipe: the bit patterns of non-negative
  // doubles are ordered like the numbers; NaN and anything with the sign bit set compare false.
  static __device__ __forceinline__ bool below(double r2, double rc2)
  {
    return (unsigned long long)__double_as_longlong(r2) < (unsigned long long)__double_as_longlong(rc2);
  }
  // v if keep, else a huge finite number (> 4e307 whatever the low word): beyond every cutoff, and
  // still finite after the few additions that follow.  One integer select on the high word.
  static __device__ __forceinline__ double keep_or_far(double v, bool keep)
  {
    return __hiloint2double(keep ? __double2hiint(v) : 0x7fe00000, __double2loint(v));
  }
  // inside ? 1/d : 0 -- the mask is applied to the seed (one integer select on its high word; a
  // zero seed stays zero through the Newton step), so that the sums need no select afterwards.
  static __device__ __forceinline__ double rcp_masked(double d, bool inside)
  {
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
    x = __hiloint2double(inside ? __double2hiint(x) : 0, __double2loint(x));
    const double e = fma(-d, x, 1.0);
    return fma(x, fma(e, e, e), x);
  }
  // sqrt(a) for a normal a > 0, branch-free so that it can be scheduled between the pair terms:
  // y = MUFU.RSQ64H seed (relative error eps < 2^-19), g = a y, r = (1 - a y^2)/2, and
  // sqrt(a) = g (1 - 2r)^(-1/2) = g (1 + r + 3/2 r^2 + O(r^3)); truncation < 2^-60.  a = 0 gives
  // NaN (callers treat NaN as "outside the FENE range").  6 fp64-pipe instructions.
  static __device__ __forceinline__ double sqrt_(double a)
  {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    const double g = a * y, h = 0.5 * y;
    const double r = fma(-h, g, 0.5);
    const double t = fma(1.5 * r, r, r);
    return fma(g, t, g);
  }
  // log(v) for a normal v > 0, branch-free.  v = 2^e m with m in [sqrt(1/2), sqrt(2)) by integer
  // arithmetic on the high word; log m = 2 atanh(s), s = (m - 1)/(m + 1), |s| < 0.1716, as the
  // odd Taylor series 2 s (1 + z/3 + z^2/5 + ... + z^10/21), z = s^2 (next term < 2^-60 relative);
  // log v = e ln2_hi + (e ln2_lo + log m).  No cancellation near v = 1 because e = 0 there.
  static __device__ __forceinline__ double log_(double v)
  {
    const int hi = __double2hiint(v);
    const int e = (hi - 0x3fe6a09e) >> 20;          // floor: high word of sqrt(1/2) is 0x3fe6a09e
    const double m = __hiloint2double(hi - (e << 20), __double2loint(v));
    const double f = m - 1.0;
    const double s = f * rcp(m + 1.0);
    const double z = s * s;
    // coefficients come from the constant bank as the DFMA's third operand (as immediates they cost
    // two UMOV per coefficient and step)
    double p = kPtLogC[9];
#pragma unroll
    for (int q = 8; q >= 0; --q) p = fma(p, z, kPtLogC[q]);
    const double logm = fma(s, p * z, s + s);
    const double de = (double)e;
    return fma(de, 0x1.62e42fefa39efp-1, fma(de, 0x1.abc9e3b39803fp-56, logm));
  }
};

template <> struct PtNum<float> {
  static __device__ __forceinline__ float sym(uint32_t w)
  {
    return (float)(2 * (int)(w >> 8) + 1 - 16777216) * (1.0f / 16777216.0f);
  }
  static __device__ __forceinline__ float u01(uint32_t w)
  {
    return ((float)(w >> 9) + 0.5f) * (1.0f / 8388608.0f);
  }
  static __device__ __forceinline__ float propose(float x, float d, float s)
  {
    return __fadd_rn(x, __fmul_rn(d, s));
  }
  static __device__ __forceinline__ float scale(float d, float s) { return __fmul_rn(d, s); }
  static __device__ __forceinline__ float shift(float x, float delta) { return __fadd_rn(x, delta); }
  static __device__ __forceinline__ float rcp(float d)
  {
    float x;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(x) : "f"(d));
    return x;
  }
  static constexpr bool kNewton = false;
  static __device__ __forceinline__ float rcp_seed(float d) { return rcp(d); }
  template <int DELTA>
  static __device__ __forceinline__ float seed_if_inside(float r2, float rc2, int j, int m, int& cnt)
  {
    const bool in = j != m && r2 < rc2;
    cnt += in ? DELTA : 0;
    return in ? rcp(r2) : 0.0f;
  }
  static __device__ __forceinline__ bool below(float r2, float rc2) { return r2 < rc2; }
  static __device__ __forceinline__ float keep_or_far(float v, bool keep)
  {
    return keep ? v : __int_as_float(0x7f000000);
  }
  static __device__ __forceinline__ float rcp_masked(float d, bool inside)
  {
    float x;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(x) : "f"(d));
    return inside ? x : 0.0f;
  }
  static __device__ __forceinline__ float sqrt_(float v) { return sqrtf(v); }
  // the paper's fp32 kernels use the fast-math intrinsics (__logf)
  static __device__ __forceinline__ float log_(float v) { return __logf(v); }
};

// ---- Eq. (1)-(2) as a function of r^2:
//   E_LJ^mod = 4 eps [(sigma/r)^12 - (sigma/r)^6] - E_LJ(r_c)  for r < r_c,  0 otherwise
//            = u (A u - B) - C,   u = 1/r^6,  A = 4 eps sigma^12,  B = 4 eps sigma^6,  C = E_LJ(r_c)
// The sums accumulate u (A u - B) with u = 0 for the pairs outside the cutoff, and count the pairs
// inside; the caller subtracts C * count once per sum.
// Section 3.3, Eq. (6): the swap test of the neighbour pair (i, i + 1) of ensemble e at exchange
// event x.  The temperature labels of the two slots are swapped; coordinates stay where they are.  Called by
// k_exchange (one thread per pair) and by the last CTA of an ensemble in k_sweep_ws (fused exchange).
__device__ __forceinline__ void pt_exchange_pair(const PtDev& d, int e, int i, uint32_t x)
{
  int* sot = d.slot_of_temp + (size_t)e * d.M;
  int* tos = d.temp_of_slot + (size_t)e * d.M;
  const int a = sot[i], b = sot[i + 1];
  const double Ea = d.erun[(size_t)e * d.M + a], Eb = d.erun[(size_t)e * d.M + b];
  const double delta = (d.beta[i] - d.beta[i + 1]) * (Ea - Eb);
  const uint4 w = pt_draw(d.keys[e], (uint32_t)i, x, (uint32_t)e, PT_TAG_SWAP, 0u);
  const double u = PtNum<double>::u01(w.x);
  const bool accept = (delta >= 0.0) ? true : (u < exp(delta));
  unsigned long long* sc = d.scount + ((size_t)e * (d.M - 1) + i) * 2;
  sc[0] += 1ull;
  if (accept) {
    sc[1] += 1ull;
    sot[i] = b; sot[i + 1] = a;
    tos[a] = i + 1; tos[b] = i;
  }
  if (d.tr_swap && (long long)x < d.cap_events)
    d.tr_swap[((size_t)e * d.cap_events + x) * (size_t)(d.M - 1) + i] = accept ? 2 : 1;
}

template <typename Real> struct PtLJ {
  Real A, nB, C, rc2, c, mhc;   // c = B / A = sigma^-6, mhc = -c / 2
  __device__ __forceinline__ explicit PtLJ(const PtDev& d)
      : A((Real)d.ljA), nB((Real)-d.ljB), C((Real)d.ljC), rc2((Real)d.rc2), c((Real)(d.ljB / d.ljA)),
        mhc((Real)(-0.5 * (d.ljB / d.ljA)))
  {
  }
  // acc += u (A u - B) for one squared distance; returns whether it lies inside the cutoff
  __device__ __forceinline__ bool add(Real r2, Real& acc) const
  {
    const bool inside = PtNum<Real>::below(r2, rc2);
    const Real inv = PtNum<Real>::rcp_masked(r2, inside);
    const Real u = inv * inv * inv;
    acc = fma(u, fma(A, u, nB), acc);
    return inside;
  }
};

template <typename Real> struct PtVec2;
template <> struct PtVec2<double> { typedef double2 type; };
template <> struct PtVec2<float> { typedef float2 type; };

// ---- packed fp32 pairs (sm_100a: add / mul / fma on two floats in one 64-bit register pair, SASS FADD2 / FMUL2 /
// FFMA2): the fp32 sweep kernels do the arithmetic of two adjacent partners with one instruction.
typedef unsigned long long PtF2;
__device__ __forceinline__ PtF2 pt_f2(float lo, float hi)
{
  PtF2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void pt_f2_split(PtF2 v, float& lo, float& hi)
{
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ PtF2 pt_add2(PtF2 a, PtF2 b)
{
  PtF2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ PtF2 pt_sub2(PtF2 a, PtF2 b)
{
  PtF2 r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ PtF2 pt_mul2(PtF2 a, PtF2 b)
{
  PtF2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ PtF2 pt_fma2(PtF2 a, PtF2 b, PtF2 c)
{
  PtF2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}

// One chain's coordinates in shared memory: (x, y) pairs in one array, z in another, so that a
// partner costs one 128-bit and one 64-bit load (fp64) with consecutive lanes on consecutive banks.
template <typename Real> struct PtCoords {
  typename PtVec2<Real>::type* xy;
  Real* z;
  __device__ __forceinline__ PtCoords(Real* base, int slots)
      : xy(reinterpret_cast<typename PtVec2<Real>::type*>(base)), z(base + 2 * (size_t)slots)
  {
  }
  __device__ __forceinline__ void get(int j, Real& x, Real& y, Real& zz) const
  {
    const typename PtVec2<Real>::type v = xy[j];
    x = v.x; y = v.y; zz = z[j];
  }
  __device__ __forceinline__ void set(int j, Real x, Real y, Real zz) const
  {
    typename PtVec2<Real>::type v;
    v.x = x; v.y = y;
    xy[j] = v;
    z[j] = zz;
  }
};

// fp32: three separate arrays x[], y[], z[], so that the coordinates of two adjacent monomers 2p, 2p+1 are one
// 64-bit load per component and arrive as packed pairs (get2).
template <> struct PtCoords<float> {
  float *x, *y, *z;
  __device__ __forceinline__ PtCoords(float* base, int slots) : x(base), y(base + slots), z(base + 2 * (size_t)slots) {}
  __device__ __forceinline__ void get(int j, float& xx, float& yy, float& zz) const { xx = x[j]; yy = y[j]; zz = z[j]; }
  __device__ __forceinline__ void set(int j, float xx, float yy, float zz) const { x[j] = xx; y[j] = yy; z[j] = zz; }
  __device__ __forceinline__ void get2(int p, PtF2& xx, PtF2& yy, PtF2& zz) const
  {
    xx = reinterpret_cast<const PtF2*>(x)[p];
    yy = reinterpret_cast<const PtF2*>(y)[p];
    zz = reinterpret_cast<const PtF2*>(z)[p];
  }
};
