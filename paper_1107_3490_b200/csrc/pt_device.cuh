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

// ---- word -> number.  Every value is exactly representable, so the proposal is bit-reproducible.
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
  static __device__ __forceinline__ double rcp(double d)
  {
    // MUFU.RCP64H seed, then one cubic Newton step: x (1 + e + e^2), e = 1 - d x.
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
    const double e = fma(-d, x, 1.0);
    const double p = fma(e, e, e);
    const double y = fma(x, p, x);
    // second (quadratic) correction keeps the result within ~1 ulp whatever the seed quality
    const double e2 = fma(-d, y, 1.0);
    return fma(y, e2, y);
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
  static __device__ __forceinline__ float rcp(float d)
  {
    float x;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(x) : "f"(d));
    return x;
  }
};

// ---- Eq. (1)-(2) as a function of r^2:
//   E_LJ^mod = 4 eps [(sigma/r)^12 - (sigma/r)^6] - E_LJ(r_c)  for r < r_c,  0 otherwise
//            = u (A u - B) - C,   u = 1/r^6,  A = 4 eps sigma^12,  B = 4 eps sigma^6,  C = E_LJ(r_c)
// The caller applies the r < r_c selection.
template <typename Real> struct PtLJ {
  Real A, B, C, rc2;
  __device__ __forceinline__ explicit PtLJ(const PtDev& d)
      : A((Real)d.ljA), B((Real)d.ljB), C((Real)d.ljC), rc2((Real)d.rc2)
  {
  }
  __device__ __forceinline__ Real inside(Real r2) const
  {
    const Real inv = PtNum<Real>::rcp(r2);
    const Real u = inv * inv * inv;
    return fma(u, fma(A, u, -B), -C);
  }
};
