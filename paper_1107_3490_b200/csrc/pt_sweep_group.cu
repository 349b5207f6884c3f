// k_sweep_group and k_sweep_cta instantiations: uniform warps (8, 16 or 32 lanes per chain), one CTA per replica.
#include "pt_sweep_kernels.cuh"

namespace {

struct SweepVariant {
  int L, NI;
  PtSweepFn f64[2], f32[2];   // [0] timed, [1] with the decision trace
};

#define PT_VARIANT(L, NI)                                                              \
  { L, NI, { k_sweep_group<double, L, NI, false>, k_sweep_group<double, L, NI, true> }, \
    { k_sweep_group<float, L, NI, false>, k_sweep_group<float, L, NI, true> } }
// Unrolled instantiations (NI = partner-loop iterations); NI = 0 is the run-time loop of the same
// lane count and must come last within its L.
const SweepVariant kVariants[] = {
    PT_VARIANT(8, 1),  PT_VARIANT(8, 2),  PT_VARIANT(8, 4),  PT_VARIANT(8, 7),  PT_VARIANT(8, 10), PT_VARIANT(8, 13),
    PT_VARIANT(8, 0),
    PT_VARIANT(16, 1), PT_VARIANT(16, 2), PT_VARIANT(16, 4), PT_VARIANT(16, 7), PT_VARIANT(16, 0),
    PT_VARIANT(32, 1), PT_VARIANT(32, 2), PT_VARIANT(32, 3), PT_VARIANT(32, 4), PT_VARIANT(32, 7), PT_VARIANT(32, 10),
    PT_VARIANT(32, 13), PT_VARIANT(32, 15), PT_VARIANT(32, 0),
};

}  // namespace

int pt_group_variant(int lanes, int ni_needed)
{
  for (const SweepVariant& v : kVariants)
    if (v.L == lanes && (v.NI == 0 || v.NI >= ni_needed)) return v.NI;
  return -1;
}

PtSweepFn pt_lookup_group(int lanes, int ni, int precision, bool trace)
{
  for (const SweepVariant& v : kVariants)
    if (v.L == lanes && v.NI == ni) return precision == PT_F32 ? v.f32[trace ? 1 : 0] : v.f64[trace ? 1 : 0];
  return nullptr;
}

PtSweepFn pt_lookup_cta(int precision, bool trace)
{
  if (precision == PT_F32) return trace ? (PtSweepFn)k_sweep_cta<float, true> : (PtSweepFn)k_sweep_cta<float, false>;
  return trace ? (PtSweepFn)k_sweep_cta<double, true> : (PtSweepFn)k_sweep_cta<double, false>;
}
