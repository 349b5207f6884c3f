// Shared body of the pt_sweep_comp<u>.cu translation units: each defines PT_COMP_UNIT (its number) and
// PT_COMP_CLASSES (its list of PT_COMP / PT_SEVEN entries, pt_sweep_classes.h) before including this file.
#include "pt_sweep_kernels.cuh"

namespace {
struct CompVariant {
  int kind, a, b;             // PT_K_COMP: a = NC; PT_K_SEVEN, PT_K_SEVEN_FULL: a = N8, b = N10
  PtSweepFn f64[2], f32[2];   // [0] timed, [1] with the decision trace
};
#define PT_COMP(NC)                                                                            \
  { PT_K_COMP, NC, 0,                                                                          \
    { k_sweep_comp<double, NC, (NC + 1) / 2, (NC + 3) / 4, false>, k_sweep_comp<double, NC, (NC + 1) / 2, (NC + 3) / 4, true> }, \
    { k_sweep_comp<float, NC, (NC + 1) / 2, (NC + 3) / 4, false>, k_sweep_comp<float, NC, (NC + 1) / 2, (NC + 3) / 4, true> } },
#define PT_SEVEN(A, B)                                                                         \
  { PT_K_SEVEN, A, B, { k_sweep_seven<double, A, B, false, false>, k_sweep_seven<double, A, B, true, false> }, \
    { k_sweep_seven<float, A, B, false, false>, k_sweep_seven<float, A, B, true, false> } },         \
  { PT_K_SEVEN_FULL, A, B, { k_sweep_seven<double, A, B, false, true>, k_sweep_seven<double, A, B, true, true> }, \
    { k_sweep_seven<float, A, B, false, true>, k_sweep_seven<float, A, B, true, true> } },
const CompVariant kComp[] = { PT_COMP_CLASSES };
#undef PT_COMP
#undef PT_SEVEN
}  // namespace

#define PT_CAT2(a, b) a##b
#define PT_CAT(a, b) PT_CAT2(a, b)
// nik = iterations per kind (8, 16, 32, 10 lanes)
PtSweepFn PT_CAT(pt_lookup_comp_, PT_COMP_UNIT)(int kind, const int nik[4], int precision, bool trace)
{
  for (const CompVariant& v : kComp)
    if (v.kind == kind && v.a == nik[0] && (kind == PT_K_COMP || v.b == nik[3]))
      return precision == PT_F32 ? v.f32[trace ? 1 : 0] : v.f64[trace ? 1 : 0];
  return nullptr;
}
