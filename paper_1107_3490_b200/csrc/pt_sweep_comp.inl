// Shared body of the pt_sweep_comp<u>.cu translation units: each defines PT_COMP_UNIT (its number) and
// PT_COMP_CLASSES (its list of PT_COMP(N8, N10, N16, N32) entries, pt_sweep_classes.h) before including this file.
#include "pt_sweep_kernels.cuh"

namespace {
struct CompVariant {
  int nik[4];
  PtSweepFn f64[2], f32[2];   // [0] timed, [1] with the decision trace
};
#define PT_COMP(A, B, C, D)                                                                              \
  { {A, B, C, D}, { k_sweep_comp<double, A, B, C, D, false>, k_sweep_comp<double, A, B, C, D, true> },   \
    { k_sweep_comp<float, A, B, C, D, false>, k_sweep_comp<float, A, B, C, D, true> } },
// PT_SEVEN(A, B): k_sweep_seven, listed as the class (A, B, -1, -1)
#define PT_SEVEN(A, B)                                                                                   \
  { {A, B, -1, -1}, { k_sweep_seven<double, A, B, false>, k_sweep_seven<double, A, B, true> },           \
    { k_sweep_seven<float, A, B, false>, k_sweep_seven<float, A, B, true> } },
const CompVariant kComp[] = { PT_COMP_CLASSES };
#undef PT_COMP
#undef PT_SEVEN
}  // namespace

#define PT_CAT2(a, b) a##b
#define PT_CAT(a, b) PT_CAT2(a, b)
PtSweepFn PT_CAT(pt_lookup_comp_, PT_COMP_UNIT)(const int nik[4], int precision, bool trace)
{
  for (const CompVariant& v : kComp)
    if (v.nik[0] == nik[0] && v.nik[1] == nik[1] && v.nik[2] == nik[2] && v.nik[3] == nik[3])
      return precision == PT_F32 ? v.f32[trace ? 1 : 0] : v.f64[trace ? 1 : 0];
  return nullptr;
}
