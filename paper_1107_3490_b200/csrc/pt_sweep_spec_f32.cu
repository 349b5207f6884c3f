// f32 instantiations of the speculative sweep kernel (pt_sweep_spec.inl).
#include "pt_sweep_common.cuh"

#define PT_SPEC_REAL float
#include "pt_sweep_spec.inl"

int pt_spec_find_f32(int L, int ni_needed)
{
  for (const SpecVariant& v : kSpec)
    if (v.L == L && (v.NI == 0 || v.NI >= ni_needed)) return v.NI;
  return -1;
}

PtSweepFn pt_spec_kernel_f32(int L, int NI, bool trace)
{
  for (const SpecVariant& v : kSpec)
    if (v.L == L && v.NI == NI) return trace ? v.trace : v.plain;
  return nullptr;
}
