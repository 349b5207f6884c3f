// k_sweep_wsg instantiations: several chains per CTA with shared stream warps (pt_sweep_wsg.cuh).
#include "pt_sweep_wsg.cuh"

namespace {

struct WsgVariant {
  int G, NI;                  // chains per CTA, partner iterations per pair thread (32 NI table slots per chain)
  PtSweepFn f64[2], f32[2];   // [0] timed, [1] with the decision trace
};

#define PT_WSG(G, NI)                                                                  \
  { G, NI, { k_sweep_wsg<double, NI, false, G>, k_sweep_wsg<double, NI, true, G> },      \
    { k_sweep_wsg<float, NI, false, G>, k_sweep_wsg<float, NI, true, G> } }
const WsgVariant kWsg[] = {
    PT_WSG(4, 1), PT_WSG(4, 2), PT_WSG(4, 3), PT_WSG(4, 4),
};

}  // namespace

// smallest instantiated NI >= ni_needed for G chains per CTA, or -1
int pt_wsg_variant(int chains_per_cta, int ni_needed)
{
  for (const WsgVariant& v : kWsg)
    if (v.G == chains_per_cta && v.NI >= ni_needed) return v.NI;
  return -1;
}

PtSweepFn pt_lookup_wsg(int chains_per_cta, int ni, int precision, bool trace)
{
  for (const WsgVariant& v : kWsg)
    if (v.G == chains_per_cta && v.NI == ni) return precision == PT_F32 ? v.f32[trace ? 1 : 0] : v.f64[trace ? 1 : 0];
  return nullptr;
}
