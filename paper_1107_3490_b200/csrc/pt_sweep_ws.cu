// k_sweep_ws instantiations: the warp-specialised kernel of the latency-bound shapes (pt_sweep_ws.cuh).
#include "pt_sweep_ws.cuh"

namespace {

struct WsVariant {
  int P, NI;                  // pair warps, partner iterations per pair thread (32 P NI table slots)
  PtSweepFn f64[2], f32[2];   // [0] timed, [1] with the decision trace
  int SW;                     // stream warps of these instantiations
};

#define PT_WS(P, NI, SW)                                                                    \
  { P, NI, { k_sweep_ws<double, P, NI, false, SW>, k_sweep_ws<double, P, NI, true, SW> },     \
    { k_sweep_ws<float, P, NI, false, SW>, k_sweep_ws<float, P, NI, true, SW> }, SW }
// One pair warp with a short partner loop is faster than two stream warps can feed it: three stream warps there
// (measured, B200 fp64: N = 30, 55, 100 7 % faster; two and three pair warps 2 - 10 % slower with three).
const WsVariant kWs[] = {
    PT_WS(1, 1, 3), PT_WS(1, 2, 3), PT_WS(1, 3, 3), PT_WS(1, 4, 3), PT_WS(1, 5, 3), PT_WS(1, 7, 3),
    PT_WS(1, 10, 2), PT_WS(1, 15, 2),
    PT_WS(2, 3, 2), PT_WS(2, 4, 2), PT_WS(2, 5, 2), PT_WS(2, 8, 2),
    PT_WS(3, 4, 2), PT_WS(3, 5, 2), PT_WS(3, 7, 2), PT_WS(3, 10, 2), PT_WS(3, 15, 2), PT_WS(3, 20, 2),
};

}  // namespace

// smallest instantiated NI >= ni_needed for P pair warps, or -1
int pt_ws_variant(int pair_warps, int ni_needed)
{
  for (const WsVariant& v : kWs)
    if (v.P == pair_warps && v.NI >= ni_needed) return v.NI;
  return -1;
}

int pt_ws_stream_warps(int pair_warps, int ni)
{
  for (const WsVariant& v : kWs)
    if (v.P == pair_warps && v.NI == ni) return v.SW;
  return 2;
}

PtSweepFn pt_lookup_ws(int pair_warps, int ni, int precision, bool trace)
{
  for (const WsVariant& v : kWs)
    if (v.P == pair_warps && v.NI == ni) return precision == PT_F32 ? v.f32[trace ? 1 : 0] : v.f64[trace ? 1 : 0];
  return nullptr;
}
