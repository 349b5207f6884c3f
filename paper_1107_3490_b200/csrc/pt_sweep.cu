// Host side of the sweep kernels: which kernel and which mapping of chains to warps (pt_plan_sweep), and the
// launch.  The kernels themselves live in pt_sweep_kernels.cuh and are instantiated in pt_sweep_group.cu
// (uniform warps, one CTA per replica) and pt_sweep_comp<u>.cu (composed CTAs).  DESIGN.md section 7 has the
// measurements behind the rules.
#include <stdio.h>

#include "pt_internal.h"
#include "pt_sweep_classes.h"

// one lookup per translation unit of pt_sweep_classes.h
#define PT_DECL(u) PtSweepFn pt_lookup_comp_##u(int kind, const int nik[4], int precision, bool trace);
PT_DECL(0) PT_DECL(1) PT_DECL(2) PT_DECL(3) PT_DECL(4) PT_DECL(5) PT_DECL(6) PT_DECL(7)
#undef PT_DECL
static_assert(PT_COMP_UNITS == 8, "declare and call the lookup of every unit");

PtSweepFn pt_lookup_comp(int kind, const int nik[4], int precision, bool trace)
{
  PtSweepFn (*const units[])(int, const int*, int, bool) = {pt_lookup_comp_0, pt_lookup_comp_1, pt_lookup_comp_2,
                                                            pt_lookup_comp_3, pt_lookup_comp_4, pt_lookup_comp_5,
                                                            pt_lookup_comp_6, pt_lookup_comp_7};
  for (auto f : units)
    if (PtSweepFn k = f(kind, nik, precision, trace)) return k;
  return nullptr;
}

namespace {

// kinds of warp: lanes per chain and chain slots per warp
const int kLanesOfKind[4] = {8, 16, 32, 10};
const int kSlotsOfKind[4] = {4, 2, 1, 3};

int round_up(int a, int b) { return (a + b - 1) / b * b; }

constexpr int kSmemCap = 200 * 1024;   // dynamic shared memory any sweep kernel may ask for

// Chains of one warp must start in different banks: stride = L (mod Q) words, where Q words span all 32
// banks (fp64: a warp's 8-byte loads go in two phases of 16 lanes, Q = 16).
int chain_stride(int Ns, int L, int real_bytes)
{
  const int Q = 128 / real_bytes;
  // fp32 unrolled kernels read 8-byte pairs: two groups of 8 (10) lanes share a 128-byte phase when the second
  // starts 64 (80) bytes after the first
  const int want = real_bytes == 4 ? (L == 8 ? 16 : (L == 10 ? 20 : L % Q)) : L % Q;
  int ss = 3 * Ns;
  while (ss % Q != want) ++ss;
  return ss;
}

// table slots per coordinate array of an unrolled kernel: L lanes x ni iterations; the fp32 kernels take two partners
// per lane and iteration (pair_group_f2), i.e. an even number of iterations
int table_slots(int L, int ni, int real_bytes) { return real_bytes == 4 ? 2 * L * ((ni + 1) / 2) : L * ni; }

// phase stagger between two warps of the same kind on one sub-partition: about the fp64 time of one partner loop
int stagger_cycles(int ni) { return (int)(2.1 * (26.0 * ni + 70.0)); }

PtSweepFn kernel_of(const PtLaunch& pl, int precision, bool trace)
{
  if (pl.kind == PT_K_CTA) return pt_lookup_cta(precision, trace);
  if (pl.kind == PT_K_WS) return pt_lookup_ws(pl.lanes / 32, pl.ni, precision, trace);
  if (pl.kind == PT_K_WSG) return pt_lookup_wsg(pl.chains_per_cta, pl.ni, precision, trace);
  if (pl.kind == PT_K_COMP || pl.kind == PT_K_SEVEN || pl.kind == PT_K_SEVEN_FULL)
    return pt_lookup_comp(pl.kind, pl.nik, precision, trace);
  return pt_lookup_group(pl.lanes, pl.ni, precision, trace);
}

struct WarpSpec { int kind, count; };   // kind < 0: no warp

// k_sweep_comp: the (at most) two warps of a sub-partition that holds `load` chains; a second candidate for
// three chains (2 x 16 + 1 x 32 lanes instead of 3 of 4 x 8), chosen by the cost model below
const WarpSpec kCompWarps[9][2] = {{{-1, 0}, {-1, 0}}, {{2, 1}, {-1, 0}}, {{1, 2}, {-1, 0}}, {{0, 3}, {-1, 0}},
                                   {{0, 4}, {-1, 0}},  {{0, 4}, {2, 1}},  {{0, 4}, {1, 2}},  {{0, 4}, {0, 3}},
                                   {{0, 4}, {0, 4}}};
const WarpSpec kThreeAlt[2] = {{1, 2}, {2, 1}};

// Cost model of one sub-partition, in cycles per step (fit to profiles/r02_paper_timing.md): a warp issues about
// 60 slots per partner iteration (26 fp64 instructions that take the fp64 pipe for two cycles each, 10 others) and
// 280 for the serial part of the step; one warp alone on a sub-partition is latency-bound (x 1.35), two warps share
// the issue port (x 1.08 of the sum).
double warp_issue(int ni) { return 60.0 * ni + 280.0; }
double subpartition_cost(const WarpSpec w[2], const int nik[4])
{
  if (w[0].kind < 0) return 0.0;
  if (w[1].kind < 0 || w[1].count == 0) return 1.35 * warp_issue(nik[w[0].kind]);
  return 1.08 * (warp_issue(nik[w[0].kind]) + warp_issue(nik[w[1].kind]));
}

const WarpSpec* comp_warps(int load, const int nik[4])
{
  if (load == 3 && subpartition_cost(kThreeAlt, nik) < subpartition_cost(kCompWarps[3], nik)) return kThreeAlt;
  return kCompWarps[load];
}

// Composed CTAs (k_sweep_comp, k_sweep_seven): chains spread evenly over the SMs, one CTA per SM and wave, every
// sub-partition one or two warps chosen for its load.  Returns false if this shape is not covered.
bool plan_comp(const PtDev& d, int precision, int real_bytes, int sms, PtLaunch* out)
{
  if (d.N < 17 || d.N > 128) return false;
  PtLaunch pl{};
  const long long cap = 32ll * sms;                       // 8 chains per sub-partition: two warps of 4
  const long long waves = (d.C + cap - 1) / cap;
  const int q = (int)((d.C + sms * waves - 1) / (sms * waves));   // chains per CTA
  const int nc = (d.N + 7) / 8;
  pl.nik[0] = nc; pl.nik[1] = (nc + 1) / 2; pl.nik[2] = (nc + 3) / 4; pl.nik[3] = (d.N + 9) / 10;
  pl.kind = PT_K_COMP;
  // the seven-chain layout (4 x 8 + up to 3 x 10 lanes) where it is instantiated for this N and predicted faster
  if (q > 16 && q <= 28) {
    PtLaunch probe = pl;
    probe.kind = PT_K_SEVEN;
    if (kernel_of(probe, precision, false)) {
      double cost_comp = 0.0, cost_seven = 0.0;
      for (int sp = 0; sp < 4; ++sp) {
        const int load = q / 4 + (sp < q % 4 ? 1 : 0);
        const WarpSpec sv[2] = {{0, load < 4 ? load : 4}, {load > 4 ? 3 : -1, load > 4 ? load - 4 : 0}};
        const double a = subpartition_cost(comp_warps(load, pl.nik), pl.nik), b = subpartition_cost(sv, pl.nik);
        if (a > cost_comp) cost_comp = a;
        if (b > cost_seven) cost_seven = b;
      }
      if (cost_seven < cost_comp) pl.kind = q == 28 ? PT_K_SEVEN_FULL : PT_K_SEVEN;
    }
  }
  pl.chains_per_cta = q;
  pl.grid = (int)((d.C + q - 1) / q);
  for (int k = 0; k < 4; ++k)
    pl.kstride[k] = chain_stride(table_slots(kLanesOfKind[k], pl.nik[k], real_bytes), kLanesOfKind[k], real_bytes);
  int first = 0, off = 0, nwarps = 4, lanes_min = 32;
  for (int w = 0; w < 8; ++w) {
    const int sp = w & 3, load = q / 4 + (sp < q % 4 ? 1 : 0), r = w >> 2;
    WarpSpec ws = comp_warps(load, pl.nik)[r];
    if (pl.kind != PT_K_COMP) ws = r == 0 ? WarpSpec{0, load < 4 ? load : 4} : WarpSpec{3, load > 4 ? load - 4 : 0};
    pl.wkind[w] = ws.kind < 0 ? 2 : ws.kind;
    pl.wfirst[w] = first;
    pl.wcount[w] = ws.kind < 0 ? 0 : ws.count;
    pl.woff[w] = off;
    if (ws.kind < 0 || ws.count == 0) continue;
    if (r == 1) nwarps = 8;
    pl.wdelay[w] = (r == 1 && comp_warps(load, pl.nik)[0].kind == ws.kind && pl.kind == PT_K_COMP) ? stagger_cycles(pl.nik[ws.kind]) : 0;
    first += ws.count;
    off += kSlotsOfKind[ws.kind] * pl.kstride[ws.kind];
    if (kLanesOfKind[ws.kind] < lanes_min) lanes_min = kLanesOfKind[ws.kind];
  }
  if (first != q) return false;
  if (pl.kind != PT_K_COMP) nwarps = 8;
  pl.lanes = lanes_min;
  pl.ni = pl.nik[0];
  pl.Ns = 8 * pl.nik[0];
  pl.threads = 32 * nwarps;
  pl.smem_bytes = off * real_bytes;
  if (!kernel_of(pl, precision, false)) return false;
  *out = pl;
  return true;
}

// Warp-specialised CTA per chain (k_sweep_ws): P pair warps + two stream warps, every pair warp alone on its SM
// sub-partition (the stream warps are busy about half of the time and may share).  Sequential order only, N >= 5.
// P grows with the chain length (a partner iteration costs a pair warp about 60 cycles beside ~450 for load,
// reduce, barrier, decide; every further pair warp adds eight partial sums and a barrier participant), as far as
// the sub-partitions last.  Measured against one warp per chain on B200
// (fp64, N = 13 ... 480, 8 ... 592 chains): 1.2x - 1.85x up to 148 chains, 1.05x - 1.2x up to ~400.
bool plan_ws(const PtDev& d, int precision, int real_bytes, long long smsp, PtLaunch* out)
{
  if (d.select_mode != PT_SEQUENTIAL || d.N < 6) return false;   // three stream warps read m - 1 .. m + 1 beside commits of m - 4 .. m - 2
  // measured on B200 (fp64, us per step at 128 chains): one pair warp 0.25 - 0.29 up to N = 128, two 0.30 - 0.36 up to
  // N = 320 (three there: 0.36 - 0.40), three 0.43 beyond (two: 0.47); N = 481 ... 1920: 0.49 - 0.93 (k_sweep_cta: 0.98 - 1.65)
  for (int P = d.N > 320 ? 3 : (d.N > 128 ? 2 : 1); P >= 1; --P) {
    if (2ll * d.C * P + d.C > 2 * smsp) continue;   // a stream warp is busy about half of the time
    const int T = 32 * P;
    const int ni = pt_ws_variant(P, (d.N + T - 1) / T);
    if (ni < 0) continue;
    PtLaunch pl{};
    pl.kind = PT_K_WS;
    pl.lanes = T;
    pl.ni = ni;
    pl.Ns = table_slots(T, ni, real_bytes);
    pl.sstride = 3 * pl.Ns;
    pl.threads = 32 * (P + pt_ws_stream_warps(P, ni));
    pl.chains_per_cta = 1;
    pl.grid = d.C;
    pl.smem_bytes = pl.sstride * real_bytes;
    if (!kernel_of(pl, precision, false)) continue;
    *out = pl;
    return true;
  }
  return false;
}

// Several chains per CTA with shared stream warps (k_sweep_wsg): G = 4 chains, one pair warp each, three stream warps.
bool plan_wsg(const PtDev& d, int precision, int real_bytes, PtLaunch* out)
{
  if (d.select_mode != PT_SEQUENTIAL || d.N < 6) return false;
  const int G = 4;
  const int ni = pt_wsg_variant(G, (d.N + 31) / 32);
  if (ni < 0) return false;
  PtLaunch pl{};
  pl.kind = PT_K_WSG;
  pl.lanes = 32;
  pl.ni = ni;
  pl.Ns = table_slots(32, ni, real_bytes);
  pl.sstride = 3 * pl.Ns;
  pl.threads = 32 * (G + 3);
  pl.chains_per_cta = G;
  pl.grid = (d.C + G - 1) / G;
  pl.smem_bytes = G * pl.sstride * real_bytes;
  if (!kernel_of(pl, precision, false)) return false;
  *out = pl;
  return true;
}

}  // namespace

cudaError_t pt_plan_sweep(const PtDev& d, int precision, int lanes_requested, PtLaunch* plan)
{
  const int real_bytes = precision == PT_F32 ? 4 : 8;
  int sms = 148;   // B200; the device is asked below
  {
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) {
      int v = 0;
      if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) sms = v;
    }
    cudaGetLastError();
  }
  const long long smsp = 4ll * sms;
  PtLaunch pl{};
  bool done = false;
  int L = lanes_requested;
  if (L == 0) {
    // More chains than SM sub-partitions: composed CTAs, chains spread evenly over the SMs (no staircase in
    // the number of replicas beyond the one of the most loaded sub-partition).
    // Short chains in batches just beyond the range of a CTA per chain: four chains per CTA with shared stream warps
    // (measured, B200 fp64, us per step: N <= 64 at 395 ... 592 chains 0.31 - 0.32 against 0.375 - 0.385 with one warp per
    // chain, N = 100 0.397 against 0.408; N <= 32 at 593 ... 1184 chains 0.39 against 0.43 - 0.44 composed; longer chains
    // and larger batches lose; two chains per CTA never beat k_sweep_ws)
    const int ni32 = (d.N + 31) / 32;
    if ((long long)d.C > smsp && (long long)d.C <= 2 * smsp && ni32 == 1) done = plan_wsg(d, precision, real_bytes, &pl);
    if (!done && (long long)d.C > smsp) done = plan_comp(d, precision, real_bytes, sms, &pl);
    // Few chains: a step is as long as its dependence chain; a second warp takes the bond stream off it.
    if (!done) done = plan_ws(d, precision, real_bytes, smsp, &pl);
    if (!done && (long long)d.C <= smsp && ni32 <= 4) done = plan_wsg(d, precision, real_bytes, &pl);
    if (!done) {
      // Few very long chains: one CTA per replica.  Otherwise the most lanes per chain (shortest partner
      // loop) that still leave every warp alone on its SM sub-partition; a second warp on a
      // sub-partition costs more than halving the lanes (measured: profiles/r01_paper_timing.md).  With more
      // than 4 chains per sub-partition there is no such choice: 8 lanes, the serial part of a step
      // (proposal, bonds, log u, decision) is then one instruction stream shared by 4 chains.
      if (d.N > 15 * 32 && (long long)d.C <= smsp) L = 128;   // beyond the unrolled one-warp variants (15 iterations)
      else {
        L = 32;
        while (L > 8 && ((long long)d.C * L + 31) / 32 > smsp && d.N > L / 2) L /= 2;
        while (L > 8 && L / 2 >= d.N) L /= 2;
      }
    }
  }
  if (done) {
  } else if (L <= 32) {
    const int G = 32 / L;
    const int ni = pt_group_variant(L, (d.N + L - 1) / L);
    if (ni < 0) return cudaErrorInvalidValue;
    pl.lanes = L;
    pl.kind = PT_K_GROUP;
    pl.ni = ni;
    pl.Ns = ni > 0 ? table_slots(L, ni, real_bytes) : round_up(d.N, L);
    pl.sstride = chain_stride(pl.Ns, L, real_bytes);
    // one CTA per SM when there are enough warps (its warps are dealt round-robin to the four
    // sub-partitions, so they are balanced by construction); single-warp CTAs otherwise
    const long long warps = ((long long)d.C + G - 1) / G;
    int wpc = 1;
    if (warps > sms) {
      wpc = (int)((warps + sms - 1) / sms);
      if (wpc > 8) wpc = 8;
    }
    pl.threads = 32 * wpc;
    pl.chains_per_cta = G * wpc;
    pl.stagger = wpc > 4 ? stagger_cycles(pl.Ns / L) : 0;
    pl.grid = (int)((d.C + pl.chains_per_cta - 1) / pl.chains_per_cta);
    pl.smem_bytes = pl.chains_per_cta * pl.sstride * real_bytes;
  } else {
    pl.lanes = L;
    pl.kind = PT_K_CTA;
    pl.ni = 0;
    pl.Ns = round_up(d.N, L);
    pl.sstride = 3 * pl.Ns;
    pl.threads = L;
    pl.chains_per_cta = 1;
    pl.grid = d.C;
    pl.smem_bytes = pl.sstride * real_bytes;
  }
  if (pl.smem_bytes > kSmemCap) return cudaErrorInvalidValue;
  for (int trace = 0; trace < 2; ++trace) {
    PtSweepFn fn = kernel_of(pl, precision, trace != 0);
    if (!fn) return cudaErrorInvalidValue;
    if (pl.smem_bytes > 48 * 1024) {
      // the attribute belongs to the kernel, not to the handle: always the same cap, so that two live
      // handles that share an instantiation cannot lower each other's limit
      cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemCap);
      if (e != cudaSuccess) return e;
    }
  }
  *plan = pl;
  return cudaSuccess;
}

void pt_sweep_kernel_desc(const PtLaunch& pl, int precision, bool trace, char* buf, size_t n)
{
  const char* real = precision == PT_F32 ? "float" : "double";
  if (pl.kind == PT_K_CTA) snprintf(buf, n, "k_sweep_cta<%s,threads=%d,trace=%d>", real, pl.threads, trace ? 1 : 0);
  else if (pl.kind == PT_K_WSG) snprintf(buf, n, "k_sweep_wsg<%s,%d,chains=%d,trace=%d>", real, pl.ni, pl.chains_per_cta, trace ? 1 : 0);
  else if (pl.kind == PT_K_WS) snprintf(buf, n, "k_sweep_ws<%s,%d,%d,trace=%d>", real, pl.lanes / 32, pl.ni, trace ? 1 : 0);
  else if (pl.kind == PT_K_SEVEN || pl.kind == PT_K_SEVEN_FULL)
    snprintf(buf, n, "k_sweep_seven<%s,%d,%d,%s,trace=%d>", real, pl.nik[0], pl.nik[3],
             pl.kind == PT_K_SEVEN_FULL ? "full" : "partial", trace ? 1 : 0);
  else if (pl.kind == PT_K_COMP)
    snprintf(buf, n, "k_sweep_comp<%s,%d,%d,%d,trace=%d>", real, pl.nik[0], pl.nik[1], pl.nik[2], trace ? 1 : 0);
  else snprintf(buf, n, "k_sweep_group<%s,%d,%d,trace=%d>", real, pl.lanes, pl.ni, trace ? 1 : 0);
}

cudaError_t pt_launch_sweep(const PtDev& d, int precision, const PtLaunch& pl, uint32_t t0, int n_sweeps,
                            cudaStream_t stream)
{
  PtSweepFn fn = kernel_of(pl, precision, d.tr_move != nullptr);
  if (!fn) return cudaErrorInvalidValue;
  if (n_sweeps <= 0) return cudaSuccess;
  fn<<<dim3(pl.grid), dim3(pl.threads), pl.smem_bytes, stream>>>(d, pl, t0, n_sweeps);
  return cudaGetLastError();
}
