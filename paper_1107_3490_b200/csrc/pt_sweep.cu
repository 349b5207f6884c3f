// Host side of the sweep kernels: which kernel and which mapping of chains to warps (pt_plan_sweep), and the
// launch.  The kernels themselves live in pt_sweep_kernels.cuh and are instantiated in pt_sweep_group.cu
// (uniform warps, one CTA per replica) and pt_sweep_comp<u>.cu (composed CTAs).  DESIGN.md section 7 has the
// measurements behind the rules.
#include <stdio.h>

#include "pt_internal.h"
#include "pt_sweep_classes.h"

// one lookup per translation unit of pt_sweep_classes.h
#define PT_DECL(u) PtSweepFn pt_lookup_comp_##u(const int nik[4], int precision, bool trace);
PT_DECL(0) PT_DECL(1) PT_DECL(2) PT_DECL(3) PT_DECL(4) PT_DECL(5) PT_DECL(6) PT_DECL(7)
#undef PT_DECL
static_assert(PT_COMP_UNITS == 8, "declare and call the lookup of every unit");

PtSweepFn pt_lookup_comp(const int nik[4], int precision, bool trace)
{
  PtSweepFn (*const units[])(const int*, int, bool) = {pt_lookup_comp_0, pt_lookup_comp_1, pt_lookup_comp_2,
                                                       pt_lookup_comp_3, pt_lookup_comp_4, pt_lookup_comp_5,
                                                       pt_lookup_comp_6, pt_lookup_comp_7};
  for (auto f : units)
    if (PtSweepFn k = f(nik, precision, trace)) return k;
  return nullptr;
}

namespace {

struct CompClass { int nik[4]; };
#define PT_COMP(A, B, C, D) {{A, B, C, D}},
#define PT_SEVEN(A, B) {{A, B, -1, -1}},
const CompClass kCompClasses[] = {PT_COMP_CLASSES_0 PT_COMP_CLASSES_1 PT_COMP_CLASSES_2 PT_COMP_CLASSES_3
                                  PT_COMP_CLASSES_4 PT_COMP_CLASSES_5 PT_COMP_CLASSES_6 PT_COMP_CLASSES_7};
#undef PT_COMP
#undef PT_SEVEN

const int kLanesOfKind[4] = {8, 10, 16, 32};
const int kChainsOfKind[4] = {4, 3, 2, 1};

int round_up(int a, int b) { return (a + b - 1) / b * b; }

constexpr int kSmemCap = 200 * 1024;   // dynamic shared memory any sweep kernel may ask for

// Chains of one warp must start in different banks: stride = L (mod Q) words, where Q words span all 32
// banks (fp64: a warp's 8-byte loads go in two phases of 16 lanes, Q = 16).
int chain_stride(int Ns, int L, int real_bytes)
{
  const int Q = 128 / real_bytes;
  int ss = 3 * Ns;
  while (ss % Q != L % Q) ++ss;
  return ss;
}

// phase stagger between two warps of the same kind on one sub-partition: about the fp64 time of one partner loop
int stagger_cycles(int ni) { return (int)(2.1 * (26.0 * ni + 70.0)); }

PtSweepFn kernel_of(const PtLaunch& pl, int precision, bool trace)
{
  if (pl.kind == PT_K_CTA) return pt_lookup_cta(precision, trace);
  if (pl.kind == PT_K_COMP) return pt_lookup_comp(pl.nik, precision, trace);
  return pt_lookup_group(pl.lanes, pl.ni, precision, trace);
}

// Composed CTAs (k_sweep_comp): chains spread evenly over the SMs, one CTA per SM and wave, every sub-partition
// one or two warps chosen for its load.  Returns false if this shape is not covered.
bool plan_comp(const PtDev& d, int real_bytes, int sms, PtLaunch* out)
{
  PtLaunch pl{};
  const long long cap = 32ll * sms;                       // 8 chains per sub-partition: two warps of 4
  const long long waves = (d.C + cap - 1) / cap;
  const int q = (int)((d.C + sms * waves - 1) / (sms * waves));   // chains per CTA
  // kinds of the (at most) two warps of a sub-partition that holds `load` chains; -1 = no warp
  static const int kWarps[9][2] = {{-1, -1}, {3, -1}, {2, -1}, {1, -1}, {0, -1}, {1, 2}, {1, 1}, {0, 1}, {0, 0}};
  if (!pt_comp_class(d.N, q == 28, pl.nik)) return false;
  pl.kind = PT_K_COMP;
  pl.chains_per_cta = q;
  pl.grid = (int)((d.C + q - 1) / q);
  for (int k = 0; k < 4; ++k)
    pl.kstride[k] = pl.nik[k] > 0 ? chain_stride(kLanesOfKind[k] * pl.nik[k], kLanesOfKind[k], real_bytes) : 0;
  int first = 0, off = 0, nwarps = 4, lanes_min = 32;
  for (int w = 0; w < 8; ++w) {
    const int sp = w & 3, load = q / 4 + (sp < q % 4 ? 1 : 0);
    const int k = kWarps[load][w >> 2];
    if (k < 0) {
      pl.wkind[w] = 3;
      pl.wfirst[w] = 1 << 30;        // beyond every chain: the warp leaves at once
      continue;
    }
    if (w >= 4) nwarps = 8;
    pl.wkind[w] = k;
    pl.wfirst[w] = first;
    pl.woff[w] = off;
    pl.wdelay[w] = (w >= 4 && kWarps[load][0] == k) ? stagger_cycles(pl.nik[k]) : 0;
    first += kChainsOfKind[k];
    off += kChainsOfKind[k] * pl.kstride[k];
    if (kLanesOfKind[k] < lanes_min) lanes_min = kLanesOfKind[k];
  }
  if (first != q) return false;
  pl.lanes = lanes_min;
  pl.ni = pl.nik[0];
  pl.Ns = 8 * pl.nik[0];
  pl.threads = 32 * nwarps;
  pl.smem_bytes = off * real_bytes;
  *out = pl;
  return true;
}

}  // namespace

bool pt_comp_class(int N, bool seven, int nik[4])
{
  if (N < 17) return false;
  const CompClass* best = nullptr;
  int best_waste = 0;
  for (const CompClass& c : kCompClasses) {
    const bool is_seven = c.nik[2] < 0;      // k_sweep_seven: exact fit only, and only for that composition
    bool ok = is_seven ? seven : true;
    int waste = is_seven ? -1 : 0;
    for (int k = 0; k < (is_seven ? 2 : 4); ++k) {
      const int need = (N + kLanesOfKind[k] - 1) / kLanesOfKind[k];
      ok = ok && (is_seven ? c.nik[k] == need : c.nik[k] >= need);
      waste += c.nik[k] - need;
    }
    if (ok && (!best || waste < best_waste)) { best = &c; best_waste = waste; }
  }
  if (!best) return false;
  for (int k = 0; k < 4; ++k) nik[k] = best->nik[k];
  return true;
}

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
    if ((long long)d.C > smsp) done = plan_comp(d, real_bytes, sms, &pl);
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
    pl.Ns = ni > 0 ? ni * L : round_up(d.N, L);
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
  else if (pl.kind == PT_K_COMP && pl.nik[2] < 0)
    snprintf(buf, n, "k_sweep_seven<%s,%d,%d,trace=%d>", real, pl.nik[0], pl.nik[1], trace ? 1 : 0);
  else if (pl.kind == PT_K_COMP)
    snprintf(buf, n, "k_sweep_comp<%s,%d,%d,%d,%d,trace=%d>", real, pl.nik[0], pl.nik[1], pl.nik[2], pl.nik[3], trace ? 1 : 0);
  else snprintf(buf, n, "k_sweep_group<%s,%d,%d,trace=%d>", real, pl.lanes, pl.ni, trace ? 1 : 0);
}

cudaError_t pt_launch_sweep(const PtDev& d, int precision, const PtLaunch& pl, uint32_t t0, int n_sweeps,
                            cudaStream_t stream)
{
  PtSweepFn fn = kernel_of(pl, precision, d.tr_move != nullptr);
  if (!fn) return cudaErrorInvalidValue;
  fn<<<dim3(pl.grid), dim3(pl.threads), pl.smem_bytes, stream>>>(d, pl, t0, n_sweeps);
  return cudaGetLastError();
}
