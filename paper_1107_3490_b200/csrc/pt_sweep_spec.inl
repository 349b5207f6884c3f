// Speculative, software-pipelined sweep kernel (sequential monomer order, N >= 4).
// Included by pt_sweep_spec_f64.cu / pt_sweep_spec_f32.cu with PT_SPEC_REAL defined.
//
// Same method as k_sweep_group (Eq. 5), same mapping (L lanes
// per chain, 32/L chains per warp, coordinates in shared memory), different schedule.  The Markov
// chain is serial: step i+1 sees the conformation step i left.  But only ONE monomer can differ
// (p = the monomer step i tried to move), proposals never depend on decisions, and a counter-based
// generator gives any step's random numbers at any time.  So step i+1 is evaluated BEFORE step i is
// decided, for both outcomes:
//   - the pair terms against every partner j other than p do not depend on step i at all;
//   - the pair term against p is computed twice, for p at its old and at its proposed position, by
//     two otherwise idle lanes of the last partner iteration (slots Ns-2, Ns-1 are padding);
//   - a bond to p is likewise computed in both versions (two more roles of the bond stream);
//   - both candidate Delta E are reduced at once (even lanes carry "step i rejected", odd lanes
//     "step i accepted"), both Metropolis tests are made, and when the decision of step i arrives
//     it only selects one of two ready decisions.
// The loop-carried dependency is one predicate select; reduction, test, commit and reload of step i
// are in the same basic block as the pair arithmetic of step i+1 and the bond stream of step i+2,
// so the fp64 pipe always has independent work.  Results are bit-identical to the serial schedule
// except for summation order inside Delta E.
//
// Loop body i (finalises step i):
//   a. tail(i):   reduce the partials of step i, test, select with D(i-1) -> D(i)
//   b. pairs(i+1): partner loop of step i+1 (reads X: commits <= i-1 are visible; slot p = m(i) is
//                  masked and replaced by the two register versions)
//   c. bonds(i+2): proposal, bond terms (both versions of the bond to m(i+1)), log u of step i+2
//   d. Philox words of step i+3 (integer pipe)
//   e. commit(i):  X[m(i)] <- x' if D(i); __syncwarp
//   f. once per sweep: measurement
// N >= 4 guarantees that nothing read in b, c is the slot that e is about to write, other than p.

namespace {

typedef PT_SPEC_REAL Real;

struct SpecStep {
  int m;
  Real xo, yo, zo, xn, yn, zn;
  Real bond_rej, bond_acc;   // this lane's bond addend if the previous step was rejected / accepted
  Real logu;                 // log of the acceptance uniform (group-uniform)
  bool brk_rej, brk_acc;     // a new bond leaves (r0-R, r0+R) in that version (group-uniform)
};

struct SpecPart {
  Real rej, acc;             // this lane's share of Delta E in the two versions
};

// c. of the header comment.  p = monomer of the previous step (-1: none), (pxn, pyn, pzn) = its
// proposed position; its old position is still in shared memory.
template <int L>
__device__ __forceinline__ SpecStep spec_bonds(const PtDev& d, const PtCoords<Real>& X, int N, int lig, unsigned gsh,
                                               Real width, int m, uint4 w, int p, Real pxn, Real pyn, Real pzn)
{
  SpecStep s;
  s.m = m;
  X.get(m, s.xo, s.yo, s.zo);
  s.xn = PtNum<Real>::propose(s.xo, width, PtNum<Real>::sym(w.x));
  s.yn = PtNum<Real>::propose(s.yo, width, PtNum<Real>::sym(w.y));
  s.zn = PtNum<Real>::propose(s.zo, width, PtNum<Real>::sym(w.z));
  const Real u = PtNum<Real>::u01(w.w);
  // roles: 0..3 = bonds (new m-1, new m+1, old m-1, old m+1) with the neighbour where shared memory
  // has it (= previous step rejected); 4 = log u; 5, 6 = (new, old) bond to p at its proposed position
  const int role = lig;
  const bool accrole = role == 5 || role == 6;
  const bool isnew = role == 0 || role == 1 || role == 5;
  const bool adj = p >= 0 && (p == m - 1 || p == m + 1);
  const int nb = accrole ? p : ((role & 1) ? m + 1 : m - 1);
  const bool isbond = accrole ? adj : (role < 4 && nb >= 0 && nb < N);
  const bool shared_p = !accrole && isbond && nb == p;
  Real xb, yb, zb;
  X.get((isbond && !accrole) ? nb : m, xb, yb, zb);
  if (accrole) { xb = pxn; yb = pyn; zb = pzn; }
  const Real dx = (isnew ? s.xn : s.xo) - xb;
  const Real dy = (isnew ? s.yn : s.yo) - yb;
  const Real dz = (isnew ? s.zn : s.zo) - zb;
  const Real r2 = isbond ? fma(dz, dz, fma(dy, dy, dx * dx)) : (Real)(d.r0 * d.r0);
  const Real r = PtNum<Real>::sqrt_(r2);
  const Real q = (r - (Real)d.r0) * (Real)d.invR;
  const Real gq = fma(-q, q, (Real)1);                 // 1 - ((r - r0)/R)^2, Eq. (3)
  const bool in_range = gq > (Real)0;                  // false for NaN as well
  const bool broke = isbond && isnew && !in_range;
  const Real lg = PtNum<Real>::log_(role == 4 ? u : ((isbond && in_range) ? gq : (Real)1));
  const Real val = (role == 4 || !isbond) ? (Real)0 : (isnew ? (Real)d.feneC : (Real)-d.feneC) * lg;
  s.bond_rej = accrole ? (Real)0 : val;
  s.bond_acc = shared_p ? (Real)0 : val;
  const unsigned grp = (L == 32 ? 0xffffffffu : ((1u << L) - 1u)) << gsh;
  s.brk_rej = (__ballot_sync(0xffffffffu, broke && !accrole) & grp) != 0u;
  s.brk_acc = (__ballot_sync(0xffffffffu, broke && !shared_p) & grp) != 0u;
  s.logu = __shfl_sync(0xffffffffu, lg, gsh + 4);
  return s;
}

// A3 for CNT partner iterations at once (iterations BEGIN .. BEGIN+CNT-1 of this lane), written stage
// by stage across the partners: every stage holds 2 CNT independent fp64 instructions, so a dependent
// instruction is never issued within the 8-cycle DFMA latency of its producer (ptxas keeps this
// order; partner-by-partner source gave a schedule with one chain in flight).  HAS_LAST: the group's
// last iteration is the loop's last one, whose lanes L-2 and L-1 (padding slots) take monomer p at
// its old / proposed position and which accumulates into its own sums (enl, eol).
template <int L, int BEGIN, int CNT, bool HAS_LAST>
__device__ __forceinline__ void spec_group(const PtLJ<Real>& lj, const PtCoords<Real>& X, int lig, int it0, int m, int p,
                                           Real pxo, Real pyo, Real pzo, Real pxn, Real pyn, Real pzn, Real xo, Real yo,
                                           Real zo, Real tdx, Real tdy, Real tdz, Real dd, Real (&en)[4], Real (&eo)[4],
                                           Real& enl, Real& eol)
{
  Real bx[CNT], by[CNT], bz[CNT], ro[CNT], rn[CNT];
  bool keep[CNT];
#pragma unroll
  for (int u = 0; u < CNT; ++u) {
    const int j = lig + (it0 + BEGIN + u) * L;
    X.get(j, bx[u], by[u], bz[u]);
    keep[u] = j != m && j != p;
  }
  if (HAS_LAST) {
    const bool sp_old = lig == L - 2, sp_new = lig == L - 1;
    bx[CNT - 1] = sp_old ? pxo : (sp_new ? pxn : bx[CNT - 1]);
    by[CNT - 1] = sp_old ? pyo : (sp_new ? pyn : by[CNT - 1]);
    bz[CNT - 1] = sp_old ? pzo : (sp_new ? pzn : bz[CNT - 1]);
    keep[CNT - 1] = (sp_old || sp_new) ? p >= 0 : keep[CNT - 1];
  }
#pragma unroll
  for (int u = 0; u < CNT; ++u) { bx[u] = xo - bx[u]; by[u] = yo - by[u]; bz[u] = zo - bz[u]; }
#pragma unroll
  for (int u = 0; u < CNT; ++u) ro[u] = bx[u] * bx[u];
#pragma unroll
  for (int u = 0; u < CNT; ++u) ro[u] = fma(by[u], by[u], ro[u]);
#pragma unroll
  for (int u = 0; u < CNT; ++u) ro[u] = fma(bz[u], bz[u], ro[u]);
#pragma unroll
  for (int u = 0; u < CNT; ++u) rn[u] = ro[u] + dd;
#pragma unroll
  for (int u = 0; u < CNT; ++u) rn[u] = fma(tdz, bz[u], rn[u]);
#pragma unroll
  for (int u = 0; u < CNT; ++u) rn[u] = fma(tdy, by[u], rn[u]);
#pragma unroll
  for (int u = 0; u < CNT; ++u) rn[u] = fma(tdx, bx[u], rn[u]);
  // Eq. (1): E_LJ(min(r, r_c)); masked partners evaluate at r_c as well
  Real dv[2 * CNT], xv[2 * CNT], ev[2 * CNT];
#pragma unroll
  for (int u = 0; u < CNT; ++u) {
    dv[2 * u] = PtNum<Real>::clamp_below(ro[u], lj.rc2, keep[u]);
    dv[2 * u + 1] = PtNum<Real>::clamp_below(rn[u], lj.rc2, keep[u]);
  }
#pragma unroll
  for (int v = 0; v < 2 * CNT; ++v) xv[v] = PtNum<Real>::rcp_seed(dv[v]);
  if (PtNum<Real>::kNewton) {
#pragma unroll
    for (int v = 0; v < 2 * CNT; ++v) ev[v] = fma(-dv[v], xv[v], (Real)1);
#pragma unroll
    for (int v = 0; v < 2 * CNT; ++v) ev[v] = fma(ev[v], ev[v], ev[v]);
#pragma unroll
    for (int v = 0; v < 2 * CNT; ++v) xv[v] = fma(xv[v], ev[v], xv[v]);
  }
#pragma unroll
  for (int v = 0; v < 2 * CNT; ++v) ev[v] = xv[v] * xv[v];
#pragma unroll
  for (int v = 0; v < 2 * CNT; ++v) xv[v] = ev[v] * xv[v];          // u = 1/r^6
#pragma unroll
  for (int v = 0; v < 2 * CNT; ++v) ev[v] = fma(lj.A, xv[v], lj.nB);
#pragma unroll
  for (int u = 0; u < CNT; ++u) {
    if (HAS_LAST && u == CNT - 1) {
      eol = fma(xv[2 * u], ev[2 * u], eol);
      enl = fma(xv[2 * u + 1], ev[2 * u + 1], enl);
    } else {
      eo[(BEGIN + u) & 3] = fma(xv[2 * u], ev[2 * u], eo[(BEGIN + u) & 3]);
      en[(BEGIN + u) & 3] = fma(xv[2 * u + 1], ev[2 * u + 1], en[(BEGIN + u) & 3]);
    }
  }
}

// b. of the header comment: the partner loop of step s, whose predecessor moved monomer p from
// (pxo, pyo, pzo) to (pxn, pyn, pzn) or not.
template <int L, int NI>
__device__ __forceinline__ SpecPart spec_pairs(const PtLJ<Real>& lj, const PtCoords<Real>& X, int lig, int nit,
                                               const SpecStep& s, int p, Real pxo, Real pyo, Real pzo, Real pxn,
                                               Real pyn, Real pzn)
{
  const Real ex = s.xn - s.xo, ey = s.yn - s.yo, ez = s.zn - s.zo;
  const Real dd = fma(ez, ez, fma(ey, ey, ex * ex));
  const Real tdx = ex + ex, tdy = ey + ey, tdz = ez + ez;
  Real en[4] = {(Real)0, (Real)0, (Real)0, (Real)0}, eo[4] = {(Real)0, (Real)0, (Real)0, (Real)0};
  Real enl = (Real)0, eol = (Real)0;
#define PT_GROUP(B, C, LASTF, IT0)                                                                             \
  spec_group<L, B, C, LASTF>(lj, X, lig, IT0, s.m, p, pxo, pyo, pzo, pxn, pyn, pzn, s.xo, s.yo, s.zo, tdx, tdy, \
                             tdz, dd, en, eo, enl, eol)
  if (NI > 0 && NI <= 7) {
    PT_GROUP(0, (NI > 0 && NI <= 7 ? NI : 1), true, 0);
  } else if (NI > 7 && NI <= 11) {
    PT_GROUP(0, 4, false, 0);
    PT_GROUP(4, (NI > 7 && NI <= 11 ? NI - 4 : 1), true, 0);
  } else if (NI > 11) {
    static_assert(NI <= 15, "add a group");
    PT_GROUP(0, 4, false, 0);
    PT_GROUP(4, 4, false, 0);
    PT_GROUP(8, (NI > 11 ? NI - 8 : 1), true, 0);
  } else {
    // run-time trip count: groups of 4, the rest (1..4 iterations, the last one special) by a uniform switch
    int it0 = 0;
    for (; it0 + 4 < nit; it0 += 4) PT_GROUP(0, 4, false, it0);
    switch (nit - it0) {
      case 1: PT_GROUP(0, 1, true, it0); break;
      case 2: PT_GROUP(0, 2, true, it0); break;
      case 3: PT_GROUP(0, 3, true, it0); break;
      default: PT_GROUP(0, 4, true, it0); break;
    }
  }
#undef PT_GROUP
  const bool sp_old = lig == L - 2, sp_new = lig == L - 1;
  const Real main = ((en[0] - eo[0]) + (en[1] - eo[1])) + ((en[2] - eo[2]) + (en[3] - eo[3]));
  const Real lastd = enl - eol;
  SpecPart r;
  r.rej = (main + (sp_new ? (Real)0 : lastd)) + s.bond_rej;
  r.acc = (main + (sp_old ? (Real)0 : lastd)) + s.bond_acc;
  return r;
}

__device__ __forceinline__ void spec_advance(int N, int& k, uint32_t& t)
{
  if (++k >= N) { k -= N; ++t; }
}

template <int L, int NI, bool TRACE>
__global__ void __launch_bounds__(256, 1) k_sweep_spec(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                    const int n_sweeps)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  static_assert(L >= 8 && L <= 32, "lanes per chain (roles 0..6 need 7 lanes)");
  constexpr int G = 32 / L;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane / L, lig = lane % L;
  const int cl = warp * G + g;
  const int N = d.N, Ns = pl.Ns;
  const int nit = NI > 0 ? NI : Ns / L;
  const unsigned gsh = (unsigned)(g * L);

  ChainCtx c;
  ctx_load(d, blockIdx.x * pl.chains_per_cta + cl, c);
  const Real width = (Real)d.width[c.i];
  const PtLJ<Real> lj(d);
  const PtCoords<Real> X(reinterpret_cast<Real*>(smem_raw) + (size_t)cl * pl.sstride, Ns);

  // A1: HBM -> shared memory; padding entries lie far outside every cutoff
  Real* gx = reinterpret_cast<Real*>(d.coords) + (size_t)c.s * 3 * d.Ng;
  for (int j = lig; j < Ns; j += L) {
    const bool in = j < N;
    X.set(j, in ? gx[j] : (Real)PT_FAR, in ? gx[d.Ng + j] : (Real)PT_FAR, in ? gx[2 * d.Ng + j] : (Real)PT_FAR);
  }
  __syncwarp();

  const bool leader = (lig == 0) && c.active;
  const bool odd = (lig & 1) != 0;
  const double nbeta = -c.beta;
  // running energy: even lanes add the Delta E of steps whose predecessor was rejected, odd lanes
  // of those whose predecessor was accepted; E_run = lane 0 + lane 1
  double erun_part = odd ? 0.0 : c.erun;
  const uint32_t e32 = (uint32_t)c.e, i32 = (uint32_t)c.i;

  // prologue: steps 0, 1 and the words of step 2
  int k = 0;
  uint32_t t = t0;
  int k1 = k, k2, k3;
  uint32_t t1 = t, t2, t3;
  spec_advance(N, k1, t1);
  k2 = k1; t2 = t1; spec_advance(N, k2, t2);
  k3 = k2; t3 = t2; spec_advance(N, k3, t3);
  SpecStep cur = spec_bonds<L>(d, X, N, lig, gsh, width, k, pt_draw(c.key, (uint32_t)k, t, e32, PT_TAG_MOVE, i32), -1,
                               (Real)PT_FAR, (Real)PT_FAR, (Real)PT_FAR);
  SpecPart part = spec_pairs<L, NI>(lj, X, lig, nit, cur, -1, (Real)PT_FAR, (Real)PT_FAR, (Real)PT_FAR,
                                    (Real)PT_FAR, (Real)PT_FAR, (Real)PT_FAR);
  SpecStep nxt = spec_bonds<L>(d, X, N, lig, gsh, width, k1, pt_draw(c.key, (uint32_t)k1, t1, e32, PT_TAG_MOVE, i32),
                               cur.m, cur.xn, cur.yn, cur.zn);
  uint4 w2 = pt_draw(c.key, (uint32_t)k2, t2, e32, PT_TAG_MOVE, i32);
  bool dprev = false;

  const int total = n_sweeps * N;
  for (int i = 0; i < total; ++i) {
    // a. tail(i): A4 for both versions at once, A6 for both, select
    const Real send = odd ? part.rej : part.acc, keepv = odd ? part.acc : part.rej;
    Real v = keepv + __shfl_xor_sync(0xffffffffu, send, 1);
#pragma unroll
    for (int o = 2; o < L; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const bool own_brk = odd ? cur.brk_acc : cur.brk_rej;
    const bool own_d = !own_brk && (v <= (Real)0 || (double)cur.logu < nbeta * (double)v);
    const unsigned bal = __ballot_sync(0xffffffffu, own_d);
    const bool accept = ((bal >> (gsh + (dprev ? 1u : 0u))) & 1u) != 0u;
    const bool broken = dprev ? cur.brk_acc : cur.brk_rej;
    if (accept && odd == dprev) erun_part += (double)v;
    c.acc += accept ? 1u : 0u;
    c.brej += broken ? 1u : 0u;

    // b. pairs(i+1)
    const SpecPart pnext = spec_pairs<L, NI>(lj, X, lig, nit, nxt, cur.m, cur.xo, cur.yo, cur.zo, cur.xn, cur.yn, cur.zn);
    // c. bonds(i+2)
    const SpecStep nn = spec_bonds<L>(d, X, N, lig, gsh, width, k2, w2, nxt.m, nxt.xn, nxt.yn, nxt.zn);
    // d. words of step i+3
    w2 = pt_draw(c.key, (uint32_t)k3, t3, e32, PT_TAG_MOVE, i32);

    // e. commit(i) (A7)
    if (lig == 0) {
      if (accept) X.set(cur.m, cur.xn, cur.yn, cur.zn);
      if (TRACE) {
        if (d.tr_move && c.active && (long long)t < d.cap_sweeps)
          d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
      }
    }
    __syncwarp();

    // f. A8 once per sweep
    if (k == N - 1) {
      if (d.observables) measure_shape<Real, L>(c, N, lig, X);
      c.erun = erun_part + __shfl_xor_sync(0xffffffffu, erun_part, 1);
      if (leader) measure_energy(d, c, t);
    }

    cur = nxt; nxt = nn; part = pnext; dprev = accept;
    k = k1; t = t1; k1 = k2; t1 = t2; k2 = k3; t2 = t3;
    spec_advance(N, k3, t3);
  }

  // A9: shared memory -> HBM
  __syncwarp();
  c.erun = erun_part + __shfl_xor_sync(0xffffffffu, erun_part, 1);
  if (c.active) {
    for (int j = lig; j < N; j += L) X.get(j, gx[j], gx[d.Ng + j], gx[2 * d.Ng + j]);
    if (lig == 0) ctx_store(d, c, n_sweeps);
  }
}

#define PT_SPEC_ROW(L, NI) { L, NI, k_sweep_spec<L, NI, false>, k_sweep_spec<L, NI, true> }
struct SpecVariant {
  int L, NI;
  PtSweepFn plain, trace;
};
// NI = 0 (run-time trip count) must come last within its L
const SpecVariant kSpec[] = {
    PT_SPEC_ROW(8, 2),  PT_SPEC_ROW(8, 4),  PT_SPEC_ROW(8, 7),  PT_SPEC_ROW(8, 10), PT_SPEC_ROW(8, 13), PT_SPEC_ROW(8, 0),
    PT_SPEC_ROW(16, 1), PT_SPEC_ROW(16, 2), PT_SPEC_ROW(16, 4), PT_SPEC_ROW(16, 7), PT_SPEC_ROW(16, 0),
    PT_SPEC_ROW(32, 1), PT_SPEC_ROW(32, 2), PT_SPEC_ROW(32, 4), PT_SPEC_ROW(32, 0),
};

}  // namespace
