// Warp-specialised sweep kernel for the latency-bound shapes: few chains (every pair warp alone on its SM
// sub-partition), sequential monomer order.  One CTA per chain:
//
//   warps 0 .. P-1   "pair warps"    A3 for their share of the partners (32 P threads stride over the table, the
//                                    unrolled stage-major groups of pt_sweep_kernels.cuh), two shuffle levels, eight
//                                    partial sums per warp into shared memory; after the step's barrier EVERY pair
//                                    thread adds the partials and the bond terms, decides (A6) and keeps the books;
//                                    the thread that owns the moved monomer's table slot commits (A7);
//   warps P .. P+SW-1 "stream warps" A2 (Philox, the proposed position), A5 (Eq. 3: sqrt and log of up to four bonds)
//                                    and log u, as plain serial code, warp P + s for the steps g = s (mod SW), AHEAD of
//                                    the pair warps and for both outcomes of the step in flight.  SW = 2, or 3 where one
//                                    pair warp with a short partner loop is faster than two streams can feed it.
//
// Why.  With one warp per chain (k_sweep_group) a step is as long as its dependence chain
//   commit -> load -> [pair stages | sqrt, log: ~30 dependent fp64 levels] -> reduce -> decide -> commit
// and the serial stream is the longest part of it (720-1270 cycles per step on BASELINE configs 1-4, of which the
// pair arithmetic needs 100-600).  Another warp can take the stream off that chain only if it does not wait for
// the decision.  In the sequential order it need not: the stream of step g (monomer m) depends on the steps before
// only through the position of m - 1, the monomer of step g - 1 and left bond neighbour of m, and that position is
// one of two known candidates.  Roles of a stream warp's lanes (bit 0: right neighbour, bit 1: old position of m,
// bit 2: step g - 1 rejected):
//   0  new bond (m, m-1), step g - 1 accepted      4  the same, rejected
//   2  old bond (m, m-1), accepted                 6  the same, rejected
//   1  new bond (m, m+1)     3  old bond (m, m+1)     5  log u
// "accepted" adds the displacement of step g - 1 to the table entry of m - 1, "rejected" reads the table entry,
// which holds the old position until the barrier of step g - 1.  Nothing that the steps before g - 1 decide enters,
// so a stream has SW steps' time, and SW warps take turns.  One shuffle level leaves b0 + b2, b1 + b3 and b4 + b6
// in lanes 0, 1, 4; they go to a ring of eight records in shared memory together with log u, the ballot of the
// broken new bonds and the proposed position (the pair warps draw no random numbers), and the deciders of step g
// pick the sums that belong to the outcome of step g - 1.
//
// Synchronisation: one named barrier per step (ids 1 .. SW in turn; all P + SW warps): the partial sums of the step
// are complete, and so is its record.  The stream warp of step g arrives at the barriers of the steps g - SW .. g - 2
// without waiting (bar.arrive) and waits at the barrier of step g - 1 (bar.sync); between two operations of a warp
// on the same id lies a wait that implies the earlier phase has completed, so an arrival is never counted for the
// wrong step.  No barrier is needed after the commit: a table slot is read in the pair loop
// by one thread only, its owner, and the owner is the thread that commits; a stream warp reads the slots m - 1,
// m, m + 1 while slots m - 2 .. m - SW - 1 may be committed (distinct for N >= 6); the moved monomer itself is
// read again N steps later.
// The paper's own mapping is one block per replica; this is that mapping with the block's warps
// given different work.  Random-pick mode, N < 6 and larger batches keep the other kernels (pt_plan_sweep).
// Measured (B200, fp64, moves/s): config 1 1.74e7 -> 2.5e7, config 2 8.22e7 -> 1.23e8, config 3 1.72e8 -> 2.58e8,
// config 4 2.14e8 -> 3.5e8 against one warp per chain.
#pragma once
#include "pt_sweep_kernels.cuh"

namespace {

// the pair groups' side stream is empty here
struct PtNoSide {
  static constexpr bool kShortChain = true;   // pair groups in the form with the shortest dependence chain
  template <int P, int NPTS, int LEVG> __device__ __forceinline__ void run() {}
};

__device__ __forceinline__ void pt_bar_sync(int id, int nthreads)
{
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void pt_bar_arrive(int id, int nthreads)
{
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// Ring of stream records, four deep, eight doubles each:
//   [0] b0 + b2 ("accepted" left bond terms)   [1] b1 + b3 (right bond terms)   [2] b4 + b6 ("rejected" left)
//   [3] log u     [4..6] the proposed position of the step's monomer (the pair warps draw no random numbers)
//   [7..10] 2 delta_x, 2 delta_y, 2 delta_z, |delta|^2 of the proposal (the terms of r_n^2 - r_o^2)
// and a mask per record: the ballot of broken NEW bonds (bits 0, 1, 4).
constexpr int kWsRec = 12;

// log(v), v normal and > 0: PtNum<double>::log_ with the series by Estrin's scheme (depth 4 instead of 10), the
// arithmetic of BondChain's levels 15..29
template <typename Real> __device__ __forceinline__ Real ws_log(Real v)
{
  if constexpr (sizeof(Real) == 8) {
    const int hi = __double2hiint(v);
    const int ex = (hi - 0x3fe6a09e) >> 20;
    const double mm = __hiloint2double(hi - (ex << 20), __double2loint(v));
    const double de = (double)ex;
    const double f = mm - 1.0, mp = mm + 1.0;
    double x = PtNum<double>::rcp_seed(mp);
    double e = fma(-mp, x, 1.0);
    e = fma(e, e, e);
    x = fma(x, e, x);
    const double sv = f * x;
    const double z = sv * sv, s2 = sv + sv;
    const double p01 = fma(kPtLogC[1], z, kPtLogC[0]), p23 = fma(kPtLogC[3], z, kPtLogC[2]);
    const double p45 = fma(kPtLogC[5], z, kPtLogC[4]), p67 = fma(kPtLogC[7], z, kPtLogC[6]);
    const double p89 = fma(kPtLogC[9], z, kPtLogC[8]), z2 = z * z;
    double q0 = fma(p23, z2, p01);
    const double q1 = fma(p67, z2, p45), z4 = z2 * z2;
    q0 = fma(q1, z4, q0);
    q0 = fma(p89, z4 * z4, q0);
    double lg = fma(sv, q0 * z, s2);
    lg = fma(de, 0x1.abc9e3b39803fp-56, lg);
    return fma(de, 0x1.62e42fefa39efp-1, lg);
  } else {
    return PtNum<float>::log_(v);
  }
}

// One pass of the stream for monomer m (old position xo.., proposed xn.., uniform u).  `ahead`: lanes 0 and 2
// take the left neighbour at its proposed position, table entry + (ex, ey, ez), instead of the table entry
// (the same separately rounded addition as the proposal itself, R7).  Returns what this lane stores
// into the record: lanes 0, 1, 4, 5 -> entries 0, 1, 2, 3; lanes 8..14 -> the proposed position and the terms of
// r_n^2 - r_o^2; *mask = ballot.
template <typename Real>
__device__ __forceinline__ double ws_stream(const PtDev& d, const PtCoords<Real>& X, int lane, int m, int N, Real xo, Real yo,
                                            Real zo, Real xn, Real yn, Real zn, Real u, bool ahead, Real ex, Real ey,
                                            Real ez, unsigned* mask)
{
  const int role = lane;
  const int nb = (role & 1) ? m + 1 : m - 1;
  const bool isbond = role < 7 && role != 5 && nb >= 0 && nb < N;
  const bool isnew = (role & 2) == 0;
  const bool moved = ahead && (role == 0 || role == 2);
  Real xb, yb, zb;
  X.get(isbond ? nb : m, xb, yb, zb);
  xb = PtNum<Real>::shift(xb, moved ? ex : (Real)0);
  yb = PtNum<Real>::shift(yb, moved ? ey : (Real)0);
  zb = PtNum<Real>::shift(zb, moved ? ez : (Real)0);
  const Real dx = (isnew ? xn : xo) - xb;
  const Real dy = (isnew ? yn : yo) - yb;
  const Real dz = (isnew ? zn : zo) - zb;
  const Real r2 = isbond ? fma(dz, dz, fma(dy, dy, dx * dx)) : (Real)(d.r0 * d.r0);
  const Real r = PtNum<Real>::sqrt_(r2);
  const Real q = (r - (Real)d.r0) * (Real)d.invR;
  const Real gq = fma(-q, q, (Real)1);              // 1 - ((r - r0)/R)^2, Eq. (3)
  const bool in_range = gq > (Real)0;               // false for NaN as well
  const bool broke = isbond && isnew && !in_range;
  const Real arg = role == 5 ? u : ((isbond && in_range) ? gq : (Real)1);
  const Real lg = ws_log<Real>(arg);
  const Real fc = isnew ? (Real)d.feneC : (Real)-d.feneC;   // -(K/2) R^2
  const Real bond = role != 5 ? fc * lg : (Real)0;
  const Real pairsum = bond + __shfl_xor_sync(0xffffffffu, bond, 2);
  *mask = __ballot_sync(0xffffffffu, broke);
  // what this lane stores, by selects (a nested conditional becomes a jump table)
  const Real px = xn - xo, py = yn - yo, pz = zn - zo;   // the displacement as a pair warp would compute it
  const Real pd = fma(pz, pz, fma(py, py, px * px));
  Real v = pairsum;
  v = lane == 5 ? lg : v;
  v = lane == 8 ? xn : v;
  v = lane == 9 ? yn : v;
  v = lane == 10 ? zn : v;
  v = lane == 11 ? px + px : v;
  v = lane == 12 ? py + py : v;
  v = lane == 13 ? pz + pz : v;
  v = lane == 14 ? pd : v;
  return (double)v;
}
// sum of n = 8, 16 or 24 numbers as a tree (depth 3, 4, 5)
template <int n> __device__ __forceinline__ double ws_tree(double* q)
{
  if constexpr (n == 1) return q[0];
  else if constexpr (n == 3) return (q[0] + q[1]) + q[2];
  else {
#pragma unroll
    for (int i = 0; i < n / 2; ++i) q[i] += q[i + n / 2];
    return ws_tree<n / 2>(q);
  }
}
// entry of the record that lane `lane` stores, or -1
__device__ __forceinline__ int ws_entry(int lane)
{
  int e = -1;
  e = lane == 0 ? 0 : e;
  e = lane == 1 ? 1 : e;
  e = lane == 4 ? 2 : e;
  e = lane == 5 ? 3 : e;
  e = (lane >= 8 && lane < 15) ? lane - 4 : e;
  return e;
}

// SW: stream warps (2 or 3); warp P + s takes the steps g = s (mod SW) and has SW steps' time for each.
template <typename Real, int P, int NI, bool TRACE, int SW>
__global__ void __launch_bounds__(32 * (P + SW), 1) k_sweep_ws(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                           const int n_sweeps)
{
  static_assert(P >= 1 && P <= 3 && NI >= 1, "pair warps and partner iterations");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int RING = 8;                  // records in flight: written up to SW steps ahead, read for one step
  __shared__ double s_rec[RING][kWsRec];  // ring of stream records
  __shared__ unsigned s_mask[RING];
  __shared__ double s_red[2][8 * P];       // eight partial pair sums per pair warp, double-buffered by step parity
  constexpr int T = 32 * P;                               // pair threads
  constexpr int NT = 32 * (P + SW);                       // + the stream warps
  static_assert(SW == 2 || SW == 3, "stream warps");
  constexpr bool F2 = sizeof(Real) == 4;                  // fp32: two partners per thread and iteration
  constexpr int NI2 = (NI + 1) / 2;
  constexpr int Ns = F2 ? 2 * T * NI2 : T * NI;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int N = d.N;
  const int total = n_sweeps * N;

  ChainCtx c;
  ctx_load(d, blockIdx.x, d.C, c);
  const Real width = (Real)d.width[c.i];
  const PtCoords<Real> X(reinterpret_cast<Real*>(smem_raw), Ns);

  // A1: HBM -> shared memory; padding entries lie far outside every cutoff
  Real* gx = reinterpret_cast<Real*>(d.coords) + (size_t)c.s * 3 * d.Ng;
  for (int j = tid; j < Ns; j += NT) {
    const bool in = j < N;
    X.set(j, in ? gx[j] : (Real)PT_FAR, in ? gx[d.Ng + j] : (Real)PT_FAR, in ? gx[2 * d.Ng + j] : (Real)PT_FAR);
  }
  __syncthreads();

  if (warp >= P) {
    // ---- stream warps: warp P + s takes the steps g = s (mod SW) ----
    // The stream of step g needs nothing that the steps before g - 1 decide (only the two candidates for the left
    // neighbour, the monomer of step g - 1), so it has SW steps' time: the warp arrives at the barriers of the steps
    // g - SW .. g - 2 without waiting and waits at the barrier of step g - 1, after which its record is complete.
    // SW barrier ids take turns, so an arrival can never be counted for the wrong step.
    const int s = warp - P;
    const int entry = ws_entry(lane);
    int blk_no = -1;
    DrawBlock<Real> blk;
    auto numbers = [&](int g) {   // the draw of step g (steps are asked for in increasing order)
      if ((g >> 3) != blk_no) {
        blk_no = g >> 3;
        blk = draw_block<Real>(c, false, N, width, t0, g & ~7, lane);
      }
      return draw_fetch<Real>(blk, g, 0u);
    };
    for (int g = s; g <= total; g += SW) {
      if (g >= SW) {                                                 // barriers of the steps g - SW .. g - 2
#pragma unroll
        for (int j = SW; j >= 2; --j) pt_bar_arrive(1 + (g - j) % SW, NT);
      }
      Real ex = (Real)0, ey = (Real)0, ez = (Real)0;
      if (g >= 1) { const DrawBlock<Real> pv = numbers(g - 1); ex = pv.dx; ey = pv.dy; ez = pv.dz; }
      const DrawBlock<Real> nx = numbers(g);
      Real xa, ya, za;
      X.get(nx.m, xa, ya, za);
      const Real xp = PtNum<Real>::shift(xa, nx.dx), yp = PtNum<Real>::shift(ya, nx.dy), zp = PtNum<Real>::shift(za, nx.dz);
      unsigned mask;
      const double val = ws_stream<Real>(d, X, lane, nx.m, N, xa, ya, za, xp, yp, zp, nx.u, g >= 1, ex, ey, ez, &mask);
      if (entry >= 0) s_rec[g & (RING - 1)][entry] = val;
      if (lane == 2) s_mask[g & (RING - 1)] = mask;
      if (g < SW) {
        __syncthreads();                                            // the records of the first SW steps precede the loop
        // the barriers of the steps before g: arrived at, the last one waited for -- between two operations of a warp
        // on one id there must be a wait that implies the earlier phase is complete, or an arrival is counted for the
        // wrong step
        for (int b = 0; b + 1 < g; ++b) pt_bar_arrive(1 + b % SW, NT);
        if (g >= 1) pt_bar_sync(1 + (g - 1) % SW, NT);
      } else {
        pt_bar_sync(1 + (g - 1) % SW, NT);                          // barrier of step g - 1
      }
    }
    // the loop ends with some g in total - SW + 1 .. total; the barriers of the steps from there on are still owed
    for (int b = total - (total - s) % SW; b < total; ++b) pt_bar_arrive(1 + b % SW, NT);
    return;
  }

  // ---- pair warps ----
  __syncthreads();
  const PtLJ<Real> lj(d);
  const double nbeta = -c.beta;
  PtNoSide noside;
  bool acc_prev = true;
  int g = 0;   // step number within the launch
  for (int sw = 0; sw < n_sweeps; ++sw) {
    const uint32_t t = t0 + (uint32_t)sw;
    for (int k = 0; k < N; ++k, ++g) {
      // A2 comes from the stream warp: the proposed position of monomer m = k is part of the step's record
      const int m = k;
      const int slot = g & (RING - 1);
      Real xo, yo, zo;
      X.get(m, xo, yo, zo);
      const Real xn = (Real)s_rec[slot][4], yn = (Real)s_rec[slot][5], zn = (Real)s_rec[slot][6];
      const Real tdx = (Real)s_rec[slot][7], tdy = (Real)s_rec[slot][8], tdz = (Real)s_rec[slot][9], dd = (Real)s_rec[slot][10];

      // A3: this thread's partners
      Real part;
      if constexpr (F2) part = pair_groups_f2<T, NI2, 1>(lj, X, tid, m, xo, yo, zo, tdx, tdy, tdz, dd, noside);
      else part = pair_groups<Real, T, NI, 1>(lj, X, tid, m, xo, yo, zo, tdx, tdy, tdz, dd, noside);
      // A4: two shuffle levels leave eight partial sums per warp; every decider adds all of them after the barrier
      // (three more shuffle levels would cost ~140 cycles of the step, the loads and adds ~60)
      part += __shfl_xor_sync(0xffffffffu, part, 16);
      part += __shfl_xor_sync(0xffffffffu, part, 8);
      if (lane < 8) s_red[g & 1][8 * warp + lane] = (double)part;
      pt_bar_sync(1 + g % SW, NT);   // partial sums and the stream record of this step are complete

      double q8[8 * P];
#pragma unroll
      for (int i = 0; i < 8 * P; ++i) q8[i] = s_red[g & 1][i];
      const double bonds = s_rec[slot][1] + (acc_prev ? s_rec[slot][0] : s_rec[slot][2]);
      const double logu = s_rec[slot][3];
      const bool bond_broken = (s_mask[slot] & (acc_prev ? 0x03u : 0x12u)) != 0u;
      const double pairs = ws_tree<8 * P>(q8);
      const Real dE = (Real)(pairs + bonds);

      // A6: Metropolis, Eq. (5): accept iff dE <= 0 or u < exp(-beta dE); NaN compares false
      const bool accept = !bond_broken && (dE <= (Real)0 || logu < nbeta * (double)dE);

      // A7: commit by the owner of the table slot (the only thread whose pair loop reads it)
      const int owner = F2 ? (m >> 1) % T : m % T;
      if (accept && tid == owner) X.set(m, xn, yn, zn);
      if (TRACE) {   // test support (pt_set_trace): a separate instantiation
        if (tid == 0 && d.tr_move && (long long)t < d.cap_sweeps)
          d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
      }
      c.erun += accept ? (double)dE : 0.0;
      c.acc += accept ? 1u : 0u;
      c.brej += bond_broken ? 1u : 0u;
      acc_prev = accept;
    }

    // A8: measurement once per sweep; the last commit may have come from another pair warp
    if (P > 1) pt_bar_sync(SW + 1, T);
    else __syncwarp();
    if (d.observables && warp == 0) measure_shape<Real, 32>(d, c, N, lane, 0, X);
    if (tid == 0) measure_energy(d, c, t);
  }

  // A9: shared memory -> HBM
  if (P > 1) pt_bar_sync(SW + 1, T);
  else __syncwarp();
  for (int j = tid; j < N; j += T) X.get(j, gx[j], gx[d.Ng + j], gx[2 * d.Ng + j]);
  if (tid == 0) ctx_store(d, c, n_sweeps);

  // B1 fused (pt_run): the exchange event that follows these sweeps is done by the CTA that is the last of its
  // ensemble to finish -- no exchange kernel and no launch gap, which are 4 us of an interval of 45 us on config 1.
  // Each CTA publishes its chain's running energy (fence), then counts itself; the one that counts M - 1 others
  // sees all of them and swaps the labels of its ensemble's neighbour pairs (Eq. 6), one thread per pair.
  if (pl.fuse_exchange) {
    __shared__ int s_last;
    __threadfence();
    if (P > 1) pt_bar_sync(SW + 1, T);
    else __syncwarp();
    if (tid == 0) {
      const unsigned before = atomicAdd(&d.done[c.e], 1u);
      s_last = before == (unsigned)(d.M - 1);
      if (s_last) d.done[c.e] = 0u;   // everyone of this ensemble has counted: ready for the next launch
    }
    if (P > 1) pt_bar_sync(SW + 1, T);
    else __syncwarp();
    if (s_last) {
      __threadfence();
      const uint32_t x = pl.x;
      const int npairs = (d.M - (int)(x & 1u)) / 2;
      for (int q = tid; q < npairs; q += T) pt_exchange_pair(d, c.e, (int)(x & 1u) + 2 * q, x);
    }
  }
}

}  // namespace
