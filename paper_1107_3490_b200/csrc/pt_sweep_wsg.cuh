// k_sweep_ws for several chains per CTA (k_sweep_wsg): G = 2 or 4 chains, one pair warp each, and three stream warps
// that serve all of them -- the stream of a chain needs seven lanes, so one pass of a stream warp (eight lanes per
// chain) does the streams of up to four chains with the same instructions.  For batches between the range of k_sweep_ws
// (a CTA per chain while the pair warps have sub-partitions of their own) and the throughput mappings: the pair warps of
// a CTA share sub-partitions with other warps there, but each of them is latency-bound and leaves most issue slots free.
// Everything else is pt_sweep_ws.cuh: roles, records, one named barrier per step for the whole CTA (the chains of a CTA
// step together), commit by the owner of the table slot, fused exchange.  Sequential order, N >= 6.
#pragma once
#include "pt_sweep_ws.cuh"

namespace {

template <typename Real, int NI, bool TRACE, int G>
__global__ void __launch_bounds__(32 * (G + 3), 1) k_sweep_wsg(const PtDev d, const PtLaunch pl, const uint32_t t0,
                                                            const int n_sweeps)
{
  static_assert(G == 2 || G == 4, "chains per CTA");
  constexpr int SW = 3;
  constexpr int RING = 8;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double s_rec[RING][G][kWsRec];
  __shared__ unsigned s_mask[RING][G];
  __shared__ double s_red[2][G][8];
  __shared__ int s_last[G];
  constexpr int NT = 32 * (G + SW);
  constexpr bool F2 = sizeof(Real) == 4;
  constexpr int NI2 = (NI + 1) / 2;
  constexpr int Ns = F2 ? 2 * 32 * NI2 : 32 * NI;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int N = d.N;
  const int total = n_sweeps * N;
  const int chain0 = blockIdx.x * G;

  // A1: HBM -> shared memory, all chains of the CTA (chains beyond the batch: clones of the last one, never stored)
  for (int cl = 0; cl < G; ++cl) {
    const int s = min(chain0 + cl, d.C - 1);
    const Real* gx = reinterpret_cast<const Real*>(d.coords) + (size_t)s * 3 * d.Ng;
    const PtCoords<Real> Xc(reinterpret_cast<Real*>(smem_raw) + (size_t)cl * 3 * Ns, Ns);
    for (int j = tid; j < Ns; j += NT) {
      const bool in = j < N;
      Xc.set(j, in ? gx[j] : (Real)PT_FAR, in ? gx[d.Ng + j] : (Real)PT_FAR, in ? gx[2 * d.Ng + j] : (Real)PT_FAR);
    }
  }
  __syncthreads();

  if (warp >= G) {
    // ---- stream warps: eight lanes per chain (roles 0..6 as in ws_stream), warp G + s takes the steps g = s (mod 3) ----
    const int s = warp - G;
    const int cl = min(lane >> 3, G - 1), role = (lane >> 3) < G ? (lane & 7) : 7;   // lanes beyond G chains idle along
    ChainCtx c;
    ctx_load(d, chain0 + cl, d.C, c);
    const Real width = (Real)d.width[c.i];
    const PtCoords<Real> X(reinterpret_cast<Real*>(smem_raw) + (size_t)cl * 3 * Ns, Ns);
    const unsigned gsh = (unsigned)(lane & ~7);
    int blk_no = -1;
    DrawBlock<Real> blk;
    auto numbers = [&](int g) {
      if ((g >> 3) != blk_no) {
        blk_no = g >> 3;
        blk = draw_block<Real>(c, false, N, width, t0, g & ~7, lane);
      }
      return draw_fetch<Real>(blk, g, gsh);
    };
    for (int g = s; g <= total; g += SW) {
      if (g >= SW) {
#pragma unroll
        for (int j = SW; j >= 2; --j) pt_bar_arrive(1 + (g - j) % SW, NT);
      }
      Real ex = (Real)0, ey = (Real)0, ez = (Real)0;
      if (g >= 1) { const DrawBlock<Real> pv = numbers(g - 1); ex = pv.dx; ey = pv.dy; ez = pv.dz; }
      const DrawBlock<Real> nx = numbers(g);
      Real xa, ya, za;
      X.get(nx.m, xa, ya, za);
      const Real xp = PtNum<Real>::shift(xa, nx.dx), yp = PtNum<Real>::shift(ya, nx.dy), zp = PtNum<Real>::shift(za, nx.dz);
      // the stream (ws_stream's arithmetic; the role is the lane within the chain's eight)
      const int m = nx.m;
      const int nb = (role & 1) ? m + 1 : m - 1;
      const bool isbond = role < 7 && role != 5 && nb >= 0 && nb < N;
      const bool isnew = (role & 2) == 0;
      const bool moved = g >= 1 && (role == 0 || role == 2);
      Real xb, yb, zb;
      X.get(isbond ? nb : m, xb, yb, zb);
      xb = PtNum<Real>::shift(xb, moved ? ex : (Real)0);
      yb = PtNum<Real>::shift(yb, moved ? ey : (Real)0);
      zb = PtNum<Real>::shift(zb, moved ? ez : (Real)0);
      const Real dx = (isnew ? xp : xa) - xb, dy = (isnew ? yp : ya) - yb, dz = (isnew ? zp : za) - zb;
      const Real r2 = isbond ? fma(dz, dz, fma(dy, dy, dx * dx)) : (Real)(d.r0 * d.r0);
      const Real r = PtNum<Real>::sqrt_(r2);
      const Real q = (r - (Real)d.r0) * (Real)d.invR;
      const Real gq = fma(-q, q, (Real)1);
      const bool in_range = gq > (Real)0;
      const bool broke = isbond && isnew && !in_range;
      const Real arg = role == 5 ? nx.u : ((isbond && in_range) ? gq : (Real)1);
      const Real lg = ws_log<Real>(arg);
      const Real fc = isnew ? (Real)d.feneC : (Real)-d.feneC;
      const Real bond = role != 5 ? fc * lg : (Real)0;
      const Real pairsum = bond + __shfl_xor_sync(0xffffffffu, bond, 2);
      const unsigned mask = (__ballot_sync(0xffffffffu, broke) >> (lane & ~7)) & 0xffu;
      // the record: every lane of the chain stores up to two entries (selects, no jump table)
      const Real px = xp - xa, py = yp - ya, pz = zp - za;
      const Real pd = fma(pz, pz, fma(py, py, px * px));
      // first entry:  lane 0 -> [0] b0 + b2, 1 -> [1] b1 + b3, 4 -> [2] b4 + b6, 5 -> [3] log u, 3 -> [7] 2 dx, 6 -> [10] |d|^2
      int e1 = -1;
      Real v1 = pairsum;
      e1 = role == 0 ? 0 : e1;
      e1 = role == 1 ? 1 : e1;
      e1 = role == 4 ? 2 : e1;
      if (role == 5) { e1 = 3; v1 = lg; }
      if (role == 3) { e1 = 7; v1 = px + px; }
      if (role == 6) { e1 = 10; v1 = pd; }
      // second entry: lane 0 -> [4] x', 1 -> [5] y', 2 -> [6] z', 4 -> [8] 2 dy, 5 -> [9] 2 dz
      int e2 = -1;
      Real v2 = xp;
      e2 = role == 0 ? 4 : e2;
      if (role == 1) { e2 = 5; v2 = yp; }
      if (role == 2) { e2 = 6; v2 = zp; }
      if (role == 4) { e2 = 8; v2 = py + py; }
      if (role == 5) { e2 = 9; v2 = pz + pz; }
      const int slot = g & (RING - 1);
      if (e1 >= 0) s_rec[slot][cl][e1] = (double)v1;
      if (e2 >= 0) s_rec[slot][cl][e2] = (double)v2;
      if (role == 2) s_mask[slot][cl] = mask;
      if (g < SW) {
        __syncthreads();
        for (int b = 0; b + 1 < g; ++b) pt_bar_arrive(1 + b % SW, NT);
        if (g >= 1) pt_bar_sync(1 + (g - 1) % SW, NT);
      } else {
        pt_bar_sync(1 + (g - 1) % SW, NT);
      }
    }
    for (int b = total - (total - s) % SW; b < total; ++b) pt_bar_arrive(1 + b % SW, NT);
    return;
  }

  // ---- pair warps: warp w owns chain chain0 + w ----
  ChainCtx c;
  ctx_load(d, chain0 + warp, d.C, c);
  const PtCoords<Real> X(reinterpret_cast<Real*>(smem_raw) + (size_t)warp * 3 * Ns, Ns);
  __syncthreads();
  const PtLJ<Real> lj(d);
  const double nbeta = -c.beta;
  PtNoSide noside;
  bool acc_prev = true;
  int g = 0;
  for (int sw = 0; sw < n_sweeps; ++sw) {
    const uint32_t t = t0 + (uint32_t)sw;
    for (int k = 0; k < N; ++k, ++g) {
      const int m = k;
      const int slot = g & (RING - 1);
      const double* rec = s_rec[slot][warp];
      Real xo, yo, zo;
      X.get(m, xo, yo, zo);
      const Real xn = (Real)rec[4], yn = (Real)rec[5], zn = (Real)rec[6];
      const Real tdx = (Real)rec[7], tdy = (Real)rec[8], tdz = (Real)rec[9], dd = (Real)rec[10];
      Real part;
      if constexpr (F2) part = pair_groups_f2<32, NI2, 1>(lj, X, lane, m, xo, yo, zo, tdx, tdy, tdz, dd, noside);
      else part = pair_groups<Real, 32, NI, 1>(lj, X, lane, m, xo, yo, zo, tdx, tdy, tdz, dd, noside);
      part += __shfl_xor_sync(0xffffffffu, part, 16);
      part += __shfl_xor_sync(0xffffffffu, part, 8);
      if (lane < 8) s_red[g & 1][warp][lane] = (double)part;
      pt_bar_sync(1 + g % SW, NT);

      double q8[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) q8[i] = s_red[g & 1][warp][i];
      const double bonds = rec[1] + (acc_prev ? rec[0] : rec[2]);
      const double logu = rec[3];
      const bool bond_broken = (s_mask[slot][warp] & (acc_prev ? 0x03u : 0x12u)) != 0u;
      const double pairs = ws_tree<8>(q8);
      const Real dE = (Real)(pairs + bonds);
      const bool accept = !bond_broken && (dE <= (Real)0 || logu < nbeta * (double)dE);
      const int owner = F2 ? (m >> 1) % 32 : m % 32;
      if (accept && lane == owner) X.set(m, xn, yn, zn);
      if (TRACE) {
        if (lane == 0 && d.tr_move && c.active && (long long)t < d.cap_sweeps)
          d.tr_move[((size_t)c.ti * d.cap_sweeps + t) * (size_t)N + k] = accept ? 1 : 0;
      }
      c.erun += accept ? (double)dE : 0.0;
      c.acc += accept ? 1u : 0u;
      c.brej += bond_broken ? 1u : 0u;
      acc_prev = accept;
    }
    __syncwarp();
    if (d.observables) measure_shape<Real, 32>(d, c, N, lane, 0, X);
    if (lane == 0 && c.active) measure_energy(d, c, t);
  }

  __syncwarp();
  if (c.active) {
    Real* gx = reinterpret_cast<Real*>(d.coords) + (size_t)c.s * 3 * d.Ng;
    for (int j = lane; j < N; j += 32) X.get(j, gx[j], gx[d.Ng + j], gx[2 * d.Ng + j]);
    if (lane == 0) ctx_store(d, c, n_sweeps);
  }
  // B1 fused (see k_sweep_ws)
  if (pl.fuse_exchange && c.active) {
    __threadfence();
    __syncwarp();
    if (lane == 0) {
      const unsigned before = atomicAdd(&d.done[c.e], 1u);
      s_last[warp] = before == (unsigned)(d.M - 1);
      if (s_last[warp]) d.done[c.e] = 0u;
    }
    __syncwarp();
    if (s_last[warp]) {
      __threadfence();
      const uint32_t x = pl.x;
      const int npairs = (d.M - (int)(x & 1u)) / 2;
      for (int q = lane; q < npairs; q += 32) pt_exchange_pair(d, c.e, (int)(x & 1u) + 2 * q, x);
    }
  }
}

}  // namespace
