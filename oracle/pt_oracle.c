/*
 * oracle/pt_oracle.c -- CPU ORACLE, TEST INFRASTRUCTURE ONLY (see pt_oracle.h).
 *
 * Plain C99, fp64, one loop per sum, libm sqrt/log/exp/pow.  Compile with
 *   gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC
 * (-ffp-contract=off: the proposal x' = x + d*s is two separately rounded
 * operations, reading R7).  No blocking, fusion or reordering beyond
 * what the paper's equations state.  Shares nothing with the CUDA path.
 *
 * Paper: Gross, Janke, Bachmann, arxiv 1107.3490; line numbers are PAPER.md's.
 */
#include "pt_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------- */
/* Random stream: Philox4x32-10 (Salmon et al., SC'11), counter-based.       */
/* The paper draws its uniforms from a host-made pool and    */
/* suggests an on-device generator instead; north_star fixes Philox keyed by  */
/* (seed, ensemble, replica, sweep, step).  DESIGN.md reading R8.             */
/* ------------------------------------------------------------------------- */

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   /* round multipliers */
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   /* Weyl key increments */
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += W0; k1 += W1; }
    uint64_t p0 = (uint64_t)M0 * c0;
    uint64_t p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* (2w + 1 - 2^32) / 2^32: 2^32 equally spaced odd numerators, in (-1,1), never 0.
 * Exact in fp64 (33-bit integer times a power of two). */
double orc_word_to_sym(uint32_t w)
{
  int64_t odd = 2 * (int64_t)w + 1 - 4294967296LL;
  return (double)odd * (1.0 / 4294967296.0);
}

/* (w + 1/2) / 2^32, in (0,1).  Exact in fp64. */
double orc_word_to_u01(uint32_t w)
{
  return ((double)w + 0.5) * (1.0 / 4294967296.0);
}

enum { TAG_MOVE = 0, TAG_PICK = 1, TAG_SWAP = 2 };

/* counter = (a, b, ensemble, tag<<24 | temperature index), key = 64-bit seed of the ensemble */
static void draw(uint64_t seed, uint32_t a, uint32_t b, uint32_t e, uint32_t tag, uint32_t i,
                 uint32_t w[4])
{
  uint32_t ctr[4] = { a, b, e, (tag << 24) | i };
  uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
  orc_philox4x32_10(ctr, key, w);
}

/* ------------------------------------------------------------------------- */
/* Model: PAPER.md:73-91 (Section 3.1, Eq. 1-4)                              */
/* ------------------------------------------------------------------------- */

static double sigma_of(const orc_params* p) { return p->r0 / pow(2.0, 1.0 / 6.0); } /* sigma = 2^(-1/6) r0 */

/* Eq. (2): E_LJ(r) = 4 eps [ (sigma/r)^12 - (sigma/r)^6 ], written in r^2. */
static double lj_plain(const orc_params* p, double r2)
{
  double sigma = sigma_of(p);
  double w = (sigma * sigma) / r2;     /* (sigma/r)^2 */
  double s6 = w * w * w;               /* (sigma/r)^6 */
  return 4.0 * p->eps * (s6 * s6 - s6);
}

/* Eq. (1): E_LJ^mod(r) = E_LJ(min(r, r_c)) - E_LJ(r_c), r_c = 2.5 sigma.
 * For r >= r_c this is exactly 0. */
double orc_lj_mod(const orc_params* p, double r2)
{
  double rc = p->rc_over_sigma * sigma_of(p);
  double rc2 = rc * rc;
  if (r2 >= rc2) return 0.0;
  return lj_plain(p, r2) - lj_plain(p, rc2);
}

/* Eq. (3): E_FENE(r) = -(K/2) R^2 log[ 1 - ((r - r0)/R)^2 ]; "diverges for r -> r0 +- R"
 * (PAPER.md:85).  Outside the open interval the energy is +infinity (reading R5);
 * the test is !(q*q < 1) so that q*q == 1 and NaN are both outside. */
double orc_fene(const orc_params* p, double r2)
{
  double r = sqrt(r2);
  double q = (r - p->r0) / p->R;
  if (!(q * q < 1.0)) return INFINITY;
  return -0.5 * p->K * p->R * p->R * log(1.0 - q * q);
}

static double dist2(const double* a, const double* b)
{
  double dx = a[0] - b[0], dy = a[1] - b[1], dz = a[2] - b[2];
  return dx * dx + dy * dy + dz * dz;
}

/* Eq. (4): E(C) = 1/2 sum_{i != j} E_LJ^mod(r_ij) + sum_{i=1}^{N-1} E_FENE(r_{i,i+1}).
 * "All monomers interact": bonded neighbours carry LJ as well (reading R1).
 * The 1/2 sum over ordered pairs is written as the sum over i < j. */
double orc_total_energy(const orc_params* p, const double* x)
{
  int N = p->N;
  double e_lj = 0.0, e_fene = 0.0;
  for (int i = 0; i < N; ++i)
    for (int j = i + 1; j < N; ++j)
      e_lj += orc_lj_mod(p, dist2(x + 3 * i, x + 3 * j));
  for (int i = 0; i + 1 < N; ++i)
    e_fene += orc_fene(p, dist2(x + 3 * i, x + 3 * (i + 1)));
  return e_lj + e_fene;
}

/* Local form of E_new - E_old (Eq. 5) for a single-monomer move:
 * only the N-1 pair terms and the <= 2 bond terms that contain monomer m change. */
double orc_delta_energy(const orc_params* p, const double* x, int m, const double* xnew,
                        int* bond_ok)
{
  int N = p->N;
  const double* xold = x + 3 * m;
  double f_new_lo = 0.0, f_new_hi = 0.0, f_old_lo = 0.0, f_old_hi = 0.0;
  *bond_ok = 1;
  if (m > 0) {
    f_new_lo = orc_fene(p, dist2(xnew, x + 3 * (m - 1)));
    f_old_lo = orc_fene(p, dist2(xold, x + 3 * (m - 1)));
    if (isinf(f_new_lo)) *bond_ok = 0;
  }
  if (m + 1 < N) {
    f_new_hi = orc_fene(p, dist2(xnew, x + 3 * (m + 1)));
    f_old_hi = orc_fene(p, dist2(xold, x + 3 * (m + 1)));
    if (isinf(f_new_hi)) *bond_ok = 0;
  }
  if (!*bond_ok) return INFINITY;            /* infinite E_new: never accepted */
  double e_new = 0.0, e_old = 0.0;
  for (int j = 0; j < N; ++j) {
    if (j == m) continue;
    e_new += orc_lj_mod(p, dist2(xnew, x + 3 * j));
    e_old += orc_lj_mod(p, dist2(xold, x + 3 * j));
  }
  e_new += f_new_lo; e_new += f_new_hi;
  e_old += f_old_lo; e_old += f_old_hi;
  return e_new - e_old;
}

/* Eq. (8): r_gyr^2 = (1/N) sum_k (r_k - r_mean)^2. */
double orc_rgyr2(int N, const double* x)
{
  double c[3] = { 0.0, 0.0, 0.0 };
  for (int k = 0; k < N; ++k) { c[0] += x[3 * k]; c[1] += x[3 * k + 1]; c[2] += x[3 * k + 2]; }
  c[0] /= N; c[1] /= N; c[2] /= N;
  double s = 0.0;
  for (int k = 0; k < N; ++k) s += dist2(x + 3 * k, c);
  return s / N;
}

/* squared end-to-end distance |r_N - r_1|^2. */
double orc_ree2(int N, const double* x) { return dist2(x + 3 * (N - 1), x); }

/* ------------------------------------------------------------------------- */
/* State                                                                     */
/* ------------------------------------------------------------------------- */

struct orc_state {
  orc_params p;
  double* T;        /* [M] */
  double* beta;     /* [M]  beta = 1/(k_B T), k_B = 1 */
  double* width;    /* [M]  half-width of the displacement cube (reading R2) */
  uint64_t* seed;   /* [E] */
  double* X;        /* [E][M][N][3], indexed by TEMPERATURE index */
  double* Erun;     /* [E][M] */
  uint64_t* hist;   /* [E][M][nbins+2] */
  double* mom;      /* [E][M][3] */
  double* obs;      /* [E][M][5] */
  uint64_t* mcount; /* [E][M][3] */
  uint64_t* scount; /* [E][M-1][2] */
  int64_t t;        /* sweeps done since init      */
  int64_t x;        /* exchange events since init  */
  int initialised;
  int nthreads;
  /* trace */
  int64_t cap_sweeps, cap_events;
  uint8_t* tr_move; uint8_t* tr_swap; double* tr_e; double* tr_ree2; double* tr_rg2;
};

orc_state* orc_create(const orc_params* p, const double* temperatures, const double* widths)
{
  if (!p || !temperatures || !widths) return NULL;
  if (p->N < 2 || p->M < 1 || p->E < 1 || p->nbins < 0 || p->e_offset < 0) return NULL;
  if (p->nbins > 0 && !(p->hist_emin < p->hist_emax)) return NULL;
  orc_state* s = (orc_state*)calloc(1, sizeof(orc_state));
  if (!s) return NULL;
  s->p = *p;
  size_t M = (size_t)p->M, E = (size_t)p->E, N = (size_t)p->N, C = E * M;
  s->T = (double*)calloc(M, sizeof(double));
  s->beta = (double*)calloc(M, sizeof(double));
  s->width = (double*)calloc(M, sizeof(double));
  s->seed = (uint64_t*)calloc(E, sizeof(uint64_t));
  s->X = (double*)calloc(C * N * 3, sizeof(double));
  s->Erun = (double*)calloc(C, sizeof(double));
  s->hist = (uint64_t*)calloc(C * (size_t)(p->nbins + 2), sizeof(uint64_t));
  s->mom = (double*)calloc(C * 3, sizeof(double));
  s->obs = (double*)calloc(C * 5, sizeof(double));
  s->mcount = (uint64_t*)calloc(C * 3, sizeof(uint64_t));
  s->scount = (uint64_t*)calloc(E * (M > 1 ? M - 1 : 1) * 2, sizeof(uint64_t));
  for (size_t i = 0; i < M; ++i) {
    if (!(temperatures[i] > 0.0) || !(widths[i] > 0.0)) { orc_destroy(s); return NULL; }
    s->T[i] = temperatures[i];
    s->beta[i] = 1.0 / temperatures[i];
    s->width[i] = widths[i];
  }
  s->nthreads = 1;
  return s;
}

void orc_destroy(orc_state* s)
{
  if (!s) return;
  free(s->T); free(s->beta); free(s->width); free(s->seed); free(s->X); free(s->Erun);
  free(s->hist); free(s->mom); free(s->obs); free(s->mcount); free(s->scount);
  free(s);
}

int orc_init(orc_state* s, const uint64_t* seeds, const double* conformations)
{
  const orc_params* p = &s->p;
  size_t M = (size_t)p->M, E = (size_t)p->E, N = (size_t)p->N, C = E * M;
  memcpy(s->seed, seeds, E * sizeof(uint64_t));
  memcpy(s->X, conformations, C * N * 3 * sizeof(double));
  memset(s->hist, 0, C * (size_t)(p->nbins + 2) * sizeof(uint64_t));
  memset(s->mom, 0, C * 3 * sizeof(double));
  memset(s->obs, 0, C * 5 * sizeof(double));
  memset(s->mcount, 0, C * 3 * sizeof(uint64_t));
  memset(s->scount, 0, E * (M > 1 ? M - 1 : 1) * 2 * sizeof(uint64_t));
  s->t = 0; s->x = 0;
  int bad = 0;
  for (size_t c = 0; c < C; ++c) {
    s->Erun[c] = orc_total_energy(p, s->X + c * N * 3);
    if (!isfinite(s->Erun[c])) bad = 1;
  }
  s->initialised = !bad;
  return bad ? -1 : 0;
}

void orc_set_trace(orc_state* s, int64_t cap_sweeps, int64_t cap_events, uint8_t* move_dec,
                   uint8_t* swap_dec, double* e_trace, double* ree2_trace, double* rg2_trace)
{
  s->cap_sweeps = cap_sweeps; s->cap_events = cap_events;
  s->tr_move = move_dec; s->tr_swap = swap_dec; s->tr_e = e_trace;
  s->tr_ree2 = ree2_trace; s->tr_rg2 = rg2_trace;
}

void orc_set_threads(orc_state* s, int n) { s->nthreads = n < 1 ? 1 : n; }
int orc_get_threads(const orc_state* s) { return s->nthreads; }

/* ------------------------------------------------------------------------- */
/* One sweep of one chain: PAPER.md:93-101 (Section 3.2, Eq. 5).             */
/* A sweep is N attempted single-monomer moves (reading R4).                 */
/* ------------------------------------------------------------------------- */
static void sweep_chain(orc_state* s, int e, int i, int64_t t)
{
  const orc_params* p = &s->p;
  int N = p->N, M = p->M;
  size_t c = (size_t)e * M + i;
  double* X = s->X + c * (size_t)N * 3;
  double beta = s->beta[i], d = s->width[i];
  for (int k = 0; k < N; ++k) {
    uint32_t w[4];
    /* "A random monomer of the chain is picked" -- or sequential order (reading R3) */
    int m = k;
    if (p->select_mode == 1) {
      draw(s->seed[e], (uint32_t)k, (uint32_t)t, (uint32_t)(p->e_offset + e), TAG_PICK, (uint32_t)i, w);
      m = (int)(((uint64_t)w[0] * (uint64_t)N) >> 32);
    }
    /* "a shift of its coordinates by a random vector ... components uniformly distributed"
     * in [-d, d] */
    draw(s->seed[e], (uint32_t)k, (uint32_t)t, (uint32_t)(p->e_offset + e), TAG_MOVE, (uint32_t)i, w);
    double xnew[3];
    for (int a = 0; a < 3; ++a) {
      double delta = d * orc_word_to_sym(w[a]);   /* one rounding */
      xnew[a] = X[3 * m + a] + delta;             /* one rounding */
    }
    double u = orc_word_to_u01(w[3]);
    int bond_ok;
    double dE = orc_delta_energy(p, X, m, xnew, &bond_ok);
    /* Eq. (5): p = min(1, exp[-beta (E_new - E_old)]) */
    int accept;
    if (!bond_ok) accept = 0;
    else if (dE <= 0.0) accept = 1;
    else accept = (u < exp(-beta * dE));           /* NaN compares false: reject */
    s->mcount[c * 3 + 0] += 1;
    if (!bond_ok) s->mcount[c * 3 + 2] += 1;
    if (accept) {
      X[3 * m] = xnew[0]; X[3 * m + 1] = xnew[1]; X[3 * m + 2] = xnew[2];
      s->Erun[c] += dE;
      s->mcount[c * 3 + 1] += 1;
    }
    if (s->tr_move && t < s->cap_sweeps)
      s->tr_move[(c * (size_t)s->cap_sweeps + (size_t)t) * (size_t)N + (size_t)k] = (uint8_t)accept;
  }
  /* measurement once per sweep (energy, R_ee, R_gyr after oneSweep) */
  double Ecur = s->Erun[c];
  if (p->nbins > 0) {
    uint64_t* h = s->hist + c * (size_t)(p->nbins + 2);
    double b = floor((Ecur - p->hist_emin) * ((double)p->nbins / (p->hist_emax - p->hist_emin)));
    if (b >= 0.0 && b < (double)p->nbins) h[(size_t)b] += 1;
    else if (b < 0.0) h[p->nbins] += 1;            /* underflow */
    else h[p->nbins + 1] += 1;                     /* overflow (and NaN) */
  }
  s->mom[c * 3 + 0] += 1.0;
  s->mom[c * 3 + 1] += Ecur;
  s->mom[c * 3 + 2] += Ecur * Ecur;
  double ree2 = orc_ree2(N, X), rg2 = orc_rgyr2(N, X);
  s->obs[c * 5 + 0] += ree2;
  s->obs[c * 5 + 1] += rg2;
  s->obs[c * 5 + 2] += rg2 * rg2;
  s->obs[c * 5 + 3] += ree2 * ree2;
  /* the cross moment of the thermal fluctuation d<r_gyr^2>/dT = beta^2 (<E r_gyr^2> - <E><r_gyr^2>)
   * that Fig. 5 plots (text around Eq. 8) */
  s->obs[c * 5 + 4] += Ecur * rg2;
  if (t < s->cap_sweeps) {
    size_t o = c * (size_t)s->cap_sweeps + (size_t)t;
    if (s->tr_e) s->tr_e[o] = Ecur;
    if (s->tr_ree2) s->tr_ree2[o] = ree2;
    if (s->tr_rg2) s->tr_rg2[o] = rg2;
  }
}

void orc_sweeps(orc_state* s, int64_t n)
{
  int C = s->p.E * s->p.M, M = s->p.M;
  int64_t t0 = s->t;
  /* chains are independent between exchange events and the random stream is
   * counter-based, so the result does not depend on the thread count */
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(s->nthreads)
#endif
  for (int c = 0; c < C; ++c)
    for (int64_t t = t0; t < t0 + n; ++t)
      sweep_chain(s, c / M, c % M, t);
  s->t = t0 + n;
}

/* ------------------------------------------------------------------------- */
/* Replica exchange: PAPER.md:103-109 (Section 3.3, Eq. 6).                  */
/* "an attempt to exchange the conformations of neighboring replicas i and   */
/* i+1", p = min(1, exp[(E_i - E_{i+1})(beta_i - beta_{i+1})]).              */
/* Pairs tried in event x: i = x mod 2, x mod 2 + 2, ... (reading R6).       */
/* ------------------------------------------------------------------------- */
void orc_exchange(orc_state* s)
{
  const orc_params* p = &s->p;
  int N = p->N, M = p->M;
  /* Re-basing of the running energy (reading R22).  The paper's kernel recomputes the whole
   * energy by Eq. (4) after every sweep (Listing 2: energy(&ps) follows oneSweep), so its
   * energies never carry history; north_star fixes the local Delta E, and E_run += Delta E keeps the
   * absolute rounding of the largest energy a chain ever held -- after a random-walk start with
   * overlaps (E ~ 1e10 and beyond) that rounding can exceed the relaxed energy itself,
   * and the swap test below would read noise.  Before the events x = 0, 1, 3, 7, ... (x + 1 a power of
   * two) E_run is therefore replaced by the Eq.-4 sum of the current conformation: a logarithmic number
   * of full recomputations per run. */
  if (((s->x + 1) & s->x) == 0) {
    size_t C = (size_t)p->E * (size_t)M;
    for (size_t c = 0; c < C; ++c) s->Erun[c] = orc_total_energy(p, s->X + c * (size_t)N * 3);
  }
  double* tmp = (double*)malloc((size_t)N * 3 * sizeof(double));
  for (int e = 0; e < p->E; ++e) {
    for (int i = (int)(s->x % 2); i + 1 < M; i += 2) {
      size_t ci = (size_t)e * M + i, cj = ci + 1;
      double delta = (s->beta[i] - s->beta[i + 1]) * (s->Erun[ci] - s->Erun[cj]);
      uint32_t w[4];
      draw(s->seed[e], (uint32_t)i, (uint32_t)s->x, (uint32_t)(p->e_offset + e), TAG_SWAP, 0u, w);
      double u = orc_word_to_u01(w[0]);
      int accept = (delta >= 0.0) ? 1 : (u < exp(delta));
      uint64_t* sc = s->scount + ((size_t)e * (M - 1) + i) * 2;
      sc[0] += 1;
      if (accept) {
        sc[1] += 1;
        double* Xi = s->X + ci * (size_t)N * 3;
        double* Xj = s->X + cj * (size_t)N * 3;
        memcpy(tmp, Xi, (size_t)N * 3 * sizeof(double));
        memcpy(Xi, Xj, (size_t)N * 3 * sizeof(double));
        memcpy(Xj, tmp, (size_t)N * 3 * sizeof(double));
        double te = s->Erun[ci]; s->Erun[ci] = s->Erun[cj]; s->Erun[cj] = te;
      }
      if (s->tr_swap && s->x < s->cap_events)
        s->tr_swap[((size_t)e * (size_t)s->cap_events + (size_t)s->x) * (size_t)(M - 1) + (size_t)i] =
            (uint8_t)(accept ? 2 : 1);
    }
  }
  free(tmp);
  s->x += 1;
}

void orc_run(orc_state* s, int64_t n_sweeps, int64_t exchange_every)
{
  int64_t done = 0;
  while (done < n_sweeps) {
    int64_t n = exchange_every;
    if (n <= 0 || n > n_sweeps - done) n = n_sweeps - done;
    orc_sweeps(s, n);
    done += n;
    if (exchange_every > 0 && n == exchange_every) orc_exchange(s);
  }
}

void orc_read(const orc_state* s, double* energies, uint64_t* histograms, double* moments,
              uint64_t* move_counts, uint64_t* swap_counts, double* conformations,
              double* obs_moments)
{
  const orc_params* p = &s->p;
  size_t M = (size_t)p->M, E = (size_t)p->E, N = (size_t)p->N, C = E * M;
  if (energies) memcpy(energies, s->Erun, C * sizeof(double));
  if (histograms) memcpy(histograms, s->hist, C * (size_t)(p->nbins + 2) * sizeof(uint64_t));
  if (moments) memcpy(moments, s->mom, C * 3 * sizeof(double));
  if (move_counts) memcpy(move_counts, s->mcount, C * 3 * sizeof(uint64_t));
  if (swap_counts && M > 1) memcpy(swap_counts, s->scount, E * (M - 1) * 2 * sizeof(uint64_t));
  if (conformations) memcpy(conformations, s->X, C * N * 3 * sizeof(double));
  if (obs_moments) memcpy(obs_moments, s->obs, C * 5 * sizeof(double));
}
