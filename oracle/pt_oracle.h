/*
 * oracle/pt_oracle.h -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, sequential fp64 restatement of the replica-exchange (parallel
 * tempering) Metropolis Monte Carlo of Gross, Janke, Bachmann, "Massively
 * parallelized replica-exchange simulations of polymers on GPUs"
 * (arxiv 1107.3490; PAPER.md).  It exists so that the CUDA path can be checked
 * against something that can be compared with the paper by eye.
 *
 *   - Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 *     --impl reference legs may load this library.  The product
 *     (paper_1107_3490_b200/) never does.
 *   - It shares no code, header, table or constant with the CUDA path.
 *   - Every function cites the PAPER.md passage it follows.  Where the paper
 *     is silent the reading is the one listed in DESIGN.md ("Readings").
 *
 * Parity pins: every function below is pinned by tests/test_oracle_pins.py
 * (closed forms, quadrature, brute force, published Philox known answers).
 * No function is "parity unpinned".
 */
#ifndef PT_ORACLE_H
#define PT_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Model + run parameters.  Constants of the paper: eps=1, r0=0.7, R=0.3,
 * K=40, rc_over_sigma=2.5; sigma = r0 / 2^(1/6). */
typedef struct {
  int32_t N;           /* monomers per chain (>= 2)                                  */
  int32_t M;           /* replicas = temperatures per ensemble (>= 1)                */
  int32_t E;           /* independent ensembles (>= 1)                               */
  int32_t select_mode; /* 0 = sequential monomer order, 1 = random pick */
  int32_t nbins;       /* interior histogram bins per temperature (0 = none)         */
  int32_t e_offset;    /* index of this state's ensemble 0 in the caller's job: the Philox counter
                          word is e_offset + e, so that a sample of the ensembles of a large job
                          can be recomputed one by one (0 = the whole job)                */
  double hist_emin, hist_emax;
  double eps, r0, R, K, rc_over_sigma;
} orc_params;

typedef struct orc_state orc_state;

/* ---- elementary pieces, exported so the pins can reach them ---- */

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11). */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* 32-bit word -> symmetric uniform in (-1,1), never 0; -> uniform in (0,1). */
double orc_word_to_sym(uint32_t w);
double orc_word_to_u01(uint32_t w);

/* Eq. (1)-(2): truncated and shifted Lennard-Jones, as a function of r^2. */
double orc_lj_mod(const orc_params* p, double r2);
/* Eq. (3): FENE bond, as a function of r^2; +inf outside (r0-R, r0+R). */
double orc_fene(const orc_params* p, double r2);
/* Eq. (4): total energy of one conformation x[N][3]. */
double orc_total_energy(const orc_params* p, const double* x);
/* Energy change of moving monomer m of x[N][3] to xnew[3] (local form of
 * E_new - E_old in Eq. 5).  *bond_ok = 0 if a new bond leaves the FENE range. */
double orc_delta_energy(const orc_params* p, const double* x, int m,
                        const double* xnew, int* bond_ok);
/* Eq. (8): squared radius of gyration; squared end-to-end distance. */
double orc_rgyr2(int N, const double* x);
double orc_ree2(int N, const double* x);

/* ---- the simulation ---- */

orc_state* orc_create(const orc_params* p, const double* temperatures /*[M]*/,
                      const double* move_halfwidths /*[M]*/);
void orc_destroy(orc_state* s);

/* Sets conformations [E][M][N][3] (temperature-index order), seeds [E];
 * E_run by Eq. (4); zeroes statistics; sweep counter t = 0, exchange counter
 * x = 0.  Returns 0, or -1 if a conformation has a non-finite energy. */
int orc_init(orc_state* s, const uint64_t* seeds, const double* conformations);

/* Optional trace buffers (NULL = off), all caller-owned:
 *   move_dec  [E][M][T][N]  one byte (0/1) per attempted move, T = capacity in sweeps
 *   swap_dec  [E][X][M-1]   one byte per pair slot and event: 0 = not attempted,
 *                           1 = attempted+rejected, 2 = attempted+accepted
 *   e_trace   [E][M][T]     E_run after every sweep
 *   ree2_trace, rg2_trace [E][M][T]  observables after every sweep          */
void orc_set_trace(orc_state* s, int64_t cap_sweeps, int64_t cap_events,
                   uint8_t* move_dec, uint8_t* swap_dec, double* e_trace,
                   double* ree2_trace, double* rg2_trace);

void orc_set_threads(orc_state* s, int nthreads); /* chains are independent between events */
int  orc_get_threads(const orc_state* s);

void orc_sweeps(orc_state* s, int64_t n);     /* n sweeps of every chain; 1 sweep = N attempted moves */
void orc_exchange(orc_state* s);              /* one exchange event (one parity) in every ensemble    */
void orc_run(orc_state* s, int64_t n_sweeps, int64_t exchange_every);

/* Everything indexed by temperature index.  NULL = skip. */
void orc_read(const orc_state* s,
              double*   energies      /*[E][M]          */,
              uint64_t* histograms    /*[E][M][nbins+2] interior, underflow, overflow */,
              double*   moments       /*[E][M][3]       n_meas, sum E, sum E^2 */,
              uint64_t* move_counts   /*[E][M][3]       attempts, accepts, bond-range rejections */,
              uint64_t* swap_counts   /*[E][M-1][2]     attempts, accepts for pair (i,i+1) */,
              double*   conformations /*[E][M][N][3]    */,
              double*   obs_moments   /*[E][M][5]       sum Ree^2, sum Rg^2, sum Rg^4, sum Ree^4, sum E Rg^2 */);

#ifdef __cplusplus
}
#endif
#endif
