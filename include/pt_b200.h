/*
 * include/pt_b200.h -- C ABI of the B200-native replica-exchange (parallel tempering)
 * Metropolis Monte Carlo for an elastic bead-spring homopolymer.
 *
 * Method: Gross, Janke, Bachmann, "Massively parallelized replica-exchange simulations of
 * polymers on GPUs", arxiv 1107.3490.  Line numbers below are those of PAPER.md.
 *
 *   model        E_LJ^mod + E_FENE, Eq. (1)-(4)                      PAPER.md:73-91  (Section 3.1)
 *   update       single-monomer displacement + Metropolis, Eq. (5)   PAPER.md:93-101 (Section 3.2)
 *   exchange     neighbouring temperatures, Eq. (6)                  PAPER.md:103-109 (Section 3.3)
 *   measurement  once per sweep: energy, R_ee, R_gyr (Eq. 8)
 *
 * Conventions that hold for every call
 *   - plain C, no torch types.  The handle is opaque.  Nothing throws or aborts across the ABI.
 *   - every function returns an int status: PT_OK (0) or a negative PT_E* code;
 *     pt_last_error(h) gives a NUL-terminated message owned by the library
 *     (h == NULL: the message of the last failed pt_create* on this thread).
 *   - pointers marked HOST are host memory, DEVICE are CUDA device memory.  A handle lives on the
 *     CUDA device that is current when it is created (with a workspace: the device that owns the
 *     workspace, which must be the current one, else PT_EINVAL); every later call makes that device
 *     current for its own duration and restores the caller's afterwards.
 *     Input arrays are caller-owned and are consumed (copied) before the call returns.
 *     Output arrays are caller-allocated; NULL for an output means "skip it".
 *   - everything returned is indexed by TEMPERATURE index i (0 = first entry of `temperatures`),
 *     never by storage slot: the device swaps temperature labels, not coordinates,
 *     which is equivalent to the exchange of conformations of PAPER.md:105.
 *   - all work is enqueued on the cudaStream_t given at creation; pt_read / pt_recompute_energy
 *     / pt_init synchronise that stream before they return, the others are asynchronous.
 *   - there is no CPU fallback: without a CUDA device every compute call returns PT_ECUDA.
 *
 * Random stream (all calls): Philox4x32-10, key = the ensemble's 64-bit seed (lo, hi),
 *   counter = (a, b, ensemble, tag << 24 | temperature index):
 *     tag 0 MOVE: a = step k within the sweep (0..N-1), b = sweep index t since pt_init;
 *                 words -> (s_x, s_y, s_z, u_accept)
 *     tag 1 PICK: same (a, b), only with PT_RANDOM_PICK: monomer = (w0 * N) >> 32
 *     tag 2 SWAP: a = lower temperature index of the pair, b = exchange event index x,
 *                 temperature field 0; w0 -> u_swap
 *     tag 3 INIT: a = monomer n, b = 0: the direction of bond (n-1, n) of the library's own random
 *                 walk (pt_init with conformations = NULL): z = s(w0), phi = 2 pi u(w1)
 *   word -> number, fp64:  s = (2w + 1 - 2^32) / 2^32 in (-1,1);  u = (w + 1/2) / 2^32 in (0,1)
 *                   fp32:  s = (2 (w >> 8) + 1 - 2^24) / 2^24;     u = ((w >> 9) + 1/2) / 2^23
 */
#ifndef PT_B200_H
#define PT_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pt_handle pt_handle;

enum { PT_F64 = 0, PT_F32 = 1 };
enum { PT_SEQUENTIAL = 0, PT_RANDOM_PICK = 1 };

enum {
  PT_OK = 0,
  PT_EINVAL = -1, /* bad parameter (N < 2, M < 1, E < 1, M >= 2^24, non-positive or non-finite T or
                     width, nbins < 0, emin >= emax, R <= 0, unknown flag, NULL required pointer,
                     workspace too small or misaligned) */
  PT_ESTATE = -2, /* sweeps / exchange / read before a successful pt_init */
  PT_EBOND = -3,  /* a supplied conformation has a non-finite energy: a non-finite coordinate or a
                     bond with |r - r0| >= R (FENE "diverges for r -> r0 +- R") */
  PT_ENOMEM = -4,
  PT_ECUDA = -5,  /* any CUDA error; the message carries cudaGetErrorString */
  PT_ERANGE = -6  /* sweep counter t or event counter x would leave 32 bits (Philox counter words) */
};

typedef struct {
  int32_t N;           /* monomers per chain, >= 2                                                    */
  int32_t M;           /* replicas = temperatures per ensemble, 1 <= M < 2^24                         */
  int32_t E;           /* independent ensembles, >= 1 (the throughput batch has 64)                   */
  int32_t precision;   /* PT_F64: the reference path.  PT_F32: coordinates and pair arithmetic in
                          fp32 (the paper's precision); E_run and moments stay fp64   */
  int32_t select_mode; /* PT_SEQUENTIAL: step k moves monomer k.  PT_RANDOM_PICK: "a random monomer
                          of the chain is picked"                                       */
  int32_t nbins;       /* interior energy-histogram bins per temperature, 0 = no histogram            */
  int32_t observables; /* != 0: accumulate R_ee^2 and R_gyr^2 (Eq. 8) once per sweep                  */
  int32_t lanes;       /* threads that share one chain's Delta-E sum: 0 = choose from N and the chain
                          count (few chains in sequential order: one CTA per chain with specialised
                          warps, see pt_launch_info); 8, 16, 32 = that many lanes of a warp; 64, 128,
                          256 = one CTA of that many threads per replica                              */
  double hist_emin, hist_emax;          /* histogram range, emin < emax (ignored if nbins == 0)       */
  double eps, r0, R, K, rc_over_sigma;  /* model constants; the paper's are 1, 0.7, 0.3, 40, 2.5
                                           (PAPER.md:81, :85); sigma = r0 / 2^(1/6) is derived        */
} pt_params;

/* Bytes of device memory a simulation with these parameters needs (0 if p is invalid). */
uint64_t pt_workspace_bytes(const pt_params* p);

/* Creates a simulation.  temperatures[M] HOST, > 0, k_B = 1, shared by all ensembles;
 * move_halfwidths[M] HOST, > 0: half-width of the uniform displacement cube at each temperature
 * (the paper's is 0.01 at every T).  cuda_stream: a cudaStream_t, or NULL for the
 * default stream.  pt_create allocates its device memory with cudaMalloc; the _with_workspace
 * form uses `device_ws` DEVICE (256-byte aligned, >= pt_workspace_bytes(p), owned by the caller
 * and kept alive until pt_destroy) -- this is how the Python binding hands in torch memory. */
int pt_create(pt_handle** out, const pt_params* p, const double* temperatures,
              const double* move_halfwidths, void* cuda_stream);
int pt_create_with_workspace(pt_handle** out, const pt_params* p, const double* temperatures,
                             const double* move_halfwidths, void* cuda_stream, void* device_ws,
                             uint64_t ws_bytes);
int pt_destroy(pt_handle* h);

/* seeds[E] HOST: one Philox key per ensemble.  conformations[E][M][N][3] HOST, fp64, the
 * conformation that starts at temperature i of ensemble e; NULL = the library generates, on the
 * host, a random walk of bond length r0 from the seeds (monomer 0 at the origin, bond directions
 * uniform on the sphere from the Philox tag INIT above; overlaps of non-bonded monomers are
 * allowed, so the initial energies can be large; read it back with pt_read).  Computes the running
 * energy of every chain by the full O(N^2) sum of Eq. (4), zeroes all statistics, sets the sweep
 * counter t = 0, the exchange-event counter x = 0 and the identity label permutation.
 * PT_EBOND if any chain's energy is not finite (state stays uninitialised). */
int pt_init(pt_handle* h, const uint64_t* seeds, const double* conformations);

/* n >= 0 sweeps of every chain, no exchange.  One sweep = N attempted single-monomer moves
 * (Section 3.2, Eq. 5), then one measurement: histogram, sum E, sum E^2, observables. */
int pt_sweeps(pt_handle* h, int64_t n);

/* One exchange event in every ensemble (Section 3.3, Eq. 6).  Event x tries the disjoint pairs
 * (i, i+1) with i = x mod 2, x mod 2 + 2, ...; accept iff Delta = (beta_i - beta_{i+1})(E_i -
 * E_{i+1}) >= 0 or u_swap < exp(Delta).  Swaps temperature labels on the device.
 * Before the events x = 0, 1, 3, 7, ... (x + 1 a power of two) the running energy of every chain is
 * replaced by the full sum of Eq. (4) (the paper's kernel recomputes the energy after every sweep,
 * PAPER.md:146), so that the rounding of a high-energy start does not stay in E_run for ever. */
int pt_exchange(pt_handle* h);

/* Repeats { pt_sweeps(exchange_every); pt_exchange() } until n_sweeps sweeps are done, without
 * host round trips; a last partial block of sweeps is not followed by an exchange.
 * exchange_every <= 0: no exchange at all.  Same results as the separate calls; where the sweep kernel is the
 * one-CTA-per-chain kernel (see pt_launch_info) the exchange is done at the end of the sweep launch itself, by
 * the last CTA of every ensemble to finish, instead of by a kernel of its own. */
int pt_run(pt_handle* h, int64_t n_sweeps, int64_t exchange_every);

/* Synchronises the stream and copies results to HOST arrays (NULL = skip). */
int pt_read(pt_handle* h,
            double*   energies      /* [E][M]           running energy at temperature i              */,
            uint64_t* histograms    /* [E][M][nbins+2]  interior bins, then underflow, overflow      */,
            double*   moments       /* [E][M][3]        n_meas, sum E, sum E^2                       */,
            uint64_t* move_counts   /* [E][M][3]        attempts, accepts, bond-range rejections     */,
            uint64_t* swap_counts   /* [E][M-1][2]      attempts, accepts of pair (i, i+1)           */,
            double*   conformations /* [E][M][N][3]     conformation currently at temperature i      */,
            double*   obs_moments   /* [E][M][5]        sum Ree^2, sum Rg^2, sum Rg^4, sum Ree^4,
                                                        sum E Rg^2 (Eq. 8 and d<Rg^2>/dT = beta^2
                                                        (<E Rg^2> - <E><Rg^2>))    */);

/* Full O(N^2) recomputation of Eq. (4) for every chain, without touching the running energy:
 * the invariant |E_run - E_full| is the caller's check.  energies_full[E][M] HOST. */
int pt_recompute_energy(pt_handle* h, double* energies_full);

/* Zeroes histograms, moments, observables and counters; keeps conformations, labels, t and x
 * (discarding thermalisation). */
int pt_reset_stats(pt_handle* h);

/* Test support: per-decision trace written by the kernels, all DEVICE, temperature-indexed,
 * NULL = off.  The library trusts the capacities: the buffers must be at least as large as stated
 * here.  move_dec != NULL selects separate instantiations of the sweep kernels (the decision
 * store sits in the step loop); with move_dec == NULL the sweep kernels are the ones a run without
 * any trace uses, and swap_dec / e_trace are still written (pt_sweep_kernel_name tells which).  move_dec[E][M][cap_sweeps][N] one byte (0/1) per attempted move;
 * swap_dec[E][cap_events][M-1] one byte per pair slot and event: 0 not attempted, 1 rejected,
 * 2 accepted; e_trace[E][M][cap_sweeps] the running energy after every sweep.  Sweeps / events
 * beyond the capacities are not recorded.  Buffers stay owned by the caller. */
int pt_set_trace(pt_handle* h, int64_t cap_sweeps, int64_t cap_events, uint8_t* move_dec,
                 uint8_t* swap_dec, double* e_trace);

/* Sweep and exchange-event counters since pt_init. */
int pt_counters(const pt_handle* h, int64_t* t_sweeps, int64_t* x_events);

/* Exact resume.  The random stream is keyed by (seed, ensemble, temperature
 * index, sweep t, step k) and by (pair, event x), and pt_read returns conformations by temperature
 * index, so a run is continued bit for bit by: pt_init(seeds, conformations read at the break) on
 * any handle with the same parameters, then pt_set_counters(t, x) with the counters read at the
 * break.  Statistics restart from zero (add them outside); the running energy is recomputed by
 * Eq. (4), i.e. it may differ from the uninterrupted one in the last bits.  0 <= t, x < 2^32;
 * PT_ESTATE before pt_init, PT_ERANGE outside the range. */
int pt_set_counters(pt_handle* h, int64_t t_sweeps, int64_t x_events);

/* How the sweep kernel is mapped: lanes per chain (as in pt_params.lanes, resolved), chains per
 * CTA, CTAs in the grid, dynamic shared memory bytes per CTA.  Any pointer may be NULL.  With
 * lanes = 0 and between 4 and 7 chains per SM sub-partition (and N in 51..56 or 97..100) the library maps
 * 4 chains x 8 lanes + 3 chains x 10 lanes on every sub-partition; it then reports 8 lanes and 28
 * chains per CTA.  With lanes = 0, PT_SEQUENTIAL, N >= 6 and few chains (about 1.5 chains per SM
 * sub-partition at most) every chain gets a CTA of P = 1..3 "pair" warps, which share the Delta-E sum, and
 * two or three "stream" warps, which evaluate the bond terms of Eq. (3) and log u ahead of the decision; it then
 * reports 32 P lanes and 1 chain per CTA (short chains in somewhat larger batches: 32 lanes, 4 chains per CTA, the
 * stream warps shared). */
int pt_launch_info(const pt_handle* h, int32_t* lanes, int32_t* chains_per_cta, int32_t* grid,
                   int32_t* smem_bytes);

/* NUL-terminated name of the sweep-kernel instantiation the next pt_sweeps will launch, e.g.
 * "k_sweep_mixed<double,13,10,trace=0>"; trace=1 while a move-decision trace is set.  buf HOST,
 * n bytes (truncated to fit). */
int pt_sweep_kernel_name(const pt_handle* h, char* buf, uint64_t n);

/* Number of kernels this handle has launched since creation (bench.py's gpu_launches). */
int64_t pt_kernel_launches(const pt_handle* h);

const char* pt_last_error(const pt_handle* h);

/* Measurement support (no handle): the sustained plain fp64 (PT_F64) or fp32 (PT_F32) FMA rate of
 * the current device in TFLOP/s (2 flops per FMA), best of `reps` launches of `iters` x 64
 * dependent-chain FMAs per thread at full occupancy, timed with CUDA events on `cuda_stream`.
 * It is the denominator of the "alu" roofline the sweep kernel is reported against (the Delta-E
 * sum of Eq. 5 is plain FMA-pipe work, no tensor cores).  tflops HOST. */
int pt_fma_peak(int precision, int iters, int reps, void* cuda_stream, double* tflops);

/* ---- the one entry point that allocates nothing ------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the full energy of Eq. (4) of n_chains conformations, the quantity pt_recompute_energy returns,
 * computed with scratch that lives in a static device array of the library instead of a workspace.
 *   p                  model constants and N (eps, r0, R, K, rc_over_sigma, N are read; the rest is ignored)
 *   dev_conformations  DEVICE pointer, [n_chains][N][3] fp64 (x, y, z of monomer 0, 1, ...), read only
 *   dev_energies       DEVICE pointer, [n_chains] fp64, written
 *   stream             a cudaStream_t (NULL = default stream); the call only enqueues, it does not synchronise
 * The current device is used.  No cudaMalloc, cudaFree or allocating library call is made; the first call on a device
 * asks for the scratch array's address (cudaGetSymbolAddress).  n_chains > PT_NOALLOC_MAX_CHAINS is PT_EINVAL: split
 * the batch.  Every GPU that loads the library holds the array (576 KiB) until the process exits.  All calls share
 * it: calls that overlap on the GPU (two streams, two host threads) race -- serialise them.  Energies agree with
 * pt_recompute_energy up to the order of summation (~1e-15 relative).  Errors: PT_EINVAL, PT_ECUDA; the message is
 * pt_noalloc_last_error() (per host thread). */
#define PT_NOALLOC_MAX_CHAINS 8192
int pt_energy_noalloc(const pt_params* p, const double* dev_conformations, double* dev_energies, int64_t n_chains,
                      void* stream);
const char* pt_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
