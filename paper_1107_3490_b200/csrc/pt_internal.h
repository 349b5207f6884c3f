// Internal declarations shared by the translation units of libpt_b200.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pt_b200.h"

// Coordinates that can never be within the cutoff of a real monomer.  Used for the padding
// entries of a chain's shared-memory arrays and to hide the moved monomer from its own sum.
#define PT_FAR 1.0e6

// observables per temperature: sum R_ee^2, R_gyr^2, R_gyr^4, R_ee^4, E R_gyr^2 (Eq. 8)
#define PT_NOBS 5

// Device-side view of one simulation; passed by value to every kernel.
struct PtDev {
  int N, M, E, C;        // C = E*M chains
  int Ng;                // padded length of one coordinate array in HBM (even)
  int nbins, select_mode, observables;
  double hist_emin, hist_scale;  // scale = nbins / (emax - emin)
  // model constants, host-computed in fp64
  double ljA;    // 4 eps sigma^12
  double ljB;    // 4 eps sigma^6
  double ljC;    // E_LJ(r_c) = 4 eps [(sigma/r_c)^12 - (sigma/r_c)^6]
  double rc2;    // r_c^2
  double sigma2; // sigma^2
  double eps4;   // 4 eps
  double r0, R, invR;
  double feneC;  // -(K/2) R^2
  // state, slot-indexed: slot s = e*M + (slot within ensemble)
  void* coords;          // Real [C][3][Ng]  SoA per chain: x[], y[], z[]
  double* erun;          // [C]
  int* temp_of_slot;     // [C] temperature index (within the ensemble) the slot currently has
  int* slot_of_temp;     // [C] slot (within the ensemble) that currently has temperature i
  // per-temperature constants and keys
  const double* beta;    // [M]
  const double* width;   // [M]
  const uint2* keys;     // [E]
  // statistics, temperature-indexed: ti = e*M + i
  unsigned long long* hist;    // [C][nbins+2]
  double* mom;                 // [C][3]
  double* obs;                 // [C][PT_NOBS]
  unsigned long long* mcount;  // [C][3]
  unsigned long long* scount;  // [E][max(M-1,1)][2]
  unsigned* done;              // [E] chains of the ensemble that have finished the launch (fused exchange, k_sweep_ws)
  // trace (test support), temperature-indexed
  unsigned char* tr_move;
  unsigned char* tr_swap;
  double* tr_e;
  long long cap_sweeps, cap_events;
};

struct PtLaunch;
typedef void (*PtSweepFn)(const PtDev, const PtLaunch, const uint32_t, const int);

struct PtLaunch {
  int lanes;           // resolved lanes per chain
  int chains_per_cta;
  int threads;         // per CTA
  int grid;
  int smem_bytes;      // dynamic shared memory per CTA
  int sstride;         // shared-memory stride between chains, in Reals
  int Ns;              // padded monomers per coordinate array in shared memory
  int ni;              // unrolled partner-loop iterations of the chosen kernel (0 = run-time loop)
  int kind;            // PT_K_GROUP, PT_K_COMP, PT_K_CTA, PT_K_SEVEN(_FULL) or PT_K_WS (then lanes = 32 x pair warps)
  int stagger;         // PT_K_GROUP: start delay in cycles per rank of a warp on its sub-partition (0 = none)
  // PT_K_COMP / PT_K_SEVEN: warps of different kinds in one CTA; kind 0, 1, 2, 3 = 8, 16, 32, 10 lanes per chain
  // (k_sweep_comp uses 0..2; k_sweep_seven 0 for warps 0..3 and 3 for warps 4..7)
  int nik[4];          // partner-loop iterations of each kind of warp (template arguments of the kernel; 0 = unused)
  int kstride[4];      // shared-memory stride between the chains of a warp of each kind, in Reals
  int wkind[8];        // kind of warp w
  int wfirst[8];       // first chain of warp w within the CTA
  int wcount[8];       // chains of warp w (<= 32 / lanes; the other chain slots stay idle)
  int woff[8];         // shared-memory offset of warp w's first chain, in Reals
  int wdelay[8];       // start delay of warp w in cycles
  // k_sweep_ws, set per launch by pt_run: the exchange event that follows the sweeps is done by the last CTA of
  // every ensemble to finish (no exchange kernel, no launch gap)
  int fuse_exchange;   // 0 = none
  unsigned x;          // index of that exchange event
};

enum { PT_K_GROUP = 0, PT_K_COMP = 1, PT_K_CTA = 2, PT_K_SEVEN = 3, PT_K_SEVEN_FULL = 4, PT_K_WS = 5, PT_K_WSG = 6 };

// Kernel tables, one per translation unit that instantiates sweep kernels (nullptr = not in this unit).
PtSweepFn pt_lookup_group(int lanes, int ni, int precision, bool trace);   // pt_sweep_group.cu
PtSweepFn pt_lookup_ws(int pair_warps, int ni, int precision, bool trace);   // pt_sweep_ws.cu
int pt_ws_variant(int pair_warps, int ni_needed);
int pt_ws_stream_warps(int pair_warps, int ni);
PtSweepFn pt_lookup_wsg(int chains_per_cta, int ni, int precision, bool trace);   // pt_sweep_wsg.cu
int pt_wsg_variant(int chains_per_cta, int ni_needed);                           // stream warps of that instantiation (2 or 3)                          // smallest instantiated NI >= ni_needed, or -1
PtSweepFn pt_lookup_cta(int precision, bool trace);                        // pt_sweep_group.cu
PtSweepFn pt_lookup_comp(int kind, const int nik[4], int precision, bool trace);   // pt_sweep_comp*.cu
// the unrolled variants of k_sweep_group: smallest NI >= ni_needed for this lane count, 0 = run-time loop
int pt_group_variant(int lanes, int ni_needed);


// pt_sweep.cu
cudaError_t pt_plan_sweep(const PtDev& d, int precision, int lanes_requested, PtLaunch* plan);
cudaError_t pt_launch_sweep(const PtDev& d, int precision, const PtLaunch& plan, uint32_t t0,
                            int n_sweeps, cudaStream_t stream);
// name of the instantiation pt_launch_sweep would start, e.g. "k_sweep_mixed<double,13,10,trace=0>"
void pt_sweep_kernel_desc(const PtLaunch& plan, int precision, bool trace, char* buf, size_t n);

// pt_aux.cu
cudaError_t pt_launch_scatter_init(const PtDev& d, int precision, const double* staging,
                                   cudaStream_t stream);
cudaError_t pt_launch_zero_stats(const PtDev& d, cudaStream_t stream);
cudaError_t pt_launch_full_energy(const PtDev& d, int precision, double* out_slot_energy,
                                  cudaStream_t stream);
cudaError_t pt_launch_exchange(const PtDev& d, uint32_t x, cudaStream_t stream);
cudaError_t pt_launch_gather(const PtDev& d, int precision, const double* slot_energy,
                             double* out_energy_by_temp, double* out_conf_by_temp,
                             cudaStream_t stream);
