// C ABI of libpt_b200.so (include/pt_b200.h): argument validation, device-memory layout, launches.
// No CPU fallback: every compute call runs CUDA kernels or fails with PT_ECUDA.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <string>
#include <vector>

#include "pt_internal.h"

// fp32 path: exchange events between two refreshes of the running energy from Eq. (4)
#define PT_F32_REFRESH_EVENTS 8

struct pt_handle {
  pt_params p;
  PtDev d;
  PtLaunch plan;
  cudaStream_t stream;
  int device;          // CUDA device ordinal the handle was created on; every call runs there
  void* ws;            // base of the device workspace
  uint64_t ws_bytes;
  bool owns_ws;
  bool initialised;
  int64_t t, x;        // sweeps / exchange events since pt_init
  int64_t launches;
  // device scratch
  double* staging;     // [C][N][3] fp64 AoS: upload at init, gather target at read
  double* e_by_temp;   // [C]
  double* e_full;      // [C] slot-indexed scratch of the full recompute
  std::string err;
};

namespace {

thread_local std::string g_create_err;

int fail(pt_handle* h, int code, const std::string& msg)
{
  if (h) h->err = msg; else g_create_err = msg;
  return code;
}

int cuda_fail(pt_handle* h, cudaError_t e, const char* where)
{
  return fail(h, PT_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

#define PT_CUDA(h, call)                                   \
  do {                                                     \
    cudaError_t e__ = (call);                              \
    if (e__ != cudaSuccess) return cuda_fail((h), e__, #call); \
  } while (0)

uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

// Makes the handle's device current for the duration of a call and restores the caller's afterwards.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(int device)
  {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != device) {
      err = cudaSetDevice(device);
      switched = err == cudaSuccess;
    }
  }
  ~DeviceGuard()
  {
    if (switched) cudaSetDevice(prev);
  }
};

#define PT_ENTER(h)                                                     \
  DeviceGuard guard__((h)->device);                                     \
  if (guard__.err != cudaSuccess) return cuda_fail((h), guard__.err, "selecting the handle's device")

// ---- host-side random walk of pt_init(conformations = NULL) (SURVEY.md 8(d) input recipe) ----
// Philox4x32-10 on the host, same stream layout as the device (include/pt_b200.h), tag 3 = INIT.
void host_philox(const uint32_t ctr[4], uint64_t seed, uint32_t out[4])
{
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = 0xD2511F53ull * c0, p1 = 0xCD9E8D57ull * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Monomer 0 at the origin; monomer n = monomer n-1 + r0 (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z),
// z = s(w0) in (-1, 1), phi = 2 pi u(w1), words from Philox(ctr = (n, 0, e, 3 << 24 | i), key = seed_e).
// Every bond has length r0 up to rounding (E_FENE ~ 0); non-bonded overlaps are allowed, so initial
// energies can be large and the first sweeps relax them.
void host_random_walk(const pt_params& p, const uint64_t* seeds, std::vector<double>* out)
{
  const size_t N = (size_t)p.N, M = (size_t)p.M, E = (size_t)p.E;
  out->assign(E * M * N * 3, 0.0);
  const double two_pi = 6.283185307179586476925286766559;
  for (size_t e = 0; e < E; ++e)
    for (size_t i = 0; i < M; ++i) {
      double* x = out->data() + (e * M + i) * N * 3;
      for (size_t n = 1; n < N; ++n) {
        const uint32_t ctr[4] = {(uint32_t)n, 0u, (uint32_t)e, (3u << 24) | (uint32_t)i};
        uint32_t w[4];
        host_philox(ctr, seeds[e], w);
        const double z = (double)(2ll * (long long)w[0] + 1ll - 4294967296ll) * (1.0 / 4294967296.0);
        const double phi = two_pi * (((double)w[1] + 0.5) * (1.0 / 4294967296.0));
        const double s = sqrt(1.0 - z * z);
        x[3 * n + 0] = x[3 * (n - 1) + 0] + p.r0 * (s * cos(phi));
        x[3 * n + 1] = x[3 * (n - 1) + 1] + p.r0 * (s * sin(phi));
        x[3 * n + 2] = x[3 * (n - 1) + 2] + p.r0 * z;
      }
    }
}

bool params_ok(const pt_params* p, std::string* why)
{
  if (!p) { *why = "params is NULL"; return false; }
  if (p->N < 2) { *why = "N must be >= 2"; return false; }
  if (p->M < 1 || p->M >= (1 << 24)) { *why = "M must be in [1, 2^24)"; return false; }
  if (p->E < 1) { *why = "E must be >= 1"; return false; }
  if ((int64_t)p->E * p->M > (int64_t)1 << 28) { *why = "E*M too large"; return false; }
  if (p->precision != PT_F64 && p->precision != PT_F32) { *why = "unknown precision"; return false; }
  if (p->select_mode != PT_SEQUENTIAL && p->select_mode != PT_RANDOM_PICK) { *why = "unknown select_mode"; return false; }
  if (p->nbins < 0) { *why = "nbins must be >= 0"; return false; }
  if (p->nbins > 0 && !(p->hist_emin < p->hist_emax && isfinite(p->hist_emin) && isfinite(p->hist_emax))) {
    *why = "histogram range must satisfy emin < emax"; return false;
  }
  switch (p->lanes) { case 0: case 8: case 16: case 32: case 64: case 128: case 256: break;
    default: *why = "lanes must be 0, 8, 16, 32, 64, 128 or 256"; return false; }
  if (!(p->eps > 0.0) || !isfinite(p->eps)) { *why = "eps must be > 0"; return false; }
  if (!(p->r0 > 0.0) || !isfinite(p->r0)) { *why = "r0 must be > 0"; return false; }
  if (!(p->R > 0.0) || !isfinite(p->R)) { *why = "R must be > 0"; return false; }
  if (!(p->K > 0.0) || !isfinite(p->K)) { *why = "K must be > 0"; return false; }
  if (!(p->rc_over_sigma > 0.0) || !isfinite(p->rc_over_sigma)) { *why = "rc_over_sigma must be > 0"; return false; }
  return true;
}

// Device workspace layout; every array 256-byte aligned.
struct Layout {
  uint64_t coords, erun, tos, sot, beta, width, keys, hist, mom, obs, mcount, scount, done, staging,
      e_by_temp, e_full, total;
};

Layout make_layout(const pt_params* p)
{
  const uint64_t C = (uint64_t)p->E * p->M, N = p->N, M = p->M, E = p->E;
  const uint64_t Ng = (N + 1) / 2 * 2;
  const uint64_t rb = p->precision == PT_F32 ? 4 : 8;
  Layout L{};
  uint64_t o = 0;
  auto take = [&](uint64_t bytes) { uint64_t at = o; o = align_up(o + bytes, 256); return at; };
  L.coords = take(C * 3 * Ng * rb);
  L.erun = take(C * 8);
  L.tos = take(C * 4);
  L.sot = take(C * 4);
  L.beta = take(M * 8);
  L.width = take(M * 8);
  L.keys = take(E * 8);
  L.hist = take(C * (uint64_t)(p->nbins + 2) * 8);
  L.mom = take(C * 3 * 8);
  L.obs = take(C * PT_NOBS * 8);
  L.mcount = take(C * 3 * 8);
  L.scount = take(E * (M > 1 ? M - 1 : 1) * 2 * 8);
  L.done = take(E * 4);
  L.staging = take(C * N * 3 * 8);
  L.e_by_temp = take(C * 8);
  L.e_full = take(C * 8);
  L.total = o;
  return L;
}

int create_common(pt_handle** out, const pt_params* p, const double* T, const double* widths, void* stream,
                  void* ws, uint64_t ws_bytes, bool own)
{
  std::string why;
  if (!out) return fail(nullptr, PT_EINVAL, "out is NULL");
  *out = nullptr;
  if (!params_ok(p, &why)) return fail(nullptr, PT_EINVAL, why);
  if (!T || !widths) return fail(nullptr, PT_EINVAL, "temperatures / move_halfwidths is NULL");
  for (int i = 0; i < p->M; ++i) {
    if (!(T[i] > 0.0) || !isfinite(T[i])) return fail(nullptr, PT_EINVAL, "temperatures must be finite and > 0");
    if (!(widths[i] > 0.0) || !isfinite(widths[i])) return fail(nullptr, PT_EINVAL, "move_halfwidths must be finite and > 0");
  }
  const Layout L = make_layout(p);
  if (!own) {
    if (!ws) return fail(nullptr, PT_EINVAL, "device_ws is NULL");
    if ((uintptr_t)ws % 256 != 0) return fail(nullptr, PT_EINVAL, "device_ws must be 256-byte aligned");
    if (ws_bytes < L.total) return fail(nullptr, PT_EINVAL, "device_ws is smaller than pt_workspace_bytes");
  }
  pt_handle* h = new (std::nothrow) pt_handle();
  if (!h) return fail(nullptr, PT_ENOMEM, "host allocation failed");
  h->p = *p;
  h->device = 0;
  {
    // the handle lives on the device that is current now (with a workspace: the device that owns it)
    cudaError_t ge = cudaGetDevice(&h->device);
    if (ge == cudaSuccess && !own) {
      cudaPointerAttributes at{};
      if (cudaPointerGetAttributes(&at, ws) == cudaSuccess && at.type == cudaMemoryTypeDevice) {
        if (at.device != h->device) {
          delete h;
          return fail(nullptr, PT_EINVAL, "device_ws lives on another device than the current one");
        }
      }
    }
    cudaGetLastError();
  }
  h->stream = (cudaStream_t)stream;
  h->owns_ws = own;
  h->initialised = false;
  h->t = h->x = 0;
  h->launches = 0;
  if (own) {
    cudaError_t e = cudaMalloc(&h->ws, L.total);
    if (e != cudaSuccess) {
      const int code = (e == cudaErrorMemoryAllocation) ? PT_ENOMEM : PT_ECUDA;
      const std::string msg = std::string("cudaMalloc: ") + cudaGetErrorString(e);
      delete h;
      return fail(nullptr, code, msg);
    }
    h->ws_bytes = L.total;
  } else {
    h->ws = ws;
    h->ws_bytes = ws_bytes;
  }
  char* base = (char*)h->ws;
  PtDev& d = h->d;
  memset(&d, 0, sizeof(d));
  d.N = p->N; d.M = p->M; d.E = p->E; d.C = p->E * p->M;
  d.Ng = (p->N + 1) / 2 * 2;
  d.nbins = p->nbins; d.select_mode = p->select_mode; d.observables = p->observables != 0;
  d.hist_emin = p->hist_emin;
  d.hist_scale = p->nbins > 0 ? (double)p->nbins / (p->hist_emax - p->hist_emin) : 0.0;
  // model constants: sigma = 2^(-1/6) r0, r_c = 2.5 sigma
  const double sigma = p->r0 / pow(2.0, 1.0 / 6.0);
  const double sigma2 = sigma * sigma;
  const double rc = p->rc_over_sigma * sigma;
  const double sigma6 = sigma2 * sigma2 * sigma2;
  const double wc = sigma2 / (rc * rc), s6c = wc * wc * wc;
  d.sigma2 = sigma2;
  d.eps4 = 4.0 * p->eps;
  d.ljA = 4.0 * p->eps * sigma6 * sigma6;
  d.ljB = 4.0 * p->eps * sigma6;
  d.ljC = 4.0 * p->eps * (s6c * s6c - s6c);
  d.rc2 = rc * rc;
  d.r0 = p->r0; d.R = p->R; d.invR = 1.0 / p->R;
  d.feneC = -0.5 * p->K * p->R * p->R;
  d.coords = base + L.coords;
  d.erun = (double*)(base + L.erun);
  d.temp_of_slot = (int*)(base + L.tos);
  d.slot_of_temp = (int*)(base + L.sot);
  d.beta = (const double*)(base + L.beta);
  d.width = (const double*)(base + L.width);
  d.keys = (const uint2*)(base + L.keys);
  d.hist = (unsigned long long*)(base + L.hist);
  d.mom = (double*)(base + L.mom);
  d.obs = (double*)(base + L.obs);
  d.mcount = (unsigned long long*)(base + L.mcount);
  d.scount = (unsigned long long*)(base + L.scount);
  d.done = (unsigned*)(base + L.done);
  h->staging = (double*)(base + L.staging);
  h->e_by_temp = (double*)(base + L.e_by_temp);
  h->e_full = (double*)(base + L.e_full);

  auto destroy = [&](int code, const std::string& msg) {
    if (own) cudaFree(h->ws);
    delete h;
    return fail(nullptr, code, msg);
  };
  cudaError_t e = pt_plan_sweep(d, p->precision, p->lanes, &h->plan);
  if (e != cudaSuccess) return destroy(PT_EINVAL, "no sweep-kernel mapping fits shared memory for this N / lanes");
  std::vector<double> beta(p->M);
  for (int i = 0; i < p->M; ++i) beta[i] = 1.0 / T[i];   // beta = 1/(k_B T), k_B = 1
  e = cudaMemcpyAsync((void*)d.beta, beta.data(), p->M * 8, cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync((void*)d.width, widths, p->M * 8, cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return destroy(PT_ECUDA, std::string("upload of temperatures: ") + cudaGetErrorString(e));
  *out = h;
  return PT_OK;
}

}  // namespace

extern "C" {

uint64_t pt_workspace_bytes(const pt_params* p)
{
  std::string why;
  if (!params_ok(p, &why)) return 0;
  return make_layout(p).total;
}

int pt_create(pt_handle** out, const pt_params* p, const double* temperatures, const double* move_halfwidths,
              void* cuda_stream)
{
  return create_common(out, p, temperatures, move_halfwidths, cuda_stream, nullptr, 0, true);
}

int pt_create_with_workspace(pt_handle** out, const pt_params* p, const double* temperatures,
                             const double* move_halfwidths, void* cuda_stream, void* device_ws, uint64_t ws_bytes)
{
  return create_common(out, p, temperatures, move_halfwidths, cuda_stream, device_ws, ws_bytes, false);
}

int pt_destroy(pt_handle* h)
{
  if (!h) return PT_OK;
  {
    DeviceGuard guard(h->device);
    cudaStreamSynchronize(h->stream);
    if (h->owns_ws) cudaFree(h->ws);
  }
  delete h;
  return PT_OK;
}

int pt_init(pt_handle* h, const uint64_t* seeds, const double* conformations)
{
  if (!h) return PT_EINVAL;
  if (!seeds) return fail(h, PT_EINVAL, "seeds is NULL");
  PT_ENTER(h);
  const PtDev& d = h->d;
  h->initialised = false;
  const size_t C = (size_t)d.C, N = (size_t)d.N;
  std::vector<double> walk;
  if (!conformations) {   // the library's own start: a seeded random walk of bond length r0
    host_random_walk(h->p, seeds, &walk);
    conformations = walk.data();
  }
  for (size_t q = 0; q < C * N * 3; ++q)
    if (!isfinite(conformations[q])) return fail(h, PT_EBOND, "a conformation has a non-finite coordinate");
  std::vector<uint2> keys(d.E);
  for (int e = 0; e < d.E; ++e) keys[e] = make_uint2((uint32_t)(seeds[e] & 0xFFFFFFFFull), (uint32_t)(seeds[e] >> 32));
  PT_CUDA(h, cudaMemcpyAsync((void*)d.keys, keys.data(), (size_t)d.E * 8, cudaMemcpyHostToDevice, h->stream));
  PT_CUDA(h, cudaMemcpyAsync(h->staging, conformations, C * N * 3 * 8, cudaMemcpyHostToDevice, h->stream));
  PT_CUDA(h, cudaMemsetAsync(d.done, 0, (size_t)d.E * 4, h->stream));
  PT_CUDA(h, pt_launch_scatter_init(d, h->p.precision, h->staging, h->stream));
  PT_CUDA(h, pt_launch_full_energy(d, h->p.precision, d.erun, h->stream));
  h->launches += 3;
  std::vector<double> e0(C);
  PT_CUDA(h, cudaMemcpyAsync(e0.data(), d.erun, C * 8, cudaMemcpyDeviceToHost, h->stream));
  PT_CUDA(h, cudaStreamSynchronize(h->stream));
  for (size_t c = 0; c < C; ++c)
    if (!isfinite(e0[c])) {
      char buf[160];
      snprintf(buf, sizeof buf, "chain %zu (ensemble %zu, temperature %zu) has a non-finite energy: a bond with |r - r0| >= R?",
               c, c / d.M, c % d.M);
      return fail(h, PT_EBOND, buf);
    }
  h->t = 0; h->x = 0;
  h->initialised = true;
  return PT_OK;
}

int pt_sweeps(pt_handle* h, int64_t n)
{
  if (!h) return PT_EINVAL;
  if (!h->initialised) return fail(h, PT_ESTATE, "pt_sweeps before pt_init");
  PT_ENTER(h);
  if (n < 0) return fail(h, PT_EINVAL, "n must be >= 0");
  if (h->t + n > 0xFFFFFFFFll) return fail(h, PT_ERANGE, "sweep counter would exceed 2^32 - 1");
  // one launch numbers its steps 0 .. chunk N - 1 (+ 8 drawn ahead) in an int
  const int64_t max_chunk = (2147483647ll - 16) / h->d.N;
  while (n > 0) {
    const int chunk = (int)(n > max_chunk ? max_chunk : n);
    PT_CUDA(h, pt_launch_sweep(h->d, h->p.precision, h->plan, (uint32_t)h->t, chunk, h->stream));
    h->launches += 1;
    h->t += chunk;
    n -= chunk;
  }
  return PT_OK;
}

int pt_exchange(pt_handle* h)
{
  if (!h) return PT_EINVAL;
  if (!h->initialised) return fail(h, PT_ESTATE, "pt_exchange before pt_init");
  PT_ENTER(h);
  if (h->x + 1 > 0xFFFFFFFFll) return fail(h, PT_ERANGE, "exchange counter would exceed 2^32 - 1");
  // Re-basing of the running energy (reading R22).  The paper's kernel recomputed the whole
  // energy after every sweep (Listing 2) and so carried no history; E_run += dE keeps the
  // absolute rounding of the largest energy a chain ever held (a random-walk start with overlaps: 1e10
  // and beyond).  Before the events x = 0, 1, 3, 7, ... (x + 1 a power of two) E_run is replaced by the
  // Eq.-4 sum of the current conformation, before the swap test reads it.  The fp32 path, whose
  // increments are only fp32-accurate (drift ~ sqrt(steps)), also does so every 8th event.
  const bool rebase = ((h->x + 1) & h->x) == 0 ||
                      (h->p.precision == PT_F32 && h->x % PT_F32_REFRESH_EVENTS == PT_F32_REFRESH_EVENTS - 1);
  if (rebase) {
    PT_CUDA(h, pt_launch_full_energy(h->d, h->p.precision, h->d.erun, h->stream));
    h->launches += 1;
  }
  PT_CUDA(h, pt_launch_exchange(h->d, (uint32_t)h->x, h->stream));
  if ((h->d.M - (int)(h->x & 1)) / 2 > 0) h->launches += 1;
  h->x += 1;
  return PT_OK;
}

int pt_run(pt_handle* h, int64_t n_sweeps, int64_t exchange_every)
{
  if (!h) return PT_EINVAL;
  if (!h->initialised) return fail(h, PT_ESTATE, "pt_run before pt_init");
  if (n_sweeps < 0) return fail(h, PT_EINVAL, "n_sweeps must be >= 0");
  int64_t done = 0;
  while (done < n_sweeps) {
    int64_t n = exchange_every;
    if (n <= 0 || n > n_sweeps - done) n = n_sweeps - done;
    const bool exchange_follows = exchange_every > 0 && n == exchange_every;
    // k_sweep_ws does the exchange itself at the end of the launch (the last CTA of every ensemble to finish), unless
    // the running energies are re-based first (pt_exchange) or the sweeps need more than one launch
    const bool rebase = ((h->x + 1) & h->x) == 0 ||
                        (h->p.precision == PT_F32 && h->x % PT_F32_REFRESH_EVENTS == PT_F32_REFRESH_EVENTS - 1);
    const bool fuse = exchange_follows && (h->plan.kind == PT_K_WS || h->plan.kind == PT_K_WSG) && !rebase && n > 0 &&
                      n <= (2147483647ll - 16) / h->d.N && h->x + 1 <= 0xFFFFFFFFll;
    h->plan.fuse_exchange = fuse ? 1 : 0;
    h->plan.x = (unsigned)h->x;
    int rc = pt_sweeps(h, n);
    h->plan.fuse_exchange = 0;
    if (rc != PT_OK) return rc;
    done += n;
    if (fuse) {
      h->x += 1;
    } else if (exchange_follows) {
      rc = pt_exchange(h);
      if (rc != PT_OK) return rc;
    }
  }
  return PT_OK;
}

int pt_read(pt_handle* h, double* energies, uint64_t* histograms, double* moments, uint64_t* move_counts,
            uint64_t* swap_counts, double* conformations, double* obs_moments)
{
  if (!h) return PT_EINVAL;
  if (!h->initialised) return fail(h, PT_ESTATE, "pt_read before pt_init");
  PT_ENTER(h);
  const PtDev& d = h->d;
  const size_t C = (size_t)d.C, N = (size_t)d.N, M = (size_t)d.M, E = (size_t)d.E;
  if (energies || conformations) {
    PT_CUDA(h, pt_launch_gather(d, h->p.precision, d.erun, energies ? h->e_by_temp : nullptr,
                                conformations ? h->staging : nullptr, h->stream));
    h->launches += 1;
    if (energies) PT_CUDA(h, cudaMemcpyAsync(energies, h->e_by_temp, C * 8, cudaMemcpyDeviceToHost, h->stream));
    if (conformations)
      PT_CUDA(h, cudaMemcpyAsync(conformations, h->staging, C * N * 3 * 8, cudaMemcpyDeviceToHost, h->stream));
  }
  if (histograms)
    PT_CUDA(h, cudaMemcpyAsync(histograms, d.hist, C * (size_t)(d.nbins + 2) * 8, cudaMemcpyDeviceToHost, h->stream));
  if (moments) PT_CUDA(h, cudaMemcpyAsync(moments, d.mom, C * 3 * 8, cudaMemcpyDeviceToHost, h->stream));
  if (move_counts) PT_CUDA(h, cudaMemcpyAsync(move_counts, d.mcount, C * 3 * 8, cudaMemcpyDeviceToHost, h->stream));
  if (swap_counts && M > 1)
    PT_CUDA(h, cudaMemcpyAsync(swap_counts, d.scount, E * (M - 1) * 2 * 8, cudaMemcpyDeviceToHost, h->stream));
  if (obs_moments) PT_CUDA(h, cudaMemcpyAsync(obs_moments, d.obs, C * PT_NOBS * 8, cudaMemcpyDeviceToHost, h->stream));
  PT_CUDA(h, cudaStreamSynchronize(h->stream));
  return PT_OK;
}

int pt_recompute_energy(pt_handle* h, double* energies_full)
{
  if (!h) return PT_EINVAL;
  if (!h->initialised) return fail(h, PT_ESTATE, "pt_recompute_energy before pt_init");
  PT_ENTER(h);
  if (!energies_full) return fail(h, PT_EINVAL, "energies_full is NULL");
  const PtDev& d = h->d;
  PT_CUDA(h, pt_launch_full_energy(d, h->p.precision, h->e_full, h->stream));
  PT_CUDA(h, pt_launch_gather(d, h->p.precision, h->e_full, h->e_by_temp, nullptr, h->stream));
  h->launches += 2;
  PT_CUDA(h, cudaMemcpyAsync(energies_full, h->e_by_temp, (size_t)d.C * 8, cudaMemcpyDeviceToHost, h->stream));
  PT_CUDA(h, cudaStreamSynchronize(h->stream));
  return PT_OK;
}

int pt_reset_stats(pt_handle* h)
{
  if (!h) return PT_EINVAL;
  if (!h->initialised) return fail(h, PT_ESTATE, "pt_reset_stats before pt_init");
  PT_ENTER(h);
  PT_CUDA(h, pt_launch_zero_stats(h->d, h->stream));
  h->launches += 1;
  return PT_OK;
}

int pt_set_trace(pt_handle* h, int64_t cap_sweeps, int64_t cap_events, uint8_t* move_dec, uint8_t* swap_dec,
                 double* e_trace)
{
  if (!h) return PT_EINVAL;
  if (cap_sweeps < 0 || cap_events < 0) return fail(h, PT_EINVAL, "trace capacities must be >= 0");
  h->d.tr_move = move_dec;
  h->d.tr_swap = swap_dec;
  h->d.tr_e = e_trace;
  h->d.cap_sweeps = cap_sweeps;
  h->d.cap_events = cap_events;
  return PT_OK;
}

int pt_counters(const pt_handle* h, int64_t* t_sweeps, int64_t* x_events)
{
  if (!h) return PT_EINVAL;
  if (t_sweeps) *t_sweeps = h->t;
  if (x_events) *x_events = h->x;
  return PT_OK;
}

int pt_set_counters(pt_handle* h, int64_t t_sweeps, int64_t x_events)
{
  if (!h) return PT_EINVAL;
  if (!h->initialised) return fail(h, PT_ESTATE, "pt_set_counters before pt_init");
  if (t_sweeps < 0 || x_events < 0 || t_sweeps > 0xFFFFFFFFll || x_events > 0xFFFFFFFFll)
    return fail(h, PT_ERANGE, "counters must lie in [0, 2^32)");
  h->t = t_sweeps;
  h->x = x_events;
  return PT_OK;
}

int pt_launch_info(const pt_handle* h, int32_t* lanes, int32_t* chains_per_cta, int32_t* grid, int32_t* smem_bytes)
{
  if (!h) return PT_EINVAL;
  if (lanes) *lanes = h->plan.lanes;
  if (chains_per_cta) *chains_per_cta = h->plan.chains_per_cta;
  if (grid) *grid = h->plan.grid;
  if (smem_bytes) *smem_bytes = h->plan.smem_bytes;
  return PT_OK;
}

int pt_sweep_kernel_name(const pt_handle* h, char* buf, uint64_t n)
{
  if (!h || !buf || n == 0) return PT_EINVAL;
  pt_sweep_kernel_desc(h->plan, h->p.precision, h->d.tr_move != nullptr, buf, (size_t)n);
  return PT_OK;
}

int64_t pt_kernel_launches(const pt_handle* h) { return h ? h->launches : 0; }

const char* pt_last_error(const pt_handle* h) { return h ? h->err.c_str() : g_create_err.c_str(); }

}  // extern "C"
