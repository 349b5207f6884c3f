"""Thin ctypes binding of libpt_b200.so: argument marshalling only.

Function names are those of include/pt_b200.h.  Every step of the path (sweeps, exchange,
accumulation, full energy) runs in the library's CUDA kernels; PyTorch is used here only for
device memory (the workspace, the trace buffers) and for the stream.  There is no CPU
fallback: if the library is missing it is built with nvcc, and if that fails the import of
this module fails.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from . import build as _build

PT_F64, PT_F32 = 0, 1
PT_SEQUENTIAL, PT_RANDOM_PICK = 0, 1
PT_OK, PT_EINVAL, PT_ESTATE, PT_EBOND, PT_ENOMEM, PT_ECUDA, PT_ERANGE = 0, -1, -2, -3, -4, -5, -6
_ERRNAMES = {-1: "PT_EINVAL", -2: "PT_ESTATE", -3: "PT_EBOND", -4: "PT_ENOMEM", -5: "PT_ECUDA",
             -6: "PT_ERANGE"}

# every symbol include/pt_b200.h declares
SYMBOLS = ("pt_workspace_bytes", "pt_create", "pt_create_with_workspace", "pt_destroy", "pt_init",
           "pt_sweeps", "pt_exchange", "pt_run", "pt_read", "pt_recompute_energy", "pt_reset_stats",
           "pt_set_trace", "pt_counters", "pt_set_counters", "pt_launch_info", "pt_sweep_kernel_name",
           "pt_kernel_launches", "pt_last_error",
           "pt_fma_peak", "pt_energy_noalloc", "pt_noalloc_last_error")


class PtParams(C.Structure):
    """pt_params of include/pt_b200.h"""
    _fields_ = [
        ("N", C.c_int32), ("M", C.c_int32), ("E", C.c_int32), ("precision", C.c_int32),
        ("select_mode", C.c_int32), ("nbins", C.c_int32), ("observables", C.c_int32),
        ("lanes", C.c_int32),
        ("hist_emin", C.c_double), ("hist_emax", C.c_double),
        ("eps", C.c_double), ("r0", C.c_double), ("R", C.c_double), ("K", C.c_double),
        ("rc_over_sigma", C.c_double),
    ]


class PtError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_ERRNAMES.get(code, code)}: {msg}")
        self.code = code


_lib = None


def lib_path() -> Path:
    return _build.LIB


def lib():
    """Loads (building first if stale) libpt_b200.so and declares the C signatures."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(str(path))
    dp, u64p, u8p, i32p, i64p = (C.POINTER(C.c_double), C.POINTER(C.c_uint64), C.POINTER(C.c_uint8),
                                 C.POINTER(C.c_int32), C.POINTER(C.c_int64))
    pp, hp = C.POINTER(PtParams), C.c_void_p
    L.pt_workspace_bytes.argtypes = [pp]; L.pt_workspace_bytes.restype = C.c_uint64
    L.pt_create.argtypes = [C.POINTER(hp), pp, dp, dp, C.c_void_p]; L.pt_create.restype = C.c_int
    L.pt_create_with_workspace.argtypes = [C.POINTER(hp), pp, dp, dp, C.c_void_p, C.c_void_p, C.c_uint64]
    L.pt_create_with_workspace.restype = C.c_int
    L.pt_destroy.argtypes = [hp]; L.pt_destroy.restype = C.c_int
    L.pt_init.argtypes = [hp, u64p, dp]; L.pt_init.restype = C.c_int
    L.pt_sweeps.argtypes = [hp, C.c_int64]; L.pt_sweeps.restype = C.c_int
    L.pt_exchange.argtypes = [hp]; L.pt_exchange.restype = C.c_int
    L.pt_run.argtypes = [hp, C.c_int64, C.c_int64]; L.pt_run.restype = C.c_int
    L.pt_read.argtypes = [hp, dp, u64p, dp, u64p, u64p, dp, dp]; L.pt_read.restype = C.c_int
    L.pt_recompute_energy.argtypes = [hp, dp]; L.pt_recompute_energy.restype = C.c_int
    L.pt_reset_stats.argtypes = [hp]; L.pt_reset_stats.restype = C.c_int
    L.pt_set_trace.argtypes = [hp, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
    L.pt_set_trace.restype = C.c_int
    L.pt_counters.argtypes = [hp, i64p, i64p]; L.pt_counters.restype = C.c_int
    L.pt_set_counters.argtypes = [hp, C.c_int64, C.c_int64]; L.pt_set_counters.restype = C.c_int
    L.pt_launch_info.argtypes = [hp, i32p, i32p, i32p, i32p]; L.pt_launch_info.restype = C.c_int
    L.pt_sweep_kernel_name.argtypes = [hp, C.c_char_p, C.c_uint64]; L.pt_sweep_kernel_name.restype = C.c_int
    L.pt_kernel_launches.argtypes = [hp]; L.pt_kernel_launches.restype = C.c_int64
    L.pt_last_error.argtypes = [hp]; L.pt_last_error.restype = C.c_char_p
    L.pt_fma_peak.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, dp]; L.pt_fma_peak.restype = C.c_int
    _lib = L
    return L


def make_params(N, M=1, E=1, precision=PT_F64, select_mode=PT_SEQUENTIAL, nbins=0, observables=0,
                lanes=0, hist_emin=0.0, hist_emax=1.0, eps=1.0, r0=0.7, R=0.3, K=40.0,
                rc_over_sigma=2.5) -> PtParams:
    """Defaults are the paper's model constants."""
    return PtParams(int(N), int(M), int(E), int(precision), int(select_mode), int(nbins),
                    int(observables), int(lanes), float(hist_emin), float(hist_emax), float(eps),
                    float(r0), float(R), float(K), float(rc_over_sigma))


def _ptr(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def _check(h, rc):
    if rc != PT_OK:
        msg = lib().pt_last_error(h)
        raise PtError(rc, msg.decode() if msg else "")


PT_NOALLOC_MAX_CHAINS = 8192


def pt_energy_noalloc(params: PtParams, dev_conformations, dev_energies, n_chains: int, stream=None):
    """pt_energy_noalloc of include/pt_b200.h: torch CUDA tensors (fp64, contiguous) in and out, nothing allocated."""
    L = lib()
    L.pt_energy_noalloc.argtypes = [C.POINTER(PtParams), C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
    L.pt_energy_noalloc.restype = C.c_int
    L.pt_noalloc_last_error.restype = C.c_char_p
    rc = L.pt_energy_noalloc(C.byref(params), C.c_void_p(dev_conformations.data_ptr() if dev_conformations is not None else 0),
                             C.c_void_p(dev_energies.data_ptr() if dev_energies is not None else 0), int(n_chains),
                             C.c_void_p(stream.cuda_stream if stream is not None else 0))
    if rc != PT_OK:
        msg = L.pt_noalloc_last_error()
        raise PtError(rc, msg.decode() if msg else "")


def pt_workspace_bytes(params: PtParams) -> int:
    return int(lib().pt_workspace_bytes(C.byref(params)))


def pt_fma_peak(precision=PT_F64, iters=4096, reps=5, stream=None) -> float:
    """Measured plain FMA rate of the current device in TFLOP/s (roofline denominator)."""
    out = C.c_double(0.0)
    sptr = C.c_void_p(stream.cuda_stream) if stream is not None else None
    rc = lib().pt_fma_peak(int(precision), int(iters), int(reps), sptr, C.byref(out))
    if rc != PT_OK:
        raise PtError(rc, "pt_fma_peak failed (no CUDA device?)")
    return out.value


class ParallelTempering:
    """One handle of the C ABI.  Methods carry the names of the C entry points."""

    def __init__(self, params: PtParams, temperatures, move_halfwidths, stream=None,
                 torch_workspace: bool = True):
        self.p = params
        self.T = np.ascontiguousarray(temperatures, dtype=np.float64)
        self.w = np.ascontiguousarray(move_halfwidths, dtype=np.float64)
        if self.T.shape != (params.M,) or self.w.shape != (params.M,):
            raise ValueError("temperatures and move_halfwidths must have shape (M,)")
        self._h = C.c_void_p()
        self._ws = None
        self._trace = {}
        self._stream = stream
        sptr = C.c_void_p(stream.cuda_stream) if stream is not None else None
        L = lib()
        if torch_workspace:
            import torch
            nbytes = pt_workspace_bytes(params)
            if nbytes == 0:
                _check(None, L.pt_create(C.byref(self._h), C.byref(params), _ptr(self.T, C.c_double),
                                         _ptr(self.w, C.c_double), sptr))
            if not torch.cuda.is_available():
                raise PtError(PT_ECUDA, "no CUDA device: the path has no CPU fallback")
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
            base = (self._ws.data_ptr() + 255) // 256 * 256
            rc = L.pt_create_with_workspace(C.byref(self._h), C.byref(params), _ptr(self.T, C.c_double),
                                            _ptr(self.w, C.c_double), sptr, C.c_void_p(base),
                                            C.c_uint64(nbytes))
        else:
            rc = L.pt_create(C.byref(self._h), C.byref(params), _ptr(self.T, C.c_double),
                             _ptr(self.w, C.c_double), sptr)
        _check(None, rc)

    # -- lifetime -------------------------------------------------------------------------
    def pt_destroy(self):
        if self._h:
            lib().pt_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None
            self._trace = {}

    close = pt_destroy

    def __del__(self):
        try:
            self.pt_destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.pt_destroy()

    # -- the path -------------------------------------------------------------------------
    def pt_init(self, seeds, conformations=None):
        """conformations = None: the library's own seeded random walk (read it back with pt_read)."""
        p = self.p
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        conf = None if conformations is None else np.ascontiguousarray(conformations, dtype=np.float64)
        if seeds.shape != (p.E,) or (conf is not None and conf.shape != (p.E, p.M, p.N, 3)):
            raise ValueError("seeds must be (E,), conformations (E, M, N, 3)")
        _check(self._h, lib().pt_init(self._h, _ptr(seeds, C.c_uint64), _ptr(conf, C.c_double)))

    def pt_sweeps(self, n: int):
        _check(self._h, lib().pt_sweeps(self._h, int(n)))

    def pt_exchange(self):
        _check(self._h, lib().pt_exchange(self._h))

    def pt_run(self, n_sweeps: int, exchange_every: int):
        _check(self._h, lib().pt_run(self._h, int(n_sweeps), int(exchange_every)))

    def pt_read(self, energies=True, histograms=True, moments=True, move_counts=True, swap_counts=True,
                conformations=True, obs_moments=True) -> dict:
        p = self.p
        out = {}
        if energies:
            out["energies"] = np.zeros((p.E, p.M), dtype=np.float64)
        if histograms:
            out["histograms"] = np.zeros((p.E, p.M, p.nbins + 2), dtype=np.uint64)
        if moments:
            out["moments"] = np.zeros((p.E, p.M, 3), dtype=np.float64)
        if move_counts:
            out["move_counts"] = np.zeros((p.E, p.M, 3), dtype=np.uint64)
        if swap_counts:
            out["swap_counts"] = np.zeros((p.E, max(p.M - 1, 0), 2), dtype=np.uint64)
        if conformations:
            out["conformations"] = np.zeros((p.E, p.M, p.N, 3), dtype=np.float64)
        if obs_moments:
            out["obs_moments"] = np.zeros((p.E, p.M, 5), dtype=np.float64)
        sc = out.get("swap_counts")
        _check(self._h, lib().pt_read(
            self._h, _ptr(out.get("energies"), C.c_double), _ptr(out.get("histograms"), C.c_uint64),
            _ptr(out.get("moments"), C.c_double), _ptr(out.get("move_counts"), C.c_uint64),
            _ptr(sc, C.c_uint64) if (sc is not None and p.M > 1) else None,
            _ptr(out.get("conformations"), C.c_double), _ptr(out.get("obs_moments"), C.c_double)))
        return out

    def pt_read_into(self, energies=None, histograms=None, moments=None, move_counts=None,
                     swap_counts=None, conformations=None, obs_moments=None):
        """pt_read into caller-allocated (e.g. pinned) NumPy arrays; None = skip."""
        _check(self._h, lib().pt_read(
            self._h, _ptr(energies, C.c_double), _ptr(histograms, C.c_uint64), _ptr(moments, C.c_double),
            _ptr(move_counts, C.c_uint64), _ptr(swap_counts, C.c_uint64),
            _ptr(conformations, C.c_double), _ptr(obs_moments, C.c_double)))

    def pt_recompute_energy(self) -> np.ndarray:
        out = np.zeros((self.p.E, self.p.M), dtype=np.float64)
        _check(self._h, lib().pt_recompute_energy(self._h, _ptr(out, C.c_double)))
        return out

    def pt_reset_stats(self):
        _check(self._h, lib().pt_reset_stats(self._h))

    # -- test support ---------------------------------------------------------------------
    def pt_set_trace(self, cap_sweeps: int, cap_events: int = 0, moves=True, swaps=True, energy=True):
        """Allocates the trace buffers as torch device tensors and hands their pointers over."""
        import torch
        p = self.p
        t = {}
        if moves and cap_sweeps > 0:
            t["move"] = torch.zeros((p.E, p.M, cap_sweeps, p.N), dtype=torch.uint8, device="cuda")
        if swaps and p.M > 1 and cap_events > 0:
            t["swap"] = torch.zeros((p.E, cap_events, p.M - 1), dtype=torch.uint8, device="cuda")
        if energy and cap_sweeps > 0:
            t["energy"] = torch.zeros((p.E, p.M, cap_sweeps), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        self._trace = t
        ptr = lambda k: C.c_void_p(t[k].data_ptr()) if k in t else None
        _check(self._h, lib().pt_set_trace(self._h, int(cap_sweeps), int(cap_events), ptr("move"),
                                           ptr("swap"), ptr("energy")))

    def trace(self, ensembles=None) -> dict:
        """Host copies of the trace buffers (synchronises); `ensembles`: indices to copy (None = all)."""
        import torch
        if self._stream is not None:
            self._stream.synchronize()
        torch.cuda.synchronize()
        if ensembles is None:
            return {k: v.cpu().numpy() for k, v in self._trace.items()}
        idx = torch.as_tensor(list(ensembles), dtype=torch.long, device="cuda")
        return {k: v.index_select(0, idx).cpu().numpy() for k, v in self._trace.items()}

    def pt_counters(self):
        t, x = C.c_int64(0), C.c_int64(0)
        _check(self._h, lib().pt_counters(self._h, C.byref(t), C.byref(x)))
        return t.value, x.value

    def pt_set_counters(self, t_sweeps: int, x_events: int):
        _check(self._h, lib().pt_set_counters(self._h, int(t_sweeps), int(x_events)))

    def pt_launch_info(self) -> dict:
        a, b, c, d = C.c_int32(0), C.c_int32(0), C.c_int32(0), C.c_int32(0)
        _check(self._h, lib().pt_launch_info(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
        return {"lanes": a.value, "chains_per_cta": b.value, "grid": c.value, "smem_bytes": d.value}

    def pt_sweep_kernel_name(self) -> str:
        buf = C.create_string_buffer(128)
        _check(self._h, lib().pt_sweep_kernel_name(self._h, buf, C.c_uint64(len(buf))))
        return buf.value.decode()

    def pt_kernel_launches(self) -> int:
        return int(lib().pt_kernel_launches(self._h))
