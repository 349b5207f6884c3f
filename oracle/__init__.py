"""CPU oracle (TEST INFRASTRUCTURE ONLY) -- ctypes loader for oracle/pt_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product package never does, and this package
never imports the product package.  See oracle/pt_oracle.h for the citations.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "pt_oracle.c"
_LIB = _HERE / "libpt_oracle.so"

CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c99", "-Wall"]


def build(force: bool = False) -> Path:
    """Compile oracle/pt_oracle.c with gcc (no tuning flags beyond -O2)."""
    hdr = _HERE / "pt_oracle.h"
    if (not force and _LIB.exists()
            and _LIB.stat().st_mtime >= max(_SRC.stat().st_mtime, hdr.stat().st_mtime)):
        return _LIB
    cmd = ["gcc", *CFLAGS, "-o", str(_LIB), str(_SRC), "-lm"]
    subprocess.run(cmd, check=True, cwd=str(_HERE))
    return _LIB


class OrcParams(C.Structure):
    _fields_ = [
        ("N", C.c_int32), ("M", C.c_int32), ("E", C.c_int32),
        ("select_mode", C.c_int32), ("nbins", C.c_int32), ("e_offset", C.c_int32),
        ("hist_emin", C.c_double), ("hist_emax", C.c_double),
        ("eps", C.c_double), ("r0", C.c_double), ("R", C.c_double), ("K", C.c_double),
        ("rc_over_sigma", C.c_double),
    ]


def make_params(N, M=1, E=1, select_mode=0, nbins=0, hist_emin=0.0, hist_emax=1.0,
                eps=1.0, r0=0.7, R=0.3, K=40.0, rc_over_sigma=2.5, e_offset=0) -> OrcParams:
    return OrcParams(N, M, E, select_mode, nbins, e_offset, hist_emin, hist_emax, eps, r0, R, K,
                     rc_over_sigma)


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = C.CDLL(str(_LIB))
    dp, u64p, u8p, u32p = (C.POINTER(C.c_double), C.POINTER(C.c_uint64),
                           C.POINTER(C.c_uint8), C.POINTER(C.c_uint32))
    pp = C.POINTER(OrcParams)
    L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
    L.orc_philox4x32_10.restype = None
    L.orc_word_to_sym.argtypes = [C.c_uint32]; L.orc_word_to_sym.restype = C.c_double
    L.orc_word_to_u01.argtypes = [C.c_uint32]; L.orc_word_to_u01.restype = C.c_double
    L.orc_lj_mod.argtypes = [pp, C.c_double]; L.orc_lj_mod.restype = C.c_double
    L.orc_fene.argtypes = [pp, C.c_double]; L.orc_fene.restype = C.c_double
    L.orc_total_energy.argtypes = [pp, dp]; L.orc_total_energy.restype = C.c_double
    L.orc_delta_energy.argtypes = [pp, dp, C.c_int, dp, C.POINTER(C.c_int)]
    L.orc_delta_energy.restype = C.c_double
    L.orc_rgyr2.argtypes = [C.c_int, dp]; L.orc_rgyr2.restype = C.c_double
    L.orc_ree2.argtypes = [C.c_int, dp]; L.orc_ree2.restype = C.c_double
    L.orc_create.argtypes = [pp, dp, dp]; L.orc_create.restype = C.c_void_p
    L.orc_destroy.argtypes = [C.c_void_p]; L.orc_destroy.restype = None
    L.orc_init.argtypes = [C.c_void_p, u64p, dp]; L.orc_init.restype = C.c_int
    L.orc_set_trace.argtypes = [C.c_void_p, C.c_int64, C.c_int64, u8p, u8p, dp, dp, dp]
    L.orc_set_trace.restype = None
    L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]; L.orc_set_threads.restype = None
    L.orc_get_threads.argtypes = [C.c_void_p]; L.orc_get_threads.restype = C.c_int
    L.orc_sweeps.argtypes = [C.c_void_p, C.c_int64]; L.orc_sweeps.restype = None
    L.orc_exchange.argtypes = [C.c_void_p]; L.orc_exchange.restype = None
    L.orc_run.argtypes = [C.c_void_p, C.c_int64, C.c_int64]; L.orc_run.restype = None
    L.orc_read.argtypes = [C.c_void_p, dp, u64p, dp, u64p, u64p, dp, dp]
    L.orc_read.restype = None
    _lib = L
    return L


def _ptr(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def lj_mod(r2, params=None):
    p = params or make_params(2)
    return lib().orc_lj_mod(C.byref(p), float(r2))


def fene(r2, params=None):
    p = params or make_params(2)
    return lib().orc_fene(C.byref(p), float(r2))


def total_energy(x, params=None):
    x = np.ascontiguousarray(x, dtype=np.float64)
    p = params or make_params(x.shape[0])
    assert x.shape == (p.N, 3)
    return lib().orc_total_energy(C.byref(p), _ptr(x, C.c_double))


def delta_energy(x, m, xnew, params=None):
    x = np.ascontiguousarray(x, dtype=np.float64)
    xnew = np.ascontiguousarray(xnew, dtype=np.float64)
    p = params or make_params(x.shape[0])
    ok = C.c_int(0)
    dE = lib().orc_delta_energy(C.byref(p), _ptr(x, C.c_double), int(m), _ptr(xnew, C.c_double),
                                C.byref(ok))
    return dE, bool(ok.value)


def rgyr2(x):
    x = np.ascontiguousarray(x, dtype=np.float64)
    return lib().orc_rgyr2(x.shape[0], _ptr(x, C.c_double))


def ree2(x):
    x = np.ascontiguousarray(x, dtype=np.float64)
    return lib().orc_ree2(x.shape[0], _ptr(x, C.c_double))


class Oracle:
    """One parallel-tempering simulation on the CPU oracle (all arrays by temperature index)."""

    def __init__(self, params: OrcParams, temperatures, widths, threads: int | None = None):
        self.p = params
        self.T = np.ascontiguousarray(temperatures, dtype=np.float64)
        self.w = np.ascontiguousarray(widths, dtype=np.float64)
        assert self.T.shape == (params.M,) and self.w.shape == (params.M,)
        self.h = lib().orc_create(C.byref(self.p), _ptr(self.T, C.c_double), _ptr(self.w, C.c_double))
        if not self.h:
            raise ValueError("orc_create rejected the parameters")
        self._trace = {}
        if threads is None:
            threads = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
        lib().orc_set_threads(self.h, int(threads))

    @property
    def threads(self) -> int:
        return lib().orc_get_threads(self.h)

    def close(self):
        if self.h:
            lib().orc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init(self, seeds, conformations):
        p = self.p
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        conf = np.ascontiguousarray(conformations, dtype=np.float64)
        assert seeds.shape == (p.E,) and conf.shape == (p.E, p.M, p.N, 3)
        rc = lib().orc_init(self.h, _ptr(seeds, C.c_uint64), _ptr(conf, C.c_double))
        if rc != 0:
            raise ValueError("orc_init: a conformation has a non-finite energy")

    def enable_trace(self, cap_sweeps: int, cap_events: int = 0, moves=True, swaps=True,
                     energy=True, obs=False):
        p = self.p
        t = {}
        if moves:
            t["move"] = np.zeros((p.E, p.M, cap_sweeps, p.N), dtype=np.uint8)
        if swaps and p.M > 1 and cap_events > 0:
            t["swap"] = np.zeros((p.E, cap_events, p.M - 1), dtype=np.uint8)
        if energy:
            t["energy"] = np.zeros((p.E, p.M, cap_sweeps), dtype=np.float64)
        if obs:
            t["ree2"] = np.zeros((p.E, p.M, cap_sweeps), dtype=np.float64)
            t["rg2"] = np.zeros((p.E, p.M, cap_sweeps), dtype=np.float64)
        self._trace = t
        lib().orc_set_trace(self.h, int(cap_sweeps), int(cap_events),
                            _ptr(t.get("move"), C.c_uint8), _ptr(t.get("swap"), C.c_uint8),
                            _ptr(t.get("energy"), C.c_double), _ptr(t.get("ree2"), C.c_double),
                            _ptr(t.get("rg2"), C.c_double))
        return t

    @property
    def trace(self):
        return self._trace

    def sweeps(self, n: int):
        lib().orc_sweeps(self.h, int(n))

    def exchange(self):
        lib().orc_exchange(self.h)

    def run(self, n_sweeps: int, exchange_every: int):
        lib().orc_run(self.h, int(n_sweeps), int(exchange_every))

    def read(self):
        p = self.p
        out = {
            "energies": np.zeros((p.E, p.M), dtype=np.float64),
            "histograms": np.zeros((p.E, p.M, p.nbins + 2), dtype=np.uint64),
            "moments": np.zeros((p.E, p.M, 3), dtype=np.float64),
            "move_counts": np.zeros((p.E, p.M, 3), dtype=np.uint64),
            "swap_counts": np.zeros((p.E, max(p.M - 1, 0), 2), dtype=np.uint64),
            "conformations": np.zeros((p.E, p.M, p.N, 3), dtype=np.float64),
            "obs_moments": np.zeros((p.E, p.M, 5), dtype=np.float64),
        }
        lib().orc_read(self.h, _ptr(out["energies"], C.c_double), _ptr(out["histograms"], C.c_uint64),
                       _ptr(out["moments"], C.c_double), _ptr(out["move_counts"], C.c_uint64),
                       _ptr(out["swap_counts"], C.c_uint64) if p.M > 1 else None,
                       _ptr(out["conformations"], C.c_double), _ptr(out["obs_moments"], C.c_double))
        return out
