"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/pt_b200.h declares; argument validation (host logic) answers without a GPU; compute calls
fail loudly (PT_ECUDA) instead of falling back to the CPU."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

import paper_1107_3490_b200 as pt
from paper_1107_3490_b200 import binding, synth

ROOT = Path(__file__).resolve().parent.parent


def _declared_symbols():
    text = (ROOT / "include" / "pt_b200.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pt_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = _declared_symbols()
    assert "pt_create" in names and "pt_read" in names and len(names) >= 15
    assert sorted(binding.SYMBOLS) == names, "binding.SYMBOLS must list exactly what the header declares"
    L = C.CDLL(str(pt.lib_path()))
    for n in names:
        assert hasattr(L, n), n


def test_params_struct_matches_header_layout():
    # 8 int32 + 7 double, no padding surprises: pt_workspace_bytes reads it correctly
    assert C.sizeof(binding.PtParams) == 8 * 4 + 7 * 8
    p = pt.make_params(100, 64, 64, nbins=4096, hist_emin=-500.0, hist_emax=300.0)
    total = pt.pt_workspace_bytes(p)
    C_ = 64 * 64
    assert total >= C_ * 3 * 100 * 8 + C_ * 4098 * 8 + C_ * 100 * 3 * 8
    assert total < 2 * (C_ * 3 * 100 * 8 + C_ * 4098 * 8 + C_ * 100 * 3 * 8)
    assert pt.pt_workspace_bytes(pt.make_params(1, 1, 1)) == 0     # N < 2 is invalid


@pytest.mark.parametrize("kw", [dict(N=1), dict(M=0), dict(E=0), dict(nbins=-1), dict(precision=7),
                                dict(select_mode=3), dict(lanes=5), dict(R=0.0), dict(eps=-1.0),
                                dict(nbins=4, hist_emin=1.0, hist_emax=1.0)])
def test_create_rejects_bad_parameters_without_a_gpu(kw):
    base = dict(N=5, M=2, E=1)
    base.update(kw)
    p = pt.make_params(**base)
    L = pt.lib()
    h = C.c_void_p()
    T = np.array([1.0, 2.0]); w = np.array([0.1, 0.1])
    rc = L.pt_create(C.byref(h), C.byref(p), T.ctypes.data_as(C.POINTER(C.c_double)),
                     w.ctypes.data_as(C.POINTER(C.c_double)), None)
    assert rc == binding.PT_EINVAL
    assert h.value is None
    assert len(L.pt_last_error(None)) > 0


def test_bad_temperatures_are_rejected_before_any_cuda_call():
    p = pt.make_params(5, 2, 1)
    L = pt.lib()
    h = C.c_void_p()
    for T, w in ((np.array([1.0, -2.0]), np.array([0.1, 0.1])), (np.array([1.0, np.nan]), np.array([0.1, 0.1])),
                 (np.array([1.0, 2.0]), np.array([0.0, 0.1])), (np.array([1.0, 2.0]), np.array([0.1, np.inf]))):
        rc = L.pt_create(C.byref(h), C.byref(p), T.ctypes.data_as(C.POINTER(C.c_double)),
                         w.ctypes.data_as(C.POINTER(C.c_double)), None)
        assert rc == binding.PT_EINVAL


def test_no_cpu_fallback():
    """Without a CUDA device creation fails with PT_ECUDA / PT_ENOMEM; with one, this test is moot."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    p = pt.make_params(5, 2, 1)
    L = pt.lib()
    h = C.c_void_p()
    T = np.array([1.0, 2.0]); w = np.array([0.1, 0.1])
    rc = L.pt_create(C.byref(h), C.byref(p), T.ctypes.data_as(C.POINTER(C.c_double)),
                     w.ctypes.data_as(C.POINTER(C.c_double)), None)
    assert rc in (binding.PT_ECUDA, binding.PT_ENOMEM)
    assert h.value is None
    out = C.c_double(0.0)
    assert L.pt_fma_peak(0, 16, 1, None, C.byref(out)) == binding.PT_ECUDA


def test_product_never_imports_the_oracle():
    for f in list((ROOT / "paper_1107_3490_b200").rglob("*.py")) + list((ROOT / "paper_1107_3490_b200" / "csrc").glob("*")):
        if f.is_file() and f.suffix in (".py", ".cu", ".cuh", ".h"):
            text = f.read_text()
            assert "import oracle" not in text and "from oracle" not in text and "pt_oracle" not in text, f


def test_synth_shapes_and_determinism():
    a, b = synth.make_inputs(1), synth.make_inputs(1)
    assert np.array_equal(a.conformations, b.conformations) and np.array_equal(a.seeds, b.seeds)
    assert a.conformations.shape == (1, 8, 13, 3)
    bonds = np.linalg.norm(np.diff(a.conformations, axis=2), axis=-1)
    assert np.allclose(bonds, 0.7, atol=1e-12)
    assert np.isclose(a.temperatures[0], 0.3) and np.isclose(a.temperatures[-1], 3.0)
    assert np.allclose(a.widths, 0.1 * np.sqrt(a.temperatures))
    sub = synth.make_inputs(5, E=2)
    assert sub.conformations.shape == (2, 64, 100, 3)
    r = [list(synth.shard_ensembles(64, 3, k)) for k in range(3)]
    assert sum(r, []) == list(range(64))
