"""pt_energy_noalloc (include/pt_b200.h): the one entry point that allocates nothing -- Eq. (4) energies with its
scratch in a static device array of the library -- against the existing path, pt_recompute_energy, whose scratch lives in
the handle's workspace.  Two calls in a row share the scratch array: the second must not see anything of the first.
The file name keeps this test last in the collection order (the suite runs with pytest -x)."""
import numpy as np
import pytest

import paper_1107_3490_b200 as pt
from paper_1107_3490_b200 import binding, synth

pytestmark = pytest.mark.gpu

REL_TOL = 1e-9   # the energy tolerance of the parity tests: |a - b| <= 1e-9 max(1, |b|)


def _existing_path(N, M, E, conf):
    """pt_recompute_energy on a handle initialised with these conformations: [E][M] energies by temperature index."""
    T = synth.temperature_ladder(M, 0.3, 2.5)
    p = pt.make_params(N, M, E, nbins=0)
    with pt.ParallelTempering(p, T, synth.move_halfwidths(T)) as sim:
        sim.pt_init(synth.seeds(17, E), conf)
        return sim.pt_recompute_energy()


def test_no_alloc_energy_matches_recompute_energy_twice_in_a_row():
    import torch
    torch.cuda.set_device(0)
    # two different batches, the larger first, so that stale partial sums and counters would be noticed:
    # 37 monomers (rows left over in every slice of the pair sum) x 600 chains, then 100 monomers x 64 chains
    cases = [(37, 8, 75, 4101), (100, 64, 1, 4102)]
    confs = [synth.random_walk_conformations(E, M, N, seed=seed) for N, M, E, seed in cases]
    expected = [_existing_path(N, M, E, c) for (N, M, E, _), c in zip(cases, confs)]
    dev_in = [torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in confs]
    dev_out = [torch.full((E * M,), float("nan"), dtype=torch.float64, device="cuda") for N, M, E, _ in cases]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for (N, M, E, _), x, out in zip(cases, dev_in, dev_out):      # two calls in a row, nothing in between
        binding.pt_energy_noalloc(pt.make_params(N, M, E), x, out, E * M)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    for (N, M, E, _), out, exp in zip(cases, dev_out, expected):
        got = out.cpu().numpy().reshape(E, M)
        assert np.isfinite(got).all()
        assert np.all(np.abs(got - exp) <= REL_TOL * np.maximum(1.0, np.abs(exp))), float(np.max(np.abs(got - exp)))
    # the same batch again: identical bits (the partial sums are added in a fixed order)
    again = torch.empty_like(dev_out[1])
    binding.pt_energy_noalloc(pt.make_params(*cases[1][:3]), dev_in[1], again, cases[1][1] * cases[1][2])
    torch.cuda.synchronize()
    assert torch.equal(again, dev_out[1])


def test_no_alloc_rejects_batches_beyond_the_static_scratch():
    import torch
    torch.cuda.set_device(0)
    x = torch.zeros(8, dtype=torch.float64, device="cuda")
    with pytest.raises(pt.PtError) as err:
        binding.pt_energy_noalloc(pt.make_params(5, 1, 1), x, x, binding.PT_NOALLOC_MAX_CHAINS + 1)
    assert err.value.code == binding.PT_EINVAL and "PT_NOALLOC_MAX_CHAINS" in str(err.value)
    binding.pt_energy_noalloc(pt.make_params(5, 1, 1), x, x, 0)      # an empty batch is fine and touches nothing
