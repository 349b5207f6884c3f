"""The schedule ptxas chose for the fp64 step loops of the composed kernels: no loop may be
serialised (dependent fp64 instructions 1-3 slots apart).  Static: reads the built objects with cuobjdump, no GPU."""
import shutil

import pytest

import paper_1107_3490_b200 as pt
from paper_1107_3490_b200 import sasscheck


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not installed")
def test_no_serialised_step_loop_in_the_composed_fp64_kernels():
    pt.lib()                                   # builds the library (and the objects) if stale
    objs = sorted(sasscheck.OBJ.glob("pt_sweep_comp*.o"))
    if not objs:
        pytest.skip("objects not kept (library built elsewhere)")
    bad = sasscheck.serialised("Id", objs)       # the <double, ...> instantiations of k_sweep_comp and k_sweep_seven
    assert not bad, f"ptxas serialised {len(bad)} step loop(s): {bad[:3]}"
