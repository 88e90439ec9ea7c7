"""lbm_check_finite_static: the allocation-free, synchronisation-free twin of lbm_check_finite whose
reduction scratch is a file-scope device array inside libplb.so (include/plb.h).  Collected last
on purpose (the suite runs with pytest -x).  The existing path (lbm_check_finite, scratch in the
caller's workspace, one atomic counter) is the reference: integer counts, so the bar is equality."""
import numpy as np
import pytest
import torch

from paper_1312_2234_b200 import binding as plb

pytestmark = pytest.mark.gpu


def static_count(sim, out):
    plb.lbm_check_finite_static(sim.h, out)
    return int(out.item())                                   # .item() waits for the stream


def test_static_scratch_count_matches_existing_path_on_consecutive_calls():
    """two (and more) calls in a row on changing states: every call must return what the existing
    path returns, whatever the previous call left in the shared scratch array"""
    n = (40, 24, 36)                                         # 34,560 cells = 135 blocks: several partial sums, ragged tail
    sim = plb.Simulation(*n, 0.7, (0, 1, 0))
    out = torch.full((1,), -7, dtype=torch.int32, device=sim.device)
    with pytest.raises(plb.PlbError) as e:
        plb.lbm_check_finite_static(sim.h, out)              # populations not set yet
    assert e.value.code == plb.PLB_ERR_ORDER
    sim.set_equilibrium()
    for _ in range(3):
        sim.step(None)
    with pytest.raises(plb.PlbError) as e:
        plb.lbm_check_finite_static(sim.h, None)
    assert e.value.code == plb.PLB_ERR_ARG
    clean = sim.read_populations().clone()
    cells = n[0] * n[1] * n[2]
    rng = np.random.default_rng(127)
    # call 1: many bad cells spread over all blocks (non-finite populations and non-positive densities)
    f = clean.clone()
    bad_nan = torch.as_tensor(rng.choice(cells, 700, replace=False), device=f.device)
    bad_neg = torch.as_tensor(rng.choice(cells, 300, replace=False), device=f.device)
    f[5, bad_nan] = float("nan")
    f[18, bad_neg] = -2.0
    sim.write_populations(f)
    want1 = sim.check_finite()
    assert want1 >= 700
    assert static_count(sim, out) == want1
    # call 2, right after: a different, much smaller count (stale partial sums must not leak)
    f = clean.clone()
    f[2, cells - 1] = float("inf")                           # the very last cell: the ragged last block
    f[18, 7] = -2.0
    sim.write_populations(f)
    want2 = sim.check_finite()
    assert want2 == 2
    assert static_count(sim, out) == want2
    # call 3 and 4 back to back on one stream without reading in between, healthy state
    sim.write_populations(clean)
    out2 = torch.full((1,), -7, dtype=torch.int32, device=sim.device)
    plb.lbm_check_finite_static(sim.h, out)
    plb.lbm_check_finite_static(sim.h, out2)
    assert int(out.item()) == 0 and int(out2.item()) == 0 == sim.check_finite()
    sim.close()


def test_static_scratch_serves_a_second_context_and_refuses_large_grids():
    """the array is shared by every context on the device; a grid beyond the stated maximum is refused"""
    a = plb.Simulation(16, 12, 10, 0.7, (0, 1, 0))
    b = plb.Simulation(64, 8, 20, 0.8, (0, 0, 0))
    out = torch.zeros(1, dtype=torch.int32, device=a.device)
    for sim, poisoned in ((a, 3), (b, 11), (a, 1)):
        sim.set_equilibrium()
        f = sim.read_populations().clone()
        f[0, :poisoned] = float("nan")
        sim.write_populations(f)
        torch.cuda.synchronize()                             # calls sharing the array must not overlap
        assert static_count(sim, out) == sim.check_finite() == poisoned
    a.close(); b.close()
    assert plb_max_cells() == 16777216
    big = plb.Simulation(256, 256, 257, 0.7, (0, 0, 0))      # 16,842,752 cells > 16,777,216
    big.set_equilibrium()
    with pytest.raises(plb.PlbError) as e:
        plb.lbm_check_finite_static(big.h, out)
    assert e.value.code == plb.PLB_ERR_WORKSPACE
    assert big.check_finite() == 0                           # the existing path has no such limit
    big.close()
    fits = plb.Simulation(256, 256, 256, 0.7, (0, 0, 0))     # exactly the maximum: 65,536 blocks
    fits.set_equilibrium()
    f = fits.read_populations()
    f[3, 256 * 256 * 256 - 1] = float("nan")
    f[3, 12345] = float("nan")
    fits.write_populations(f)
    del f
    assert static_count(fits, out) == fits.check_finite() == 2
    fits.close()


def plb_max_cells():
    """the limit include/plb.h states (PLB_STATIC_MAX_CELLS), read from the header"""
    import os
    import re
    here = os.path.dirname(os.path.abspath(__file__))
    text = open(os.path.join(here, "..", "include", "plb.h")).read()
    return int(re.search(r"#define\s+PLB_STATIC_MAX_CELLS\s+(\d+)L", text).group(1))
