"""GPU-vs-oracle parity for the Hecht-Harting on-site velocity wall (
PAPER.md Eq. 23-30), through the C-ABI.  The oracle side is pinned in
tests/test_oracle_hecht_harting.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import orc                                    # noqa: E402
from paper_1312_2234_b200 import binding as plb            # noqa: E402
from paper_1312_2234_b200 import workloads as wl           # noqa: E402
import parity_utils as pu                                  # noqa: E402

DEV = "cuda:0"
HH = 2


def dev(a, dtype=torch.float32):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to(DEV).contiguous()


def hh_kind(axis):
    k = [0, 0, 0]
    k[axis] = HH
    return tuple(k)


def wall_velocities(axis, seed, normal=True):
    rng = np.random.default_rng(seed)
    u_lo = np.zeros((3, 3)); u_hi = np.zeros((3, 3))
    u_lo[axis] = 0.04 * (2 * rng.random(3) - 1)
    u_hi[axis] = 0.04 * (2 * rng.random(3) - 1)
    if not normal:
        u_lo[axis, axis] = u_hi[axis, axis] = 0.0
    return u_lo, u_hi


# shapes: ragged generic path; vector path (nx % 4 == 0, x periodic) incl. a warp spanning rows
SHAPES = [(37, 19, 23), (40, 9, 11), (128, 7, 5), (8, 5, 5), (4, 2, 2)]


@pytest.mark.parametrize("n", SHAPES)
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("forced", [False, True])
def test_steps_match_oracle_on_every_face(n, axis, forced):
    cells = n[0] * n[1] * n[2]
    rho, u = wl.random_fields(211 + axis, cells)
    u_lo, u_hi = wall_velocities(axis, 5 + axis)             # incl. a wall-normal component
    sim = plb.Simulation(*n, 0.7, hh_kind(axis), u_lo, u_hi)
    ora = orc.Oracle(*n, 0.7, hh_kind(axis), u_lo, u_hi)
    sim.set_equilibrium(dev(rho), dev(u), 1e-4, 31)
    ora.set_equilibrium(rho, u, 1e-4, 31)
    # the initial state is closed on both sides (reading G25)
    f_g = sim.read_populations().cpu().numpy().astype(np.float64)
    assert np.abs(f_g - ora.read_populations()).max() <= 3e-7
    rng = np.random.default_rng(19)
    for s in range(6):
        g = 1e-3 * (2 * rng.random((3, cells)) - 1) if forced else None
        gd = pu.soa_to_forcing(sim, g) if forced else None
        sim.step(gd)
        ora.step(g)
        f_g = sim.read_populations().cpu().numpy().astype(np.float64)
        assert np.abs(f_g - ora.read_populations()).max() <= 4e-7, "step %d" % s
        rho_g, u_g = sim.read_macros()
        rho_o, u_o = ora.read_macros()
        assert np.abs(rho_g.cpu().numpy() - rho_o).max() <= 8e-7
        assert np.abs(u_g.cpu().numpy() - u_o).max() <= 8e-7
    sim.status()
    sim.close(); ora.close()


def test_population_write_read_round_trip_closes_the_wall():
    n = (12, 6, 5)
    cells = n[0] * n[1] * n[2]
    _, w = orc.lattice()
    rng = np.random.default_rng(3)
    f = w[:, None] * (1 + 0.05 * rng.standard_normal((19, cells)))
    u_lo, u_hi = wall_velocities(1, 9)
    sim = plb.Simulation(*n, 0.8, hh_kind(1), u_lo, u_hi)
    ora = orc.Oracle(*n, 0.8, hh_kind(1), u_lo, u_hi)
    sim.write_populations(dev(f).view(-1))
    ora.write_populations(f)
    back = sim.read_populations().cpu().numpy().astype(np.float64)
    assert np.abs(back - ora.read_populations()).max() <= 3e-7
    sim.close(); ora.close()


def test_couette_with_the_wall_on_the_node_on_gpu():
    nx, ny, nz, tau, uw = 8, 17, 4, 0.8, 0.05
    u_hi = np.zeros((3, 3)); u_hi[1, 0] = uw
    sim = plb.Simulation(nx, ny, nz, tau, hh_kind(1), None, u_hi)
    sim.set_equilibrium(None, None, 0.0, 0)
    for _ in range(12000):
        sim.step(None)
    rho, u = sim.read_macros()
    ux = u[0].view(nz, ny, nx).cpu().numpy()
    assert np.abs(ux - (uw * np.arange(ny) / (ny - 1))[None, :, None]).max() <= 1e-4 * uw
    assert float((rho - rho.mean()).abs().max()) <= 1e-6
    assert float(u[1:].abs().max()) <= 1e-4 * uw
    sim.close()


def test_coupled_config1_with_onsite_walls():
    """config 1 (one platelet in a Couette cell, 200 coupled steps) with the paper's own wall,
    at the north_star tolerances"""
    w = wl.with_onsite_walls(wl.config1())
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, w.steps)
    print("C1-onsite", pu.compare(w, sim, ora))
    sim.close(); ora.close()


def test_coupled_config3_scaled_with_onsite_walls():
    w = wl.with_onsite_walls(wl.config3(nx=64, ny=32, nz=128, n_meshes=4, steps=300))
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, w.steps)
    print("C3-onsite scaled", pu.compare(w, sim, ora))
    sim.close(); ora.close()


def test_node_crossing_an_onsite_wall_is_reported():
    """the on-site wall lies ON layer 0: a node pushed below y = 0 has left the channel"""
    nx, ny, nz = 16, 12, 16
    u_lo = np.zeros((3, 3)); u_lo[1] = [0.0, -0.05, 0.0]     # lower wall sucks fluid out
    sim = plb.Simulation(nx, ny, nz, 0.8, hh_kind(1), u_lo, None, max_nodes=4, max_edges=1)
    u0 = np.zeros((3, nx * ny * nz)); u0[1] = -0.05
    sim.set_equilibrium(None, dev(u0), 0.0, 0)
    xyz = np.array([[8.0, 0.02, 8.0], [8.0, 5.0, 8.0]])
    sim.add_mesh(xyz, np.array([[0, 1]], dtype=np.int32), None, 0.0)
    sim.coupled_step(0.0, 0, 0)
    with pytest.raises(plb.PlbError) as e:
        sim.status()
    assert e.value.code == plb.PLB_ERR_NODE_LEFT
    sim.close()


def test_rejected_configurations():
    for kind in ((0, HH, 1), (HH, HH, 0)):
        with pytest.raises(plb.PlbError) as e:
            plb.Simulation(8, 8, 8, 0.8, kind)
        assert e.value.code == plb.PLB_ERR_ARG
    with pytest.raises(plb.PlbError):
        plb.Simulation(8, 1, 8, 0.8, (0, HH, 0))
