"""GPU-vs-oracle parity for SURVEY.md NEXT-4: the stochastic dynamic adhesion model (PAPER.md section
3.2, Eq. 12-14, rules L147-149) and the wall repulsion (L246), through the C-ABI.

Bond tables are integer state: they must be BIT-EXACT (both sides evaluate the probabilities in fp64
and compare them with the same Philox uniform).  Forces are fp32 on the GPU: relative 2e-6."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import orc                                    # noqa: E402
from paper_1312_2234_b200 import binding as plb            # noqa: E402
from paper_1312_2234_b200 import workloads as wl           # noqa: E402
import parity_utils as pu                                  # noqa: E402

PRM = dict(wall_axis=1, max_per_site=4, k_on0=0.3, k_off0=0.05, s=3.0, gamma=0.2, sigma=0.05, l_b=0.3, l_max=0.64,
           F0=2e-4, tau_rep=4.0)


def pair(xyz, nx=24, ny=8, nz=20, kind=(0, 1, 0)):
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = xyz.shape[0]
    no_edges = np.zeros((0, 2), dtype=np.int32)
    sim = plb.Simulation(nx, ny, nz, 0.8, kind, max_nodes=n, max_edges=0)
    sim.set_equilibrium()
    sim.add_mesh(xyz, no_edges)
    ora = orc.Oracle(nx, ny, nz, 0.8, kind)
    ora.set_equilibrium()
    ora.add_mesh(xyz, no_edges, None, 0.0)
    return sim, ora


def near_wall_cloud(rng, n, nx, nz, plane=-0.5):
    return np.stack([-3 + (nx + 6) * rng.random(n), plane + 0.02 + 0.9 * rng.random(n), -3 + (nz + 6) * rng.random(n)], axis=1)


@pytest.mark.parametrize("n_rec,min_total,min_on", [(8000, 8000, 300), (20000, 20000, 500)])
@pytest.mark.parametrize("kind,plane", [((0, 1, 0), -0.5), ((0, 2, 0), 0.0)])
def test_bond_tables_are_bit_exact_over_many_updates(kind, plane, n_rec, min_total, min_on):
    """3000 nodes jittering near the wall (some across the periodic seams), 8000 or 20,000
    receptors (the larger case puts dozens of same-step candidates on one site), 30 updates with
    the same positions on both sides: break, form, contention for the 4 places"""
    rng = np.random.default_rng(41)
    nx, nz = 24, 20
    xyz = near_wall_cloud(rng, 3000, nx, nz, plane)
    sim, ora = pair(xyz, nx=nx, nz=nz, kind=kind)
    rec = rng.integers(0, 3000, size=n_rec)
    sim.set_receptors(rec, PRM); ora.set_receptors(rec, PRM)
    total = 0
    for step in range(30):
        sim.adhesion_update(1234, step); ora.adhesion_update(1234, step)
        bg, bo = sim.read_bonds(), ora.read_bonds()
        assert (bg == bo).all(), (step, int((bg != bo).any(axis=1).sum()))
        total += int(bo[:, 0].sum())
        xyz = xyz + 0.05 * rng.standard_normal(xyz.shape)
        xyz[:, 1] = np.clip(xyz[:, 1], plane + 0.01, None)
        sim.write_nodes(xyz); ora.write_nodes(xyz)
    on = bo[bo[:, 0] == 1]
    assert total > min_total and len(on) > min_on                      # plenty of bonds formed and broke
    _, counts = np.unique((on[:, 1] % nx) + nx * (on[:, 2] % nz), return_counts=True)
    assert counts.max() == 4                                            # rule 2 was binding somewhere
    sim.close(); ora.close()


def test_contention_lowest_indices_win_and_overflow_is_reported():
    prm = dict(PRM, k_on0=1e9, k_off0=0.0, F0=0.0)
    xyz = [[3.2, -0.1, 5.3], [9.0, 4.0, 9.0]]
    sim, ora = pair(xyz)
    node = np.zeros(30, dtype=np.int32); node[25:] = 1
    sim.set_receptors(node, prm); ora.set_receptors(node, prm)
    for step in range(3):
        sim.adhesion_update(1, step); ora.adhesion_update(1, step)
        assert (sim.read_bonds() == ora.read_bonds()).all()
    assert sim.read_bonds()[:, 0].tolist() == [1] * 4 + [0] * 26
    b = sim.read_bonds(); b[1] = 0; b[3] = 0
    sim.write_bonds(b); ora.write_bonds(b)
    sim.adhesion_update(1, 9); ora.adhesion_update(1, 9)
    assert (sim.read_bonds() == ora.read_bonds()).all() and sim.read_bonds()[:4, 0].tolist() == [1, 1, 1, 1]
    sim.close(); ora.close()
    # any number of same-step candidates for one site: 500 receptors on one node, 4 places
    sim, ora = pair(xyz)
    node = np.zeros(500, dtype=np.int32)
    sim.set_receptors(node, prm); ora.set_receptors(node, prm)
    sim.adhesion_update(1, 0); ora.adhesion_update(1, 0)
    sim.status()
    assert (sim.read_bonds() == ora.read_bonds()).all() and sim.read_bonds()[:, 0].tolist() == [1] * 4 + [0] * 496
    sim.close(); ora.close()


def test_bond_and_repulsion_forces_match_oracle():
    rng = np.random.default_rng(43)
    nx, nz = 24, 20
    xyz = near_wall_cloud(rng, 2000, nx, nz)
    sim, ora = pair(xyz, nx=nx, nz=nz)
    rec = rng.integers(0, 2000, size=9000)
    sim.set_receptors(rec, PRM); ora.set_receptors(rec, PRM)
    b = np.zeros((9000, 3), dtype=np.int32)
    b[:, 0] = rng.random(9000) < 0.5
    b[:, 1] = np.round(xyz[rec, 0]) + rng.integers(-2, 3, size=9000)
    b[:, 2] = np.round(xyz[rec, 2]) + rng.integers(-2, 3, size=9000)
    b[b[:, 0] == 0, 1:] = 0
    sim.write_bonds(b); ora.write_bonds(b)
    assert (sim.read_bonds() == b).all()
    sim.compute_membrane_forces(); ora.compute_membrane_forces()
    Fg, Fo = sim.read_forces().astype(np.float64), ora.read_forces()
    scale = np.abs(Fo).max()
    assert scale > 1e-3
    assert np.abs(Fg - Fo).max() <= 2e-6 * scale, np.abs(Fg - Fo).max() / scale
    sim.close(); ora.close()


def test_wall_on_the_z_axis():
    """wall axis 2: sites on the (x, y) lattice of the low z face"""
    rng = np.random.default_rng(47)
    n = 1500
    xyz = np.stack([-2 + 20 * rng.random(n), -2 + 16 * rng.random(n), -0.5 + 0.02 + 0.8 * rng.random(n)], axis=1)
    sim, ora = pair(xyz, nx=16, ny=12, nz=8, kind=(0, 0, 1))
    rec = rng.integers(0, n, size=4000)
    prm = dict(PRM, wall_axis=2)
    sim.set_receptors(rec, prm); ora.set_receptors(rec, prm)
    for step in range(8):
        sim.adhesion_update(77, step); ora.adhesion_update(77, step)
        assert (sim.read_bonds() == ora.read_bonds()).all(), step
    sim.compute_membrane_forces(); ora.compute_membrane_forces()
    Fg, Fo = sim.read_forces().astype(np.float64), ora.read_forces()
    assert ora.read_bonds()[:, 0].sum() > 200
    assert np.abs(Fg - Fo).max() <= 2e-6 * np.abs(Fo).max()
    sim.close(); ora.close()


def test_node_through_the_wall_is_reported():
    sim, ora = pair([[3.0, -0.6, 3.0]])
    sim.set_receptors([0], PRM)
    sim.compute_membrane_forces()
    with pytest.raises(plb.PlbError) as e:
        sim.status()
    assert e.value.code == plb.PLB_ERR_NODE_LEFT
    sim.close(); ora.close()


def test_call_order_and_arguments():
    sim, ora = pair([[3.0, 0.2, 3.0]])
    with pytest.raises(plb.PlbError) as e:
        sim.adhesion_update(0, 0)
    assert e.value.code == plb.PLB_ERR_ORDER
    with pytest.raises(plb.PlbError) as e:
        sim.set_receptors([0], dict(PRM, wall_axis=0))          # x is periodic: not a wall axis
    assert e.value.code == plb.PLB_ERR_ARG
    with pytest.raises(plb.PlbError) as e:
        sim.set_receptors([5], PRM)                             # node out of range
    assert e.value.code == plb.PLB_ERR_ARG
    sim.close(); ora.close()


def test_bad_parameters_and_bad_bonds_are_refused():
    """F0 > 0 needs tau_rep > 0 (F_rep would be 0/0); a bond to a site outside a non-periodic
    tangential axis is refused before it reaches the device table"""
    sim = plb.Simulation(12, 8, 10, 0.8, (1, 1, 0), max_nodes=2, max_edges=0)
    sim.set_equilibrium()
    sim.add_mesh(np.array([[3.0, 0.1, 3.0], [5.5, 2.0, 4.0]]), np.zeros((0, 2), dtype=np.int32))
    with pytest.raises(plb.PlbError) as e:
        sim.set_receptors([0, 1], dict(PRM, F0=1e-4, tau_rep=0.0))
    assert e.value.code == plb.PLB_ERR_ARG
    sim.set_receptors([0, 1], PRM)
    ok = np.array([[1, 3, 3], [0, 0, 0]], dtype=np.int32)
    sim.write_bonds(ok)
    for bad in ([[1, -1, 3], [0, 0, 0]], [[1, 12, 3], [0, 0, 0]]):      # x is a wall axis here: sites 0..11 only
        with pytest.raises(plb.PlbError) as e:
            sim.write_bonds(np.array(bad, dtype=np.int32))
        assert e.value.code == plb.PLB_ERR_ARG
    assert (sim.read_bonds() == ok).all()                               # the table still holds the last good one
    sim.adhesion_update(1, 0)
    sim.status()
    sim.close()


def test_no_receptors_leaves_only_the_repulsion():
    """empty receptor list: the update is a no-op, the bond table is empty, every node still feels F_rep"""
    xyz = np.array([[3.0, 0.1, 3.0], [5.5, 2.0, 4.0]])
    sim, ora = pair(xyz)
    none = np.zeros(0, dtype=np.int32)
    sim.set_receptors(none, PRM); ora.set_receptors(none, PRM)
    sim.adhesion_update(3, 0); ora.adhesion_update(3, 0)
    assert sim.read_bonds().shape == (0, 3)
    sim.compute_membrane_forces(); ora.compute_membrane_forces()
    Fg, Fo = sim.read_forces().astype(np.float64), ora.read_forces()
    assert (Fo[:, 1] > 0).all() and np.abs(Fo[:, [0, 2]]).max() == 0.0
    assert np.abs(Fg - Fo).max() <= 2e-6 * np.abs(Fo).max()
    sim.close(); ora.close()


def test_adhering_platelets_coupled_parity():
    """the NEXT-4 workload (4 platelets flat on the wall, 5344 receptors each, constraints on), 120
    coupled steps with the Monte-Carlo update after every advance: north_star tolerances on the
    fields and node positions, identical bond tables"""
    w = wl.adhering_platelets(nx=48, ny=24, nz=48, n_side=2, steps=120)
    assert w.receptor_node.shape[0] == 4 * 5344
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, w.steps)
    out = pu.compare(w, sim, ora)
    bg, bo = sim.read_bonds(), ora.read_bonds()
    out["bonds"] = int(bo[:, 0].sum())
    out["bond_mismatch"] = int((bg != bo).any(axis=1).sum())
    print("adhering platelets", out)
    assert out["bonds"] > 200
    assert out["bond_mismatch"] == 0
    sim.close(); ora.close()
