"""GPU-vs-oracle parity for the area / volume constraint forces (PAPER.md
Eq. 4-5), through the C-ABI.  The oracle side is pinned in tests/test_oracle_constraints.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import orc                                    # noqa: E402
from paper_1312_2234_b200 import binding as plb            # noqa: E402
from paper_1312_2234_b200 import workloads as wl           # noqa: E402
import parity_utils as pu                                  # noqa: E402


def deformed_meshes(seed, n_meshes, subdiv, centre_scale):
    """n_meshes randomly placed, randomly rotated, randomly deformed (6, 6, 1.5) ellipsoids"""
    rng = np.random.default_rng(seed)
    v, tris, edges = wl.icosphere(subdiv)
    ref = v * np.array([6.0, 6.0, 1.5])
    R = wl.random_rotations(rng, n_meshes)
    xyz = np.einsum("mab,nb->mna", R, ref) + centre_scale * rng.random((n_meshes, 1, 3))
    xyz = xyz + 0.08 * rng.standard_normal(xyz.shape)
    return ref, xyz, tris, edges


@pytest.mark.parametrize("subdiv,n_meshes", [(1, 3), (2, 5), (3, 2)])
@pytest.mark.parametrize("ks,kt,kv", [(0.09, 0.0, 0.0), (0.0, 0.09, 0.0), (0.0, 0.0, 0.09), (0.088, 0.088, 0.088)])
def test_constraint_forces_match_oracle(subdiv, n_meshes, ks, kt, kv):
    """positions up to ~1000 lattice units from the origin (the C4 box is 512 x 128 x 1024)"""
    ref, xyz, tris, edges = deformed_meshes(100 + subdiv, n_meshes, subdiv, np.array([500.0, 100.0, 1000.0]))
    nn = ref.shape[0]
    sim = plb.Simulation(8, 8, 8, 0.8, max_nodes=n_meshes * nn, max_edges=n_meshes * len(edges))
    ora = orc.Oracle(8, 8, 8, 0.8)
    first = sim.add_meshes(xyz, edges, wl.edge_lengths(ref, edges), 0.0)
    sim.set_triangles(first, n_meshes, tris, ref, ks, kt, kv)
    for m in range(n_meshes):
        ora.add_mesh(xyz[m], edges, wl.edge_lengths(ref, edges), 0.0)
        ora.set_triangles(m, tris, ref, ks, kt, kv)
    sim.compute_membrane_forces()
    ora.compute_membrane_forces()
    F_g, F_o = sim.read_forces().astype(np.float64), ora.read_forces()
    scale = np.abs(F_o).max()
    assert scale > 1e-4
    assert np.abs(F_g - F_o).max() <= 2e-6 * scale
    sim.close(); ora.close()


def test_springs_constraints_and_noise_add_up():
    ref, xyz, tris, edges = deformed_meshes(7, 4, 2, np.array([100.0, 50.0, 100.0]))
    nn = ref.shape[0]
    rest = wl.edge_lengths(ref, edges)
    sim = plb.Simulation(8, 8, 8, 0.8, max_nodes=4 * nn, max_edges=4 * len(edges))
    ora = orc.Oracle(8, 8, 8, 0.8)
    first = sim.add_meshes(xyz, edges, rest, 0.02)
    sim.set_triangles(first + 1, 2, tris, ref, 0.088, 0.088, 0.088)     # meshes 1, 2 only
    for m in range(4):
        ora.add_mesh(xyz[m], edges, rest, 0.02)
        if m in (1, 2):
            ora.set_triangles(m, tris, ref, 0.088, 0.088, 0.088)
    sim.compute_membrane_forces(1e-4, 99, 3)
    ora.compute_membrane_forces(1e-4, 99, 3)
    F_g, F_o = sim.read_forces().astype(np.float64), ora.read_forces()
    assert np.abs(F_g - F_o).max() <= 2e-6 * np.abs(F_o).max()
    sim.close(); ora.close()


def test_null_reference_takes_the_current_shape_and_gives_no_force():
    ref, xyz, tris, edges = deformed_meshes(9, 3, 2, np.array([60.0, 60.0, 60.0]))
    nn = ref.shape[0]
    sim = plb.Simulation(8, 8, 8, 0.8, max_nodes=3 * nn, max_edges=3 * len(edges))
    first = sim.add_meshes(xyz, edges, None, 0.0)
    sim.set_triangles(first, 3, tris, None, 0.1, 0.1, 0.1)
    sim.compute_membrane_forces()
    assert np.abs(sim.read_forces()).max() <= 1e-7
    sim.close()


def test_argument_and_order_errors():
    ref, xyz, tris, edges = deformed_meshes(9, 2, 1, np.array([6.0, 6.0, 6.0]))
    nn = ref.shape[0]
    sim = plb.Simulation(8, 8, 8, 0.8, max_nodes=2 * nn + 5, max_edges=2 * len(edges) + 4)
    first = sim.add_meshes(xyz, edges, None, 0.0)
    bad = tris.copy(); bad[0, 0] = nn
    for args in ((first, 2, bad, ref), (first, 3, tris, ref), (first, 2, tris[:, ::-1], ref)):
        with pytest.raises(plb.PlbError) as e:
            sim.set_triangles(*args, 0.1, 0.1, 0.1)
        assert e.value.code == plb.PLB_ERR_ARG
    sim.set_triangles(first, 1, tris, ref, 0.1, 0.1, 0.1)
    with pytest.raises(plb.PlbError) as e:                      # once per mesh
        sim.set_triangles(first, 2, tris, ref, 0.1, 0.1, 0.1)
    assert e.value.code == plb.PLB_ERR_ORDER
    other = sim.add_mesh(np.array([[1.0, 1, 1], [2, 1, 1], [1, 2, 1], [1, 1, 2], [2, 2, 2]]), np.array([[0, 1]], dtype=np.int32))
    with pytest.raises(plb.PlbError) as e:                      # meshes of different size in one call
        sim.set_triangles(first + 1, 2, tris, ref, 0.1, 0.1, 0.1)
    assert e.value.code == plb.PLB_ERR_ARG
    sim.close()


def test_coupled_config1_constrained_whole():
    """config 1 with the paper's area / volume constraints on (k ratios of Table 2), 200 coupled
    steps at the north_star tolerances"""
    w = wl.with_area_volume_constraints(wl.config1())
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, w.steps)
    print("C1-constrained", pu.compare(w, sim, ora))
    sim.close(); ora.close()


def test_coupled_config4_scaled_constrained_with_onsite_walls():
    """the paper's own membrane + wall together: springs + area/volume constraints, Hecht-Harting walls"""
    w = wl.with_onsite_walls(wl.with_area_volume_constraints(wl.config4(nx=96, ny=48, nz=128, n_meshes=12, steps=150)))
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, w.steps)
    print("C4-scaled constrained on-site", pu.compare(w, sim, ora))
    sim.close(); ora.close()
