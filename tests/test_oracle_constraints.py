"""Pins for the area / volume constraint forces of the CPU oracle (
PAPER.md Eq. 4-5, force = -dH/dX per Eq. 11 read with the minus sign, G2).
Expected values: exact polyhedra, closed-form sphere / spheroid surface and volume, finite
differences of the energy, invariances.  None comes from the oracle's force code or from CUDA."""
import math

import numpy as np
import pytest

from oracle import orc
from paper_1312_2234_b200 import workloads as wl


def box():
    return orc.Oracle(8, 8, 8, 0.8)


CUBE_V = np.array([[0, 0, 0], [1, 0, 0], [1, 1, 0], [0, 1, 0], [0, 0, 1], [1, 0, 1], [1, 1, 1], [0, 1, 1]], dtype=float)
CUBE_T = np.array([[0, 2, 1], [0, 3, 2], [4, 5, 6], [4, 6, 7], [0, 1, 5], [0, 5, 4],
                   [1, 2, 6], [1, 6, 5], [2, 3, 7], [2, 7, 6], [3, 0, 4], [3, 4, 7]], dtype=np.int32)
NO_EDGES = np.zeros((0, 2), dtype=np.int32)


def mesh_oracle(xyz, tris, ref=None, k_s=0.0, k_t=0.0, k_v=0.0, edges=NO_EDGES, k=0.0):
    o = box()
    o.add_mesh(xyz, edges, None, k)
    o.set_triangles(0, tris, ref, k_s, k_t, k_v)
    return o


# ------------------------------------------------------------------ S and V
@pytest.mark.parametrize("shift", [0.0, 517.25])
def test_cube_and_tetrahedron_exact(shift):
    """exact polyhedra, also far from the origin (V is translation invariant for a closed surface)"""
    o = mesh_oracle(2.0 * CUBE_V + shift, CUBE_T)
    S, V = o.mesh_area_volume(0)
    assert S == pytest.approx(24.0, rel=1e-13) and V == pytest.approx(8.0, rel=1e-10)
    tet = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=float) + shift   # edge 2 sqrt 2
    tt = np.array([[0, 1, 2], [0, 3, 1], [0, 2, 3], [1, 3, 2]], dtype=np.int32)
    o = mesh_oracle(tet, tt)
    S, V = o.mesh_area_volume(0)
    a = 2 * math.sqrt(2)
    assert S == pytest.approx(math.sqrt(3) * a * a, rel=1e-13)
    assert V == pytest.approx(a ** 3 / (6 * math.sqrt(2)), rel=1e-10)


def test_inward_orientation_is_rejected():
    o = box()
    o.add_mesh(CUBE_V, NO_EDGES, None, 0.0)
    with pytest.raises(orc.OracleError):
        o.set_triangles(0, CUBE_T[:, ::-1], None, 1.0, 1.0, 1.0)


def test_icosphere_converges_to_the_sphere_at_second_order():
    r = 3.0
    errS, errV = [], []
    for s in (1, 2, 3):
        v, t, _ = wl.icosphere(s)
        S, V = mesh_oracle(r * v + 4.0, t).mesh_area_volume(0)
        errS.append(4 * math.pi * r * r - S)
        errV.append(4 * math.pi * r ** 3 / 3 - V)
    assert all(e > 0 for e in errS + errV)                    # inscribed polyhedron
    for e in (errS, errV):
        assert 3.5 < e[0] / e[1] < 4.5 and 3.7 < e[1] / e[2] < 4.3
    assert errS[2] / (4 * math.pi * r * r) < 5e-3 and errV[2] / (4 * math.pi * r ** 3 / 3) < 1e-2


def test_oblate_ellipsoid_matches_the_spheroid_closed_forms():
    """the platelet shape of L81 with the configs' semi-axes (6, 6, 1.5)"""
    a, c = 6.0, 1.5
    e = math.sqrt(1 - c * c / (a * a))
    S_exact = 2 * math.pi * a * a * (1 + (1 - e * e) / e * math.atanh(e))
    V_exact = 4 * math.pi * a * a * c / 3
    v, t, _ = wl.icosphere(4)
    S, V = mesh_oracle(v * np.array([a, a, c]) + 20.0, t).mesh_area_volume(0)
    assert S == pytest.approx(S_exact, rel=4e-3) and S < S_exact
    assert V == pytest.approx(V_exact, rel=4e-3) and V < V_exact


# ------------------------------------------------------------------ forces
def perturbed_icosphere(seed, subdiv=1, r=2.5, amp=0.15):
    v, t, e = wl.icosphere(subdiv)
    rng = np.random.default_rng(seed)
    ref = r * v * np.array([1.0, 1.0, 0.6]) + np.array([3.3, 4.1, 3.7])
    return ref, ref + amp * rng.standard_normal(ref.shape), t, e


@pytest.mark.parametrize("ks,kt,kv", [(0.7, 0, 0), (0, 0.5, 0), (0, 0, 0.9), (0.3, 0.4, 0.6)])
def test_force_is_minus_gradient_of_the_energy(ks, kt, kv):
    ref, X, t, _ = perturbed_icosphere(7)
    o = mesh_oracle(X, t, ref, ks, kt, kv)
    o.compute_membrane_forces()
    F = o.read_forces()
    assert np.abs(F).max() > 1e-3
    d = 1e-6
    for m, comp in [(0, 0), (5, 1), (17, 2), (30, 0), (41, 1)]:
        Xp = X.copy(); Xp[m, comp] += d
        Xm = X.copy(); Xm[m, comp] -= d
        o.write_nodes(Xp); Hp = o.area_volume_energy()
        o.write_nodes(Xm); Hm = o.area_volume_energy()
        assert F[m, comp] == pytest.approx(-(Hp - Hm) / (2 * d), rel=2e-7, abs=1e-9)


def test_energy_matches_its_definition_on_a_scaled_cube():
    """cube of side 1 stretched to side L: S_tot = 6 L^2, each triangle L^2/2, V = L^3"""
    L, ks, kt, kv = 1.1, 0.3, 0.2, 0.5
    o = mesh_oracle(L * CUBE_V + 2.0, CUBE_T, CUBE_V + 2.0, ks, kt, kv)
    H = ks * (6 * L * L - 6) ** 2 / (2 * 6) + 12 * kt * (L * L / 2 - 0.5) ** 2 / (2 * 0.5) + kv * (L ** 3 - 1) ** 2 / 2
    assert o.area_volume_energy() == pytest.approx(H, rel=1e-12)


def test_forces_sum_to_zero_and_carry_no_torque():
    ref, X, t, _ = perturbed_icosphere(9, subdiv=2)
    o = mesh_oracle(X, t, ref, 0.3, 0.4, 0.6)
    o.compute_membrane_forces()
    F = o.read_forces()
    scale = np.abs(F).sum()
    assert np.abs(F.sum(0)).max() <= 1e-13 * scale
    assert np.abs(np.cross(X, F).sum(0)).max() <= 1e-12 * scale


def test_unstressed_shape_feels_no_force_wherever_it_is():
    ref, _, t, _ = perturbed_icosphere(3)
    rot = wl.rot_x(0.7)
    X = ref @ rot.T + np.array([0.4, -0.3, 0.2])
    o = mesh_oracle(X, t, ref, 0.3, 0.4, 0.6)
    o.compute_membrane_forces()
    assert np.abs(o.read_forces()).max() <= 1e-13


@pytest.mark.parametrize("ks,kt,kv", [(1, 0, 0), (0, 1, 0), (0, 0, 1)])
def test_inflated_sphere_is_pushed_back_in(ks, kt, kv):
    v, t, _ = wl.icosphere(2)
    c0 = np.array([4.0, 4.0, 4.0])
    o = mesh_oracle(1.05 * 2.0 * v + c0, t, 2.0 * v + c0, ks, kt, kv)
    o.compute_membrane_forces()
    F = o.read_forces()
    radial = (F * v).sum(1)
    assert (radial < 0).all()
    assert np.abs(F - radial[:, None] * v).max() <= 0.05 * np.abs(radial).max()


def test_springs_and_constraints_add_and_other_meshes_are_untouched():
    ref, X, t, e = perturbed_icosphere(5)
    a = box(); a.add_mesh(X, e, wl.edge_lengths(ref, e), 0.02); a.compute_membrane_forces()
    b = mesh_oracle(X, t, ref, 0.3, 0.4, 0.6); b.compute_membrane_forces()
    both = box()
    both.add_mesh(X + 0.0, e, wl.edge_lengths(ref, e), 0.02)
    both.add_mesh(X, e, wl.edge_lengths(ref, e), 0.02)          # second mesh: springs only
    both.set_triangles(0, t, ref, 0.3, 0.4, 0.6)
    both.compute_membrane_forces()
    F = both.read_forces()
    n = X.shape[0]
    assert np.allclose(F[:n], a.read_forces() + b.read_forces(), rtol=0, atol=1e-15)
    assert np.allclose(F[n:], a.read_forces(), rtol=0, atol=1e-15)
