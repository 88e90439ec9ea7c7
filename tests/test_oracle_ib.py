"""Pins for the immersed-boundary, spring and random-number parts of the CPU oracle:
SURVEY.md 8(c) P9-P16 and O-8.  Expected values come from the paper, closed forms, invariants,
brute force written a different way, or the published Philox known-answer vectors -- never from
the oracle itself or from the CUDA path."""
import math
import os

import numpy as np
import pytest

from oracle import orc
from paper_1312_2234_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ delta kernel (Eq. 35-36)
def test_P9_delta_kernel_identities():
    gold = [l.split("#")[0].split() for l in open(os.path.join(GOLD, "paper_constants.txt")) if l.startswith("phi_integer")][0]
    assert [orc.phi(r) for r in (1, 0, -1, -2)] == pytest.approx([float(x) for x in gold[1:]], abs=1e-16)
    assert orc.phi(2.0) == 0.0 and orc.phi(-2.0) == 0.0 and orc.phi(2.5) == 0.0 and orc.phi(-7) == 0.0
    assert orc.phi(0.3) == orc.phi(-0.3)
    h = [orc.phi(r) for r in (1.5, 0.5, -0.5, -1.5)]
    assert h == pytest.approx([0.25 * (1 - math.sqrt(0.5)), 0.25 * (1 + math.sqrt(0.5))] * 1 + [0.25 * (1 + math.sqrt(0.5)), 0.25 * (1 - math.sqrt(0.5))], abs=1e-15)
    assert h == pytest.approx([0.07322, 0.42678, 0.42678, 0.07322], abs=5e-6)
    for r in np.random.default_rng(0).random(50):
        pts = np.array([orc.phi(r - j) for j in range(-3, 5)])
        js = np.arange(-3, 5)
        assert pts.sum() == pytest.approx(1.0, abs=1e-15)                  # partition of unity
        assert (pts ** 2).sum() == pytest.approx(3.0 / 8.0, abs=1e-15)     # Peskin's sum-of-squares
        assert pts[js % 2 == 0].sum() == pytest.approx(0.5, abs=1e-15)     # even/odd balance
        assert (pts > 0).sum() <= 4


# ------------------------------------------------------------------ Philox (O-8)
def test_philox_known_answers():
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        h = [int(x, 16) for x in line.split()]
        assert orc.philox4x32_10(h[0:4], h[4:6]) == h[6:10]


def test_uniform_and_normal_variates():
    assert orc.lib().orc_uniform01(0) == 0.5 / 2 ** 24
    assert orc.lib().orc_uniform01(0xFFFFFFFF) == 1 - 0.5 / 2 ** 24
    assert orc.lib().orc_uniform01(0x80000000) == (2 ** 23 + 0.5) / 2 ** 24
    seed = 131222345
    # normals are Box-Muller of the four uniforms of the same counter
    for idx, step in ((0, 0), (12345, 7), (2 ** 33 + 5, 199)):
        xi = orc.noise_uniform(seed, idx, step, 2)
        r = orc.philox4x32_10([idx & 0xFFFFFFFF, idx >> 32, step, 2], [seed & 0xFFFFFFFF, seed >> 32])
        assert np.allclose(xi, [((w >> 8) + 0.5) / 2 ** 24 for w in r], rtol=0, atol=0)
        z = orc.noise_normal3(seed, idx, step, 2)
        r0, r2 = math.sqrt(-2 * math.log(xi[0])), math.sqrt(-2 * math.log(xi[2]))
        assert z == pytest.approx([r0 * math.cos(2 * math.pi * xi[1]), r0 * math.sin(2 * math.pi * xi[1]),
                                   r2 * math.cos(2 * math.pi * xi[3])], abs=1e-14)
    z = np.array([orc.noise_normal3(seed, m, 3, 2) for m in range(20000)])
    assert np.abs(z.mean(0)).max() < 0.03 and np.abs(z.std(0) - 1).max() < 0.03
    assert np.abs(np.corrcoef(z.T) - np.eye(3)).max() < 0.03
    assert abs((z ** 4).mean() - 3.0) < 0.15                               # Gaussian kurtosis
    # different step / tag / seed -> different stream
    assert not np.allclose(orc.noise_normal3(seed, 5, 3, 2), orc.noise_normal3(seed, 5, 4, 2))
    assert not np.allclose(orc.noise_uniform(seed, 5, 0, 1), orc.noise_uniform(seed, 5, 0, 2))
    assert not np.allclose(orc.noise_uniform(seed, 5, 0, 1), orc.noise_uniform(seed + 2 ** 32, 5, 0, 1))


# ------------------------------------------------------------------ springs (Eq. 2-3)
def _icosa_oracle(seed=0, k=0.37, perturb=0.2):
    v, _, e = wl.icosphere(0)
    rng = np.random.default_rng(seed)
    rest = wl.edge_lengths(v, e)
    x = 3.0 * v + perturb * rng.standard_normal(v.shape) + np.array([10.0, 9.0, 8.0])
    o = orc.Oracle(20, 20, 20, 0.8)
    o.add_mesh(x, e, 3.0 * rest, k)
    return o, x, e, 3.0 * rest, k


def test_P14_spring_force_is_minus_energy_gradient():
    o, x, e, rest, k = _icosa_oracle()
    o.compute_membrane_forces()
    F = o.read_forces()
    # energy written independently from Eq. 2
    H = lambda xx: 0.5 * k * ((wl.edge_lengths(xx, e) - rest) ** 2).sum()
    assert o.spring_energy() == pytest.approx(H(x), rel=1e-14)
    d = 1e-6
    for m in range(x.shape[0]):
        for a in range(3):
            xp = x.copy(); xp[m, a] += d
            xm = x.copy(); xm[m, a] -= d
            assert F[m, a] == pytest.approx(-(H(xp) - H(xm)) / (2 * d), rel=1e-6, abs=1e-9)
    assert np.abs(F.sum(0)).max() < 1e-15                                  # Newton's third law
    assert np.abs(np.cross(x, F).sum(0)).max() < 1e-13                     # central forces: no torque
    assert np.abs(F).max() > 1e-2


def test_P14_rest_shape_and_two_node_spring():
    v, _, e = wl.icosphere(1)
    o = orc.Oracle(8, 8, 8, 0.8)
    o.add_mesh(2 * v + 4, e, None, 0.5)                  # rest = NULL: lengths of the given shape
    o.compute_membrane_forces()
    assert np.abs(o.read_forces()).max() < 1e-15
    for dist, L in ((1.5, 1.0), (0.6, 1.0)):
        o = orc.Oracle(8, 8, 8, 0.8)
        k = 0.25
        o.add_mesh(np.array([[2.0, 3.0, 4.0], [2.0 + dist, 3.0, 4.0]]), np.array([[0, 1]]), np.array([L]), k)
        o.compute_membrane_forces()
        F = o.read_forces()
        # stretched (dist > L): node 0 is pulled towards node 1 (+x); compressed: pushed away
        assert F[0] == pytest.approx([k * (dist - L), 0, 0], abs=1e-16)
        assert F[1] == pytest.approx([-k * (dist - L), 0, 0], abs=1e-16)


def test_force_noise_definition():
    """O-5: F_m,d += sigma z_d with Philox normals keyed on (global node, step, tag 2)."""
    v, _, e = wl.icosphere(0)
    o = orc.Oracle(8, 8, 8, 0.8)
    o.add_mesh(v + 4, e, None, 0.1)
    o.add_mesh(v + 3, e, None, 0.1)                      # second mesh: global node index continues
    seed, sigma, step = 99, 1e-4, 17
    o.compute_membrane_forces(sigma, seed, step)
    F = o.read_forces()
    for m in (0, 11, 12, 23):
        assert F[m] == pytest.approx(sigma * orc.noise_normal3(seed, m, step, 2), abs=1e-18)


# ------------------------------------------------------------------ spread / interpolate (Eq. 33-34)
def _brute_weights(X, n, kind):
    """W[m, cell] by looping over ALL cells with minimum-image distances (periodic axes) or plain
    distances (wall axes) -- no floor(), no stencil indexing."""
    nx, ny, nz = n
    out = np.zeros((X.shape[0], nx * ny * nz))
    for m, xm in enumerate(X):
        w1 = []
        for a, na in enumerate(n):
            d = np.arange(na) - xm[a]
            if kind[a] == 0:
                d = d - na * np.round(d / na)
            w1.append(np.where(np.abs(d) < 2, 0.25 * (1 + np.cos(np.pi * d / 2)), 0.0))
        out[m] = (w1[2][:, None, None] * w1[1][None, :, None] * w1[0][None, None, :]).ravel()
    return out


@pytest.mark.parametrize("kind", [(0, 0, 0), (0, 1, 0)])
def test_P12_brute_force_spread_and_interpolate(kind):
    n = (8, 8, 8)
    rng = np.random.default_rng(21)
    X = rng.random((5, 3)) * 8
    X[0] = (0.2, 3.3, 7.9)            # straddles the periodic seam
    X[1] = (4.0, 5.0, 2.0)            # exactly on integers (G16)
    X[2] = (7.99, 4.5, 0.01)
    if kind[1] == 1:
        X[3, 1] = 0.3                 # stencil crosses the low wall: cells dropped (G15)
        X[4, 1] = 7.2                 # and the high wall
    F = rng.standard_normal((5, 3))
    o = orc.Oracle(*n, 0.8, kind)
    o.add_mesh(X, np.zeros((0, 2), dtype=np.int32), None, 0.0)
    o.write_forces(F)
    g = o.spread()
    W = _brute_weights(X, n, kind)
    assert np.allclose(g, np.einsum("mq,md->dq", W, F), rtol=0, atol=1e-15)
    w = rng.standard_normal((3, 512))
    assert np.allclose(o.interpolate_field(w), np.einsum("mq,dq->md", W, w), rtol=0, atol=1e-14)


def test_P10_P11_total_force_and_adjointness():
    w3 = wl.config1()
    o = orc.Oracle.from_workload(w3)
    o.compute_membrane_forces()
    F = o.read_forces()
    g = o.spread()
    assert np.allclose(g.sum(1), F.sum(0), rtol=0, atol=1e-16)             # P10 (full support)
    assert np.abs(g.sum(1) - 0).max() < 1e-15                              # springs: zero net force
    assert (np.abs(g).sum(0) > 0).sum() > 500
    rng = np.random.default_rng(3)
    w = rng.standard_normal((3, o.cells))
    U = o.interpolate_field(w)
    assert (g * w).sum() == pytest.approx((F * U).sum(), rel=1e-12)        # P11
    # adjointness also with dropped wall cells
    X = o.read_nodes(); X[:, 1] -= X[:, 1].min() - 0.2
    o.write_nodes(X); o.write_forces(F + 0.01)
    g = o.spread(); U = o.interpolate_field(w)
    assert abs(g.sum(1)[0] - (F + 0.01).sum(0)[0]) > 1e-4                  # force IS lost at the wall
    assert (g * w).sum() == pytest.approx(((F + 0.01) * U).sum(), rel=1e-12)


def test_P13_rigid_translation_in_uniform_flow_across_seam():
    nx, ny, nz = 12, 10, 9
    v, _, e = wl.icosphere(1)
    x0 = 2.5 * v + np.array([nx - 3.0, 5.0, 4.5])       # will cross x = nx
    o = orc.Oracle(nx, ny, nz, 0.8)
    u0 = np.array([0.09, -0.02, 0.035])
    o.set_equilibrium(None, np.tile(u0[:, None], (1, o.cells)))
    o.add_mesh(x0 * (1 + 0.0), e, 0.9 * wl.edge_lengths(x0, e), 0.3)   # pre-stressed: non-zero forces
    o.compute_membrane_forces()
    F0 = o.read_forces()
    assert np.abs(F0).max() > 1e-2
    for n in range(1, 61):
        o.step(None)                                     # uniform state: fixed point (P6)
        o.interpolate_advance()
        assert np.allclose(o.read_nodes(), x0 + n * u0, rtol=0, atol=1e-12)
        assert np.allclose(o.read_node_velocities(), u0, rtol=0, atol=1e-15)
    assert o.read_nodes()[:, 0].max() > nx + 2           # unwrapped storage (G17)
    o.compute_membrane_forces()
    assert np.allclose(o.read_forces(), F0, rtol=0, atol=1e-13)


def test_P15_ib_leaves_fluid_momentum_unchanged_in_periodic_box():
    c, _ = orc.lattice()
    nx = ny = nz = 16
    v, _, e = wl.icosphere(1)
    x0 = 3.0 * v * np.array([1, 1, 0.4]) + 8.0
    o = orc.Oracle(nx, ny, nz, 0.8)
    rho, u = wl.random_fields(5, o.cells, rho_amp=0.0, u_amp=0.01)
    o.set_equilibrium(rho, u)
    o.add_mesh(x0, e, 0.8 * wl.edge_lengths(x0, e), 0.05)
    j0 = np.einsum("id,iq->d", c.astype(float), o.read_populations())
    for s in range(25):
        o.coupled_step()
    j1 = np.einsum("id,iq->d", c.astype(float), o.read_populations())
    assert np.allclose(j1, j0, rtol=0, atol=2e-12)       # sum over 78k populations: round-off only
    assert np.abs(o.read_nodes() - x0).max() > 1e-2      # the mesh did move


def test_interpolated_velocity_is_post_step_with_half_force():
    """G11 reading A: U = interp of v^{n+1} = (sum c f^{n+1} + g^n/2)/rho^{n+1}."""
    c, _ = orc.lattice()
    o = orc.Oracle(10, 10, 10, 0.7)
    rho, u = wl.random_fields(9, o.cells, rho_amp=0.01, u_amp=0.02)
    o.set_equilibrium(rho, u)
    X = np.array([[4.3, 5.1, 4.9], [5.2, 4.4, 5.6]])
    o.add_mesh(X, np.array([[0, 1]]), np.array([0.5]), 0.2)
    o.compute_membrane_forces()
    g = o.spread()
    o.step(g)
    f1 = o.read_populations()
    v1 = (np.einsum("id,iq->dq", c.astype(float), f1) + g / 2) / f1.sum(0)
    rho1, vm = o.read_macros()
    assert np.allclose(vm, v1, rtol=0, atol=1e-16)
    U = o.interpolate_field(v1)
    o.interpolate_advance()
    assert np.allclose(o.read_node_velocities(), U, rtol=0, atol=1e-16)
    assert np.allclose(o.read_nodes(), X + U, rtol=0, atol=1e-15)


def test_node_leaving_channel_is_reported():
    kind, u_lo, u_hi = wl._walls_y(0.0)
    o = orc.Oracle(6, 6, 6, 0.8, kind, u_lo, u_hi)
    o.set_equilibrium(None, np.tile(np.array([0.0, -0.3, 0.0])[:, None], (1, o.cells)))
    o.add_mesh(np.array([[3.0, -0.4, 3.0]]), np.zeros((0, 2), dtype=np.int32), None, 0.0)
    with pytest.raises(orc.OracleError) as ei:
        o.interpolate_advance()
    assert ei.value.code == -5


def test_spread_requires_forces():
    o = orc.Oracle(6, 6, 6, 0.8)
    o.add_mesh(np.array([[3.0, 3.0, 3.0]]), np.zeros((0, 2), dtype=np.int32), None, 0.0)
    with pytest.raises(orc.OracleError) as ei:
        o.spread()
    assert ei.value.code == -4


# ------------------------------------------------------------------ C1 magnitudes (P16)
def test_P16_config1_expected_magnitudes():
    w = wl.config1()
    assert w.mesh_xyz.shape == (1, 162, 3) and w.edges.shape == (480, 2)
    o = orc.Oracle.from_workload(w)
    o.compute_membrane_forces()
    assert 5e-4 < np.abs(o.read_forces()).max() < 1e-2
    c0 = o.read_nodes().mean(0)
    m0 = o.read_populations().sum()
    for s in range(w.steps):
        o.coupled_step()
    X = o.read_nodes()
    drift = X.mean(0) - c0
    assert drift[0] == pytest.approx(200 * 0.05 * 16.5 / 32, rel=2e-2)     # advected with the shear at y = 16
    assert abs(drift[1]) < 5e-3 and abs(drift[2]) < 5e-3
    assert np.isfinite(X).all()
    rho, v = o.read_macros()
    assert np.abs(rho - 1).max() < 5e-3
    assert o.read_populations().sum() == pytest.approx(m0, rel=1e-13)
