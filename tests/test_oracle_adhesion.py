"""Pins for the oracle's NEXT-4 functions: the stochastic dynamic adhesion model (PAPER.md section
3.2, Eq. 12-14, rules L147-149, P_f / P_r L151) and the short-range wall repulsion (L244-246).

The paper prints no worked example for this submodel and Table 2 lacks sigma, gamma and l_b, so the
pins are what the printed formulas and rules fix by themselves:
  * P_f = 1 - exp(-k_on dt), P_r = 1 - exp(-k_off dt) (L151): with force-independent rates the number
    of surviving bonds decays as exp(-k_off t) -- the log-survival slope is -k_off, which is how the
    paper itself reads k_off off its simulations (Fig. 7) -- and the fraction of in-range
    receptors that bind in one step is P_f;
  * Bell's law (Eq. 12): stretching the bond so that gamma sigma d / k_BT = ln 2 doubles the slope;
  * Eq. 13 as printed: the exponent sigma d (gamma - d/2)/k_BT vanishes at d = 0 and d = 2 gamma and
    peaks at d = gamma with value sigma gamma^2 / 2 k_BT;
  * the two rules (one vWF per receptor, at most 4 receptors per vWF) under any contention;
  * capture distance: no bond forms at or beyond l_max (L149);
  * Eq. 14: the bond force is minus the gradient of sigma/2 (x_b - l_b)^2, zero at x_b = l_b;
  * F_rep (L246) = -d/d eps of -F0 ln(1 - exp(-tau eps)); -> F0/eps as eps -> 0, -> F0 tau exp(-tau eps)
    far away."""
import math

import numpy as np
import pytest

from oracle import orc

PRM = dict(wall_axis=1, max_per_site=4, k_on0=0.05, k_off0=0.02, s=3.0, gamma=0.2, sigma=0.05, l_b=0.3, l_max=0.64,
           F0=0.0, tau_rep=0.0)


def cloud(n_nodes, xyz, nx=16, ny=8, nz=16, kind=(0, 1, 0)):
    """an oracle context with one edgeless 'mesh' of free nodes at xyz"""
    o = orc.Oracle(nx, ny, nz, 0.8, kind)
    o.set_equilibrium()
    xyz = np.asarray(xyz, dtype=np.float64).reshape(n_nodes, 3)
    o.add_mesh(xyz, np.zeros((0, 2), dtype=np.int32), None, 0.0)
    return o


def test_probabilities_follow_the_printed_forms():
    p = dict(PRM)
    # Eq. 13 exponent: zero at d = 0 and d = 2 gamma, maximal at d = gamma
    pf0, pr0 = orc.adhesion_probabilities(p, p["l_b"])
    assert pf0 == pytest.approx(1 - math.exp(-p["k_on0"]), rel=1e-14)
    assert pr0 == pytest.approx(1 - math.exp(-p["k_off0"]), rel=1e-14)
    for sign in (+1, -1):                                        # |x_b - l_b|: stretch and compression alike
        pf2, _ = orc.adhesion_probabilities(p, p["l_b"] + sign * 2 * p["gamma"])
        assert pf2 == pytest.approx(pf0, rel=1e-13)
        pfm, prm = orc.adhesion_probabilities(p, p["l_b"] + sign * p["gamma"])
        k_on_max = -math.log1p(-pfm)
        assert k_on_max / p["k_on0"] == pytest.approx(math.exp(p["s"] * p["gamma"] ** 2 / 2), rel=1e-12)
        ds = np.linspace(0.0, 0.5, 101)
        k_on = np.array([-math.log1p(-orc.adhesion_probabilities(p, p["l_b"] + sign * d)[0]) for d in ds])
        assert abs(ds[int(np.argmax(k_on))] - p["gamma"]) <= 0.005
    # Bell (Eq. 12): gamma * F_b / k_BT = ln 2 doubles k_off; F_b = sigma d
    d2 = math.log(2.0) / (p["gamma"] * p["s"])
    _, pr2 = orc.adhesion_probabilities(p, p["l_b"] + d2)
    assert -math.log1p(-pr2) == pytest.approx(2 * p["k_off0"], rel=1e-12)


def bound_cloud(n, height, prm):
    """n receptors, one per node, every node directly above its own vWF site at the given height
    above the wall plane, all bonds formed"""
    side = int(math.ceil(math.sqrt(n)))
    ii, kk = np.meshgrid(np.arange(side), np.arange(side), indexing="ij")
    xyz = np.stack([ii.ravel()[:n], np.full(n, -0.5 + height), kk.ravel()[:n]], axis=1).astype(np.float64)
    o = cloud(n, xyz, nx=side, nz=side)
    o.set_receptors(np.arange(n), prm)
    b = np.stack([np.ones(n, dtype=np.int32), ii.ravel()[:n], kk.ravel()[:n]], axis=1)
    o.write_bonds(b)
    return o


@pytest.mark.parametrize("stretch,factor", [(0.0, 1.0), (math.log(2.0) / (0.2 * 3.0), 2.0)])
def test_log_survival_slope_is_minus_k_off(stretch, factor):
    """Fig. 7's reading of k_off: ln(number of surviving bonds) against time has slope -k_off; with
    the bond held at x_b = l_b the rate is k_off0, stretched by ln2/(gamma s) it is twice that"""
    p = dict(PRM, k_on0=0.0)                                    # no re-formation
    n = 40000
    o = bound_cloud(n, p["l_b"] + stretch, p)
    alive = [n]
    for step in range(40):
        o.adhesion_update(seed=77, step=step)
        alive.append(int(o.read_bonds()[:, 0].sum()))
    o.close()
    t = np.arange(41)
    slope = np.polyfit(t, np.log(alive), 1)[0]
    k = factor * p["k_off0"]
    # binomial noise of the fit: ~ sqrt(k t)/sqrt(n)/t ~ 1e-4 -> 3 % is > 5 sigma
    assert slope == pytest.approx(-k, rel=0.03), (slope, -k)
    assert alive[-1] == pytest.approx(n * math.exp(-k * 40), rel=0.02)


def test_formation_fraction_is_P_f_and_respects_capture_distance():
    p = dict(PRM, k_off0=0.0)
    n = 40000
    side = 200
    ii, kk = np.meshgrid(np.arange(side), np.arange(side), indexing="ij")
    xyz = np.stack([ii.ravel(), np.full(n, -0.5 + 0.4), kk.ravel()], axis=1).astype(np.float64)
    xyz[n // 2:, 1] = -0.5 + 0.64                                # second half exactly AT the capture distance
    o = cloud(n, xyz, nx=side, nz=side)
    o.set_receptors(np.arange(n), p)
    o.adhesion_update(seed=5, step=0)
    b = o.read_bonds()
    o.close()
    pf, _ = orc.adhesion_probabilities(p, 0.4)
    got = b[: n // 2, 0].mean()
    assert abs(got - pf) <= 5 * math.sqrt(pf * (1 - pf) / (n // 2)), (got, pf)
    assert b[n // 2:, 0].sum() == 0                               # "separated less than" 128 nm (L149)
    on = b[:, 0] == 1
    assert (b[on, 1] == ii.ravel()[on]).all() and (b[on, 2] == kk.ravel()[on]).all()


def test_rules_one_bond_per_receptor_and_four_receptors_per_site():
    """30 receptors on ONE node sitting over one vWF site, P_f = 1: exactly 4 bind (rule 2), the
    lowest indices; a second update changes nothing (rule 1: bound receptors are not re-tested for
    formation, the site is full); freeing two places lets exactly the next two in"""
    p = dict(PRM, k_on0=1e9, k_off0=0.0)
    o = cloud(2, [[3.2, -0.1, 5.3], [9.0, 4.0, 9.0]])           # node 1 is far from the wall
    node = np.zeros(30, dtype=np.int32); node[25:] = 1
    o.set_receptors(node, p)
    o.adhesion_update(seed=1, step=0)
    b = o.read_bonds()
    assert b[:, 0].tolist() == [1] * 4 + [0] * 26
    assert (b[:4, 1] == 3).all() and (b[:4, 2] == 5).all()        # nearest site of (3.2, 5.3)
    o.adhesion_update(seed=1, step=1)
    assert (o.read_bonds() == b).all()
    b2 = b.copy(); b2[1] = 0; b2[3] = 0
    o.write_bonds(b2)
    o.adhesion_update(seed=1, step=2)
    b3 = o.read_bonds()
    assert b3[:, 0].tolist() == [1, 1, 1, 1] + [0] * 26           # receptors 1 and 3 are the lowest unbound
    o.close()


def test_nearest_site_wraps_on_periodic_axes_and_bond_keeps_its_site():
    p = dict(PRM, k_on0=1e9, k_off0=0.0)
    o = cloud(1, [[15.7, -0.2, -0.4]])                           # nx = nz = 16: nearest site (16, 0) == (0, 0) wrapped
    o.set_receptors([0], p)
    o.adhesion_update(seed=3, step=0)
    assert o.read_bonds().tolist() == [[1, 16, 0]]                # unwrapped site coordinates
    o.write_nodes([[17.9, 0.3, 1.2]])                            # the node moves on; the bond stays with its site
    o.adhesion_update(seed=3, step=1)
    assert o.read_bonds().tolist() == [[1, 16, 0]]
    o.compute_membrane_forces()
    F = o.read_forces()[0]
    R = np.array([16.0 - 17.9, -0.5 - 0.3, 0.0 - 1.2]); x_b = np.linalg.norm(R)
    assert np.allclose(F, p["sigma"] * (x_b - p["l_b"]) * R / x_b, rtol=1e-12)     # pulls back towards the site
    o.close()


def test_bond_and_repulsion_forces_are_minus_the_gradient_of_their_potential():
    rng = np.random.default_rng(11)
    p = dict(PRM, F0=3e-4, tau_rep=5.0)
    n = 12
    xyz = np.stack([4 + 6 * rng.random(n), -0.5 + 0.1 + 0.6 * rng.random(n), 4 + 6 * rng.random(n)], axis=1)
    o = cloud(n, xyz)
    rec = rng.integers(0, n, size=40)
    o.set_receptors(rec, p)
    b = np.zeros((40, 3), dtype=np.int32)
    b[:, 0] = rng.random(40) < 0.7
    b[:, 1] = np.round(xyz[rec, 0]) + rng.integers(-1, 2, size=40)
    b[:, 2] = np.round(xyz[rec, 2]) + rng.integers(-1, 2, size=40)
    o.write_bonds(b)
    o.compute_membrane_forces()
    F = o.read_forces()
    num = np.zeros_like(F)
    h = 1e-6
    for m in range(n):
        for d in range(3):
            xp = xyz.copy(); xp[m, d] += h; o.write_nodes(xp); ep = o.adhesion_energy()
            xm = xyz.copy(); xm[m, d] -= h; o.write_nodes(xm); em = o.adhesion_energy()
            num[m, d] = -(ep - em) / (2 * h)
    o.close()
    assert np.abs(F - num).max() <= 1e-8 * np.abs(F).max() + 1e-12
    assert (F[:, 1] != 0).all()


def test_repulsion_limits_and_zero_bond_force_at_rest_length():
    p = dict(PRM, F0=2e-4, tau_rep=4.0, k_on0=0.0)
    eps = np.array([1e-5, 1e-3, 0.3, 3.0, 8.0])
    xyz = np.stack([np.arange(5) + 2.0, -0.5 + eps, np.full(5, 3.0)], axis=1)
    o = cloud(5, xyz)
    o.set_receptors([2], p)
    o.write_bonds([[1, 4, 3]])                                   # node 2 at (4, -0.2, 3): x_b = 0.3 = l_b
    o.compute_membrane_forces()
    F = o.read_forces()
    o.close()
    assert np.allclose(F[:, [0, 2]], 0.0, atol=1e-18)              # repulsion is along the normal; bond at rest length
    assert F[0, 1] == pytest.approx(p["F0"] / eps[0], rel=1e-4)   # tau e^-x/(1 - e^-x) -> 1/eps
    assert F[1, 1] == pytest.approx(p["F0"] / eps[1], rel=3e-3)
    assert F[3, 1] == pytest.approx(p["F0"] * p["tau_rep"] * math.exp(-p["tau_rep"] * eps[3]), rel=1e-5)
    assert 0 < F[4, 1] < 1e-16
    assert (np.diff(F[:, 1]) < 0).all()                           # monotonically decaying
    # on-site (Hecht-Harting) walls lie ON layer 0: the same node is 0.5 closer to that wall
    o2 = cloud(1, [[4.0, 0.3, 3.0]], kind=(0, 2, 0))
    o2.set_receptors([0], p)
    o2.compute_membrane_forces()
    e = math.exp(-p["tau_rep"] * 0.3)
    assert o2.read_forces()[0, 1] == pytest.approx(p["F0"] * p["tau_rep"] * e / (1 - e), rel=1e-12)
    o2.close()


def test_coupled_platelet_adheres_and_bonds_slow_it_down():
    """end-to-end sanity on the NEXT-4 workload (tiny): bonds form under the platelet, every site obeys
    rule 2, and the tethered platelet is carried less far by the shear flow than a free one"""
    from paper_1312_2234_b200 import workloads as wl
    kw = dict(nx=24, ny=16, nz=24, a=4.0, subdiv=2, receptors_per_platelet=600, steps=150)
    w = wl.adhering_platelets(**kw)
    free = wl.adhering_platelets(adhesion=dict(k_on0=0.0), **kw)
    out = []
    for ww in (w, free):
        o = orc.Oracle.from_workload(ww)
        for s in range(ww.steps):
            o.coupled_step(0.0, 0, s)
        b = o.read_bonds()
        X = o.read_nodes()
        out.append((int(b[:, 0].sum()), X.mean(axis=0), X[:, 1].min()))
        if b[:, 0].any():
            on = b[b[:, 0] == 1]
            _, counts = np.unique(on[:, 1] * 4096 + on[:, 2], return_counts=True)
            assert counts.max() <= 4
        o.close()
    (nb, c_b, ymin_b), (nf, c_f, ymin_f) = out
    assert nb > 20 and nf == 0
    assert ymin_b > -0.5 and ymin_f > -0.5                         # repulsion keeps the membrane off the wall
    drift_b, drift_f = c_b[0] - w.mesh_xyz[0].mean(axis=0)[0], c_f[0] - free.mesh_xyz[0].mean(axis=0)[0]
    assert 0 <= drift_b < 0.8 * drift_f, (drift_b, drift_f)


def test_wall_axis_relabelling_gives_the_same_bonds():
    """the same receptor cloud over a wall on axis y, and with y and z exchanged over a wall on axis
    z: identical bond table (tangential axes in x, y, z order: (x, z) becomes (x, y)) and forces
    with the two components exchanged"""
    rng = np.random.default_rng(5)
    p = dict(PRM, F0=1e-4, tau_rep=3.0, k_on0=0.4)
    n = 400
    xyz = np.stack([12 * rng.random(n), -0.5 + 0.05 + 0.7 * rng.random(n), 10 * rng.random(n)], axis=1)
    rec = rng.integers(0, n, size=1500)
    tables, forces = [], []
    for axis in (1, 2):
        pts = xyz if axis == 1 else xyz[:, [0, 2, 1]]
        dims = dict(nx=12, ny=8, nz=10) if axis == 1 else dict(nx=12, ny=10, nz=8)
        kind = (0, 1, 0) if axis == 1 else (0, 0, 1)
        o = cloud(n, pts, kind=kind, **dims)
        o.set_receptors(rec, dict(p, wall_axis=axis))
        for step in range(6):
            o.adhesion_update(seed=9, step=step)
        o.compute_membrane_forces()
        tables.append(o.read_bonds()); forces.append(o.read_forces())
        o.close()
    assert tables[0][:, 0].sum() > 100
    assert (tables[0] == tables[1]).all()
    assert np.allclose(forces[0], forces[1][:, [0, 2, 1]], rtol=1e-13, atol=1e-18)
