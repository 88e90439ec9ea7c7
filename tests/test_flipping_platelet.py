"""the paper's own validation case (section 4.1, Fig. 5-6) -- one
stiff platelet flipping in a linear shear flow, compared with the Jeffery orbit of a spheroid.

What the paper fixes: the shape (oblate spheroid, aspect ratio lambda = 0.25, L81), tau = 1.379
(L215), the two cases H/a = 2.4 and H/a > 20, and the statement that the far-wall orbit is the
Jeffery orbit.  The curve of Fig. 6 exists only as an image and the 2.65 % figure refers to it, so
the pin is the Jeffery solution itself (Jeffery 1922, the theory the paper cites through Mody & King):
for a spheroid of axis ratio r (symmetry axis : diameter) whose axis lies in the shear plane, with
phi the angle from the velocity-gradient direction towards the flow direction,

    tan(phi) = r tan(G t / (r + 1/r)),   dphi/dt = G (r^2 cos^2 phi + sin^2 phi) / (r^2 + 1),

period T = 2 pi (r + 1/r) / G, G the shear rate.  An immersed-boundary surface is hydrodynamically
about one lattice spacing thicker than its mesh (the width of the delta kernel), so a disc of
half-thickness 1.25 cells behaves as a spheroid with r_eff > lambda: the tests pin (a) periodic
flipping in the direction of the flow vorticity, (b) the fast-phase angular velocity, which Jeffery
fixes at G/(1 + r^2) -- between 0.86 G and 0.94 G for every r in [0.25, 0.4] -- and (c), on the GPU,
a whole orbit: the measured half period gives r_eff, and the whole phi(t) curve must then be the
Jeffery curve of that single parameter.

The CPU test runs the oracle on a reduced box (it is the oracle's pin for this workload); the GPU
tests run the full-size far-wall and near-wall cases through the C-ABI and a lock-step parity check
against the oracle on the first steps."""
import math

import numpy as np
import pytest

from oracle import orc
from paper_1312_2234_b200 import workloads as wl


def axis_angle(xyz, prev=None):
    """phi of the disc axis from +y towards +x, unwrapped against the previous sample (the axis is
    a director: n and -n are the same orientation, so phi is continued modulo pi)"""
    n = wl.disc_axis(xyz)
    phi = math.atan2(n[0], n[1])
    if prev is not None:
        phi += math.pi * round((prev - phi) / math.pi)
    return phi, abs(n[2])


def jeffery_phi(t, r, G):
    """Jeffery's orbit tan(phi) = r tan(a), a = G t/(r + 1/r), continuous in t: phi - a stays within
    (-pi/2, pi/2) and tan(phi - a) = (r - 1) sin a cos a / (cos^2 a + r sin^2 a)"""
    a = G / (r + 1.0 / r) * np.asarray(t, dtype=np.float64)
    s, c = np.sin(a), np.cos(a)
    return a + np.arctan((r - 1.0) * s * c / (c * c + r * s * s))


def crossing_times(ts, phis, level):
    """times at which the (increasing) phi(t) samples cross level + n pi, by linear interpolation"""
    out = []
    ts = np.asarray(ts, dtype=np.float64); phis = np.asarray(phis, dtype=np.float64)
    n0 = math.ceil((phis[0] - level) / math.pi)
    n1 = math.floor((phis[-1] - level) / math.pi)
    for n in range(n0, n1 + 1):
        target = level + n * math.pi
        i = int(np.argmax(phis >= target))
        if i == 0:
            continue
        f = (target - phis[i - 1]) / (phis[i] - phis[i - 1])
        out.append(ts[i - 1] + f * (ts[i] - ts[i - 1]))
    return out


def test_workload_geometry():
    w = wl.flipping_platelet(nx=32, ny=48, nz=32, a=4.0, subdiv=2, theta0=0.3)
    X = w.mesh_xyz[0]
    n = wl.disc_axis(X)
    n = n * np.sign(n[1])
    assert np.allclose(n, [math.sin(0.3), math.cos(0.3), 0.0], atol=1e-12)
    assert np.allclose(X.mean(axis=0), [16.0, 23.5, 16.0], atol=1e-9)
    assert w.shear_rate == pytest.approx(2 * 0.1 / 48)
    # the initial flow is the Couette profile between walls at -1/2 and ny - 1/2 moving at -+u_wall
    u = w.u0.reshape(3, 32, 48, 32)
    assert u[0, 0, 0, 0] == pytest.approx(-0.1 + 0.5 * w.shear_rate) and u[0, 0, 47, 0] == pytest.approx(0.1 - 0.5 * w.shear_rate)
    d = X - X.mean(axis=0)
    semi = np.sqrt(3.0 * np.linalg.eigvalsh(d.T @ d / len(X)))
    assert semi[0] / semi[2] == pytest.approx(0.25, rel=0.03)
    nw = wl.flipping_platelet(nx=32, ny=48, nz=32, a=5.0, height=12.0)
    assert nw.mesh_xyz[0].mean(axis=0)[1] == pytest.approx(11.5) and nw.shear_rate == pytest.approx(0.1 / 48)
    assert nw.u_lo[1, 0] == 0.0 and nw.u_hi[1, 0] == 0.1


def test_jeffery_formula_is_self_consistent():
    """the closed form above satisfies Jeffery's rate equation and has the stated period"""
    r, G = 0.3, 2e-3
    T = 2 * math.pi * (r + 1 / r) / G
    t = np.linspace(0.0, 1.5 * T, 30001)
    phi = jeffery_phi(t, r, G)
    rate = np.gradient(phi, t)
    want = G * (r * r * np.cos(phi) ** 2 + np.sin(phi) ** 2) / (r * r + 1)
    assert np.abs(rate - want)[5:-5].max() <= 2e-3 * G
    assert phi[20000] - phi[0] == pytest.approx(2 * math.pi, abs=1e-9)     # t = T: one full turn
    assert rate.max() == pytest.approx(G / (1 + r * r), rel=1e-4)


def test_oracle_platelet_flips_at_the_jeffery_fast_rate():
    """oracle pin for NEXT-3 on a reduced box (32 x 48 x 32, a = 4, 162 nodes, ~20 s of CPU): after
    the start-up the axis turns monotonically in the sense of the flow vorticity, stays in the shear
    plane, and passes the broadside orientation (phi = pi/2) at G/(1 + r^2) with r in [0.25, 0.45]"""
    w = wl.flipping_platelet(nx=32, ny=48, nz=32, a=4.0, subdiv=2, k_spring=0.1)
    G = w.shear_rate
    o = orc.Oracle.from_workload(w)
    ts, phis, prev = [], [], None
    for s in range(1750):
        o.coupled_step(0.0, 0, s)
        if (s + 1) % 50 == 0:
            phi, out_of_plane = axis_angle(o.read_nodes(), prev)
            assert out_of_plane < 1e-6           # symmetric set-up: the axis never leaves the x-y plane
            ts.append(s + 1); phis.append(phi); prev = phi
    X = o.read_nodes()
    o.close()
    ts = np.asarray(ts, dtype=np.float64); phis = np.asarray(phis) - round(phis[0] / math.pi) * math.pi
    later = ts >= 600
    assert (np.diff(phis[later]) > 0).all()                                # turns with the vorticity
    assert phis[-1] > 0.5 * math.pi + 0.3                                   # went through broadside
    rate = np.diff(phis) / np.diff(ts)
    assert 0.83 <= rate.max() / G <= 0.95, rate.max() / G                   # G/(1 + r^2), r in [0.25, 0.45]
    assert np.abs(X.mean(axis=0) - [16.0, 23.5, 16.0]).max() < 1e-6          # centre on the zero-velocity plane


# ------------------------------------------------------------------------------------------ GPU
def run_gpu_orbit(w, steps, every):
    from paper_1312_2234_b200 import binding as plb
    sim = plb.Simulation.from_workload(w)
    ts, phis, centres, semis, prev = [0], [], [], [], None
    phi, _ = axis_angle(w.mesh_xyz[0]); phis.append(phi); prev = phi
    centres.append(w.mesh_xyz[0].mean(axis=0))
    for s in range(steps):
        sim.coupled_step(0.0, 0, s)
        if (s + 1) % every == 0:
            X = sim.read_nodes()
            phi, out_of_plane = axis_angle(X, prev)
            assert out_of_plane < 1e-3
            d = X - X.mean(axis=0)
            ts.append(s + 1); phis.append(phi); prev = phi
            centres.append(X.mean(axis=0)); semis.append(np.sqrt(3.0 * np.linalg.eigvalsh(d.T @ d / len(X))))
    sim.status()
    sim.close()
    return np.asarray(ts, dtype=np.float64), np.asarray(phis), np.asarray(centres), np.asarray(semis)


@pytest.mark.gpu
def test_gpu_far_wall_orbit_is_a_jeffery_orbit():
    """H/a = 20 (64 x 200 x 64, a = 5, 642 nodes): 1.25 Jeffery periods of lambda = 0.25 on the GPU"""
    w = wl.flipping_platelet()
    assert (w.nx, w.ny, w.nz, w.n_nodes, w.tau) == (64, 200, 64, 642, 1.379)
    G = w.shear_rate
    T025 = 2 * math.pi * (0.25 + 4.0) / G
    ts, phis, centres, semis = run_gpu_orbit(w, int(1.25 * T025), 100)
    cross = crossing_times(ts, phis, 0.5 * math.pi)
    assert len(cross) >= 2, cross                                            # flipped at least twice
    half = cross[1] - cross[0]
    ratio = half / (0.5 * T025)
    # period -> effective axis ratio: r + 1/r = G * (2 half) / (2 pi), the root below 1
    s = G * half / math.pi
    r_eff = 0.5 * (s - math.sqrt(s * s - 4.0))
    # Jeffery curve of r_eff through the first crossing: jeffery_phi is pi/2 a quarter period after 0
    sel = (ts >= cross[0]) & (ts <= cross[1])
    fit = jeffery_phi(ts - cross[0] + 0.5 * half, r_eff, G)
    fit += math.pi * round(float(np.mean(phis[sel] - fit[sel])) / math.pi)
    rms = float(np.sqrt(np.mean((phis[sel] - fit[sel]) ** 2)))
    rate = np.diff(phis) / np.diff(ts)
    print("far wall: half period %.0f steps = %.3f of Jeffery(0.25); r_eff = %.3f; fast rate %.3f G (Jeffery %.3f); "
          "rms deviation from the Jeffery curve of r_eff %.3f rad; semi-axes %s .. %s; centre drift %.2e"
          % (half, ratio, r_eff, rate.max() / G, 1 / (1 + r_eff ** 2), rms, np.round(semis.min(axis=0), 2),
             np.round(semis.max(axis=0), 2), np.abs(centres - centres[0]).max()))
    assert 0.6 <= ratio <= 1.05, ratio
    assert 0.25 <= r_eff <= 0.45, r_eff
    assert rate.max() / G == pytest.approx(1 / (1 + r_eff ** 2), rel=0.08)
    assert rms <= 0.12, rms
    assert np.abs(centres - centres[0]).max() < 0.05                          # stays on the zero-velocity plane
    assert semis[:, 0].max() / semis[:, 2].min() < 0.32                      # stayed a stiff disc (started at 0.25)


@pytest.mark.gpu
def test_gpu_near_wall_platelet_flips_periodically():
    """H = 2.4 a above the resting wall (64 x 200 x 64, top wall moving): the 'modified Jeffery orbit'
    of L284 -- qualitative pin only (periodic flipping in the flow direction, no wall contact); the
    paper's 2.65 % refers to a curve printed only as an image (parity unpinned)"""
    w = wl.flipping_platelet(height=12.0, u_wall=0.1)
    G = w.shear_rate
    T025 = 2 * math.pi * (0.25 + 4.0) / G
    ts, phis, centres, semis = run_gpu_orbit(w, int(1.1 * T025), 200)
    cross = crossing_times(ts, phis, 0.5 * math.pi)
    assert len(cross) >= 2, cross
    half = cross[1] - cross[0]
    print("near wall: half period %.0f steps = %.3f of Jeffery(0.25); height %.2f .. %.2f; advected %.1f cells in x"
          % (half, half / (0.5 * T025), centres[:, 1].min() + 0.5, centres[:, 1].max() + 0.5, centres[-1, 0] - centres[0, 0]))
    assert 0.6 <= half / (0.5 * T025) <= 1.4
    assert centres[:, 1].min() > 6.0                                         # never touches the wall
    assert centres[-1, 0] - centres[0, 0] > 0.8 * G * 12.0 * ts[-1]          # carried along by the flow


@pytest.mark.gpu
def test_gpu_flipping_workload_matches_oracle():
    """lock-step parity on a reduced box (48 x 64 x 48, a = 5, 642 nodes, constraints on), 150 steps"""
    import parity_utils as pu
    w = wl.flipping_platelet(nx=48, ny=64, nz=48, theta0=0.4, steps=150)
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, w.steps)
    out = pu.compare(w, sim, ora)
    print("flipping workload parity", out)
    sim.close(); ora.close()
