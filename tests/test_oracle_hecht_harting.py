"""Pins for the Hecht-Harting on-site velocity wall of the CPU oracle (
PAPER.md Eq. 23-30).  Expected values come from the paper's printed equations (typed
below with the paper's own 1-based indices, for the plane the paper prints), from algebra (the
closed populations must carry exactly rho and rho*v) and from closed-form channel flows; none
comes from the oracle or from the CUDA path."""
import numpy as np
import pytest

from oracle import orc

HH = 2


def stream_only_reference(f, n, axis):
    """Plain streaming f_i(x + c_i) <- f_i(x), periodic in all axes (np.roll).  On the wall
    layers of `axis` the populations that would have come from outside are garbage here; the
    tests only use the ones that arrive from inside."""
    c, _ = orc.lattice()
    nx, ny, nz = n
    out = np.empty_like(f)
    for i in range(19):
        a = f[i].reshape(nz, ny, nx)
        out[i] = np.roll(a, shift=(c[i][2], c[i][1], c[i][0]), axis=(0, 1, 2)).reshape(-1)
    return out


def run_one_step_from_random(n, axis, tau, u_lo, u_hi, seed):
    """random positive populations -> write -> tau -> infinity is not available, so use the
    oracle's own collision but read the post-collision state back through a periodic twin:
    the twin (all periodic) shares the collision and the streaming of the interior links."""
    rng = np.random.default_rng(seed)
    cells = n[0] * n[1] * n[2]
    c, w = orc.lattice()
    f0 = w[:, None] * (1 + 0.05 * rng.standard_normal((19, cells)))
    kind = [0, 0, 0]
    kind[axis] = HH
    lo = np.zeros((3, 3)); hi = np.zeros((3, 3))
    lo[axis] = u_lo; hi[axis] = u_hi
    wall = orc.Oracle(*n, tau, kind, lo, hi)
    twin = orc.Oracle(*n, tau, (0, 0, 0))
    # the twin is given the SAME pre-collision state the wall run has after its own closure
    wall.write_populations(f0)
    f_start = wall.read_populations()
    twin.write_populations(f_start)
    wall.step()
    twin.step()
    return c, w, f_start, wall.read_populations(), twin.read_populations()


# ------------------------------------------------------------------ the paper's printed plane
def test_z0_plane_equals_the_printed_equations():
    """Eq. 23-30 exactly as printed (plane z = 0, paper's 1-based indices; 'rho/eps' read rho/6)."""
    n = (4, 3, 5)
    v = np.array([0.03, -0.02, 0.01])           # wall velocity incl. a normal component
    c, w, f_start, fw, ft = run_one_step_from_random(n, 2, 0.8, v, [0, 0, 0], seed=1)
    nx, ny, nz = n
    plane = np.arange(nx * ny)                   # cells with z = 0
    F = {i: ft[i - 1][plane] for i in range(1, 20)}      # arrived by streaming (twin), 1-based
    vx, vy, vz = v
    rho = (F[1] + F[2] + F[3] + F[4] + F[7] + F[8] + F[11] + F[12] + F[19]
           + 2 * (F[6] + F[10] + F[14] + F[16] + F[18])) / (1 - vz)
    Nx = 0.5 * (F[1] + F[7] + F[8] - (F[2] + F[11] + F[12])) - rho * vx / 3
    Ny = 0.5 * (F[3] + F[7] + F[11] - (F[4] + F[8] + F[12])) - rho * vy / 3
    expect = {
        5: F[6] + rho * vz / 3,
        9: F[14] + rho / 6 * (vz + vx) - Nx,
        13: F[10] + rho / 6 * (vz - vx) + Nx,
        15: F[18] + rho / 6 * (vz + vy) - Ny,
        17: F[16] + rho / 6 * (vz - vy) + Ny,
    }
    for i in range(1, 20):
        got = fw[i - 1][plane]
        if i in expect:
            assert np.allclose(got, expect[i], rtol=0, atol=1e-15), i
        else:                                     # "can be obtained from the streaming step"
            assert np.array_equal(got, F[i]), i
    # interior layers are untouched by the wall
    inner = np.arange(nx * ny, nx * ny * (nz - 1))
    assert np.array_equal(fw[:, inner], ft[:, inner])


# ------------------------------------------------------------------ algebra: every face
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_closed_populations_carry_rho_and_rho_v_on_both_faces(axis):
    """After the closure sum f = rho and sum c f = rho v_wall exactly, with rho from the density
    formula; the populations that arrived by streaming are unchanged.  Fixes every coefficient
    (1/3, 1/6, the sign and the 1/2 of the transverse correction) on all six faces."""
    n = [5, 4, 6]
    u_lo = np.array([0.02, -0.03, 0.015])
    u_hi = np.array([-0.01, 0.025, 0.02])
    c, w, f_start, fw, ft = run_one_step_from_random(tuple(n), axis, 0.7, u_lo, u_hi, seed=2 + axis)
    cf = c.astype(float)
    idx = np.arange(n[0] * n[1] * n[2]).reshape(n[2], n[1], n[0])
    for face, uw in ((0, u_lo), (1, u_hi)):
        sl = [slice(None)] * 3
        sl[2 - axis] = 0 if face == 0 else n[axis] - 1
        cells = idx[tuple(sl)].ravel()
        sgn = 1 if face == 0 else -1
        cn = sgn * c[:, axis]
        known = cn <= 0
        assert np.array_equal(fw[known][:, cells], ft[known][:, cells])
        S0 = ft[cn == 0][:, cells].sum(0)
        Sm = ft[cn == -1][:, cells].sum(0)
        rho = (S0 + 2 * Sm) / (1 - sgn * uw[axis])
        assert np.allclose(fw[:, cells].sum(0), rho, rtol=0, atol=2e-15)
        j = cf.T @ fw[:, cells]
        assert np.allclose(j, rho[None, :] * uw[:, None], rtol=0, atol=2e-15)
        # non-equilibrium bounce-back of the normal population: f_n - f_-n = rho v_n / 3 * sgn
        i_n = int(np.nonzero((cn == 1) & (np.abs(c).sum(1) == 1))[0][0])
        i_m = int(np.nonzero((cn == -1) & (np.abs(c).sum(1) == 1))[0][0])
        assert np.allclose(fw[i_n, cells] - fw[i_m, cells], rho * sgn * uw[axis] / 3, rtol=0, atol=2e-15)


def test_axis_relabelling_symmetry():
    """The y-wall result equals the z-wall result of the relabelled problem (x,y,z) -> (x,z,y):
    the generalisation from the printed plane to other axes is a pure renaming."""
    c, w = orc.lattice()
    nx, ny, nz = 4, 5, 3
    rng = np.random.default_rng(11)
    f0 = w[:, None] * (1 + 0.05 * rng.standard_normal((19, nx * ny * nz)))
    uy_hi = np.array([0.04, -0.01, 0.02])
    a = orc.Oracle(nx, ny, nz, 0.9, (0, HH, 0), None, np.array([[0, 0, 0], uy_hi, [0, 0, 0]]))
    a.write_populations(f0)
    for _ in range(3):
        a.step()
    fa = a.read_populations().reshape(19, nz, ny, nx)
    # relabelled: swap y <-> z of the grid, of the population index and of the wall velocity
    swap = lambda v: (v[0], v[2], v[1])
    perm = [int(np.nonzero((c == np.array(swap(ci))).all(1))[0][0]) for ci in c]
    f0s = f0.reshape(19, nz, ny, nx)[perm].transpose(0, 2, 1, 3).reshape(19, -1)
    b = orc.Oracle(nx, nz, ny, 0.9, (0, 0, HH), None, np.array([[0, 0, 0], [0, 0, 0], swap(uy_hi)]))
    b.write_populations(f0s)
    for _ in range(3):
        b.step()
    fb = b.read_populations().reshape(19, ny, nz, nx)
    assert np.allclose(fa[perm].transpose(0, 2, 1, 3), fb, rtol=0, atol=1e-15)


# ------------------------------------------------------------------ closed-form channel flows
@pytest.mark.parametrize("tau,uw", [(0.8, 0.05), (0.65, 0.08), (1.379, 0.05)])
def test_couette_with_the_wall_on_the_node(tau, uw):
    """SURVEY NEXT-1 pin: steady Couette flow between on-site walls is exactly linear with the
    walls ON layers 0 and n_y - 1: u_x(j) = u_w j/(n_y - 1), rho uniform."""
    nx, ny, nz = 2, 9, 2
    hi = np.zeros((3, 3)); hi[1] = [uw, 0, 0]
    o = orc.Oracle(nx, ny, nz, tau, (0, HH, 0), None, hi)
    o.set_equilibrium()
    for _ in range(int(4 * ny * ny / ((tau - 0.5) / 3)) + 500):
        o.step()
    rho, u = o.read_macros()
    ux = u[0].reshape(nz, ny, nx)
    assert np.abs(ux - (uw * np.arange(ny) / (ny - 1))[None, :, None]).max() <= 1e-12 * uw
    assert np.abs(u[1:]).max() <= 1e-14
    assert np.abs(rho - rho.mean()).max() <= 1e-13


@pytest.mark.parametrize("tau", [0.6, 0.8, 1.379])
def test_body_force_poiseuille_has_no_slip_at_any_tau(tau):
    """Uniform g along x between resting on-site walls: the steady profile is the exact parabola
    with zero slip at the wall nodes, v_x(j) = (g/2nu) j (n_y-1-j) + g/2 -- independent of tau
    (halfway bounce-back has the tau-dependent slip of P8 instead).  The uniform g/2 is the
    half-force term of v = u + g/2rho (L201): the wall condition fixes sum c f = rho v_wall = 0
    (paper-literal, reading G24).  Pins wall position, closure and forcing together."""
    nx, ny, nz = 2, 13, 2
    g0 = 1e-6
    g = np.zeros((3, nx * ny * nz)); g[0] = g0
    o = orc.Oracle(nx, ny, nz, tau, (0, HH, 0))
    o.set_equilibrium()
    nu = (tau - 0.5) / 3
    for _ in range(int(6 * ny * ny / nu) + 1000):
        o.step(g)
    rho, u = o.read_macros()
    ux = u[0].reshape(nz, ny, nx)
    j = np.arange(ny)
    exact = g0 / (2 * nu) * j * (ny - 1 - j) + g0 / 2
    assert np.abs(ux - exact[None, :, None]).max() <= 1e-9 * exact.max()
    assert np.abs(u[1:]).max() <= 1e-14


def test_initial_state_is_closed_and_stays_an_equilibrium_fixed_point():
    """lbm_set_equilibrium / lbm_write_populations re-close the wall layers (reading G25): a
    uniform fluid moving with both walls is a fixed point and its macros are exact from step 0."""
    nx, ny, nz = 3, 5, 4
    v = np.array([0.03, 0.0, -0.02])             # tangential to the y walls
    lo = np.zeros((3, 3)); hi = np.zeros((3, 3)); lo[1] = v; hi[1] = v
    o = orc.Oracle(nx, ny, nz, 0.75, (0, HH, 0), lo, hi)
    u0 = np.repeat(v[:, None], nx * ny * nz, axis=1)
    o.set_equilibrium(None, u0)
    f_a = o.read_populations()
    rho, u = o.read_macros()
    assert np.abs(rho - 1).max() <= 1e-15 and np.abs(u - u0).max() <= 1e-15
    for _ in range(5):
        o.step()
    assert np.abs(o.read_populations() - f_a).max() <= 1e-15


def test_rejected_configurations():
    with pytest.raises(orc.OracleError):          # edges between two closed axes are undefined
        orc.Oracle(4, 4, 4, 0.8, (0, HH, 1))
    with pytest.raises(orc.OracleError):
        orc.Oracle(4, 4, 4, 0.8, (HH, HH, 0))
    with pytest.raises(orc.OracleError):          # the two faces must be different layers
        orc.Oracle(4, 1, 4, 0.8, (0, HH, 0))
