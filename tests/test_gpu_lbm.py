"""GPU parity tests of the lattice-Boltzmann part of libplb against the fp64 CPU oracle, through
the C-ABI (binding = argument marshalling only).  Same seeded inputs on both sides; no oracle
input and no expected value comes from the CUDA path.

Tolerances (BASELINE.json north_star): max|dv| <= 1e-4 u_ref, max|drho| <= 1e-6 at the end of a
run.  Single calls are held to what fp32 arithmetic on O(1) / O(1e-2) values gives: 2e-7."""
import math
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import orc                                    # noqa: E402
from paper_1312_2234_b200 import binding as plb            # noqa: E402
from paper_1312_2234_b200 import workloads as wl           # noqa: E402
import parity_utils as pu                                  # noqa: E402

FULL = os.environ.get("PLB_FULL", "0") == "1"
DEV = "cuda:0"


def dev(a, dtype=torch.float32):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to(DEV).contiguous()


def make_pair(n, tau, kind, u_lo=None, u_hi=None):
    sim = plb.Simulation(*n, tau, kind, u_lo, u_hi)
    ora = orc.Oracle(*n, tau, kind, u_lo, u_hi)
    return sim, ora


def wall_velocities(kind, seed):
    rng = np.random.default_rng(seed)
    u_lo = 0.05 * (2 * rng.random((3, 3)) - 1)
    u_hi = 0.05 * (2 * rng.random((3, 3)) - 1)
    for a in range(3):                       # a wall moves tangentially only (mass conservation)
        u_lo[a, a] = 0.0
        u_hi[a, a] = 0.0
        if kind[a] == 0:
            u_lo[a] = 0.0
            u_hi[a] = 0.0
    return u_lo, u_hi


KINDS = [(0, 0, 0), (0, 1, 0), (1, 0, 0), (0, 0, 1), (1, 1, 0), (1, 1, 1)]
# ragged sizes: not multiples of 32 / 256, several thread blocks, tails in every axis
RAGGED = (37, 19, 23)


# ------------------------------------------------------------------ O-2 set_equilibrium
@pytest.mark.parametrize("amp", [0.0, 1e-4])
def test_set_equilibrium_matches_oracle(amp):
    n = RAGGED
    cells = n[0] * n[1] * n[2]
    rho, u = wl.random_fields(7, cells)
    sim, ora = make_pair(n, 0.8, (0, 1, 0))
    sim.set_equilibrium(dev(rho), dev(u), amp, 1234567890123)
    ora.set_equilibrium(rho, u, amp, 1234567890123)
    f_g = sim.read_populations().cpu().numpy().astype(np.float64)
    f_o = ora.read_populations()
    assert np.abs(f_g - f_o).max() <= 2e-7
    if amp > 0:      # the noise is really there and is the oracle's stream, not just small
        ora0 = orc.Oracle(*n, 0.8, (0, 1, 0))
        ora0.set_equilibrium(rho, u, 0.0, 0)
        noise_g = f_g - ora0.read_populations()
        noise_o = f_o - ora0.read_populations()
        assert np.abs(noise_o).max() > 0.9 * amp
        assert np.abs(noise_g - noise_o).max() <= 2e-7
        assert np.corrcoef(noise_g.ravel(), noise_o.ravel())[0, 1] > 0.999


def test_set_equilibrium_defaults_rho1_rest():
    sim, ora = make_pair((8, 8, 8), 0.8, (0, 0, 0))
    sim.set_equilibrium()
    ora.set_equilibrium()
    assert np.abs(sim.read_populations().cpu().numpy() - ora.read_populations()).max() <= 1e-7
    rho, u = sim.read_macros()
    assert float((rho - 1).abs().max()) <= 1e-7 and float(u.abs().max()) <= 1e-7


# ------------------------------------------------------------------ population round trip
@pytest.mark.parametrize("kind", KINDS)
def test_population_write_read_round_trip(kind):
    n = RAGGED
    cells = n[0] * n[1] * n[2]
    rng = np.random.default_rng(3)
    c, w = orc.lattice()
    f = (w[:, None] * (1 + 0.05 * (2 * rng.random((19, cells)) - 1))).astype(np.float32)
    u_lo, u_hi = wall_velocities(kind, 5)
    sim = plb.Simulation(*n, 0.7, kind, u_lo, u_hi)
    sim.write_populations(dev(f).view(-1))
    back = sim.read_populations().cpu().numpy()
    assert np.abs(back.astype(np.float64) - f.astype(np.float64)).max() <= 1.5e-7


# ------------------------------------------------------------------ O-3 / O-4 lbm_step, read_macros
@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("forced", [False, True])
def test_steps_match_oracle_all_boundaries(kind, forced):
    n = RAGGED
    cells = n[0] * n[1] * n[2]
    rho, u = wl.random_fields(11, cells)
    u_lo, u_hi = wall_velocities(kind, 13)
    sim, ora = make_pair(n, 0.65, kind, u_lo, u_hi)
    sim.set_equilibrium(dev(rho), dev(u), 1e-4, 77)
    ora.set_equilibrium(rho, u, 1e-4, 77)
    rng = np.random.default_rng(17)
    for s in range(6):
        g = 1e-3 * (2 * rng.random((3, cells)) - 1) if forced else None
        gd = pu.soa_to_forcing(sim, g) if forced else None     # must outlive read_macros (it adds g/2)
        sim.step(gd)
        ora.step(g)
        f_g = sim.read_populations().cpu().numpy().astype(np.float64)
        assert np.abs(f_g - ora.read_populations()).max() <= 3e-7, "step %d" % s
        rho_g, u_g = sim.read_macros()
        rho_o, u_o = ora.read_macros()
        assert np.abs(rho_g.cpu().numpy() - rho_o).max() <= 6e-7
        assert np.abs(u_g.cpu().numpy() - u_o).max() <= 6e-7
    sim.status()


# grids that take the vectorised kernel (nx % 4 == 0, x periodic): a warp spanning several rows
# (nx = 8, 40), exactly one row (128), part of a row (256); partial last warp; walls in y and z
VEC_SHAPES = [(40, 9, 11), (128, 7, 5), (8, 5, 5), (256, 4, 3), (4, 3, 2)]


@pytest.mark.parametrize("n", VEC_SHAPES)
@pytest.mark.parametrize("kind", [(0, 0, 0), (0, 1, 0), (0, 0, 1), (0, 1, 1)])
@pytest.mark.parametrize("forced", [False, True])
def test_steps_match_oracle_vector_path(n, kind, forced):
    cells = n[0] * n[1] * n[2]
    rho, u = wl.random_fields(41, cells)
    u_lo, u_hi = wall_velocities(kind, 43)
    sim, ora = make_pair(n, 0.7, kind, u_lo, u_hi)
    sim.set_equilibrium(dev(rho), dev(u), 1e-4, 99)
    ora.set_equilibrium(rho, u, 1e-4, 99)
    rng = np.random.default_rng(47)
    for s in range(5):
        g = 1e-3 * (2 * rng.random((3, cells)) - 1) if forced else None
        gd = pu.soa_to_forcing(sim, g) if forced else None
        sim.step(gd)
        ora.step(g)
        f_g = sim.read_populations().cpu().numpy().astype(np.float64)
        assert np.abs(f_g - ora.read_populations()).max() <= 3e-7, "step %d" % s
    rho_g, u_g = sim.read_macros()
    rho_o, u_o = ora.read_macros()
    assert np.abs(rho_g.cpu().numpy() - rho_o).max() <= 6e-7
    assert np.abs(u_g.cpu().numpy() - u_o).max() <= 6e-7
    sim.status()


def test_macros_before_any_step_and_null_outputs():
    n = (16, 8, 8)
    cells = n[0] * n[1] * n[2]
    rho, u = wl.random_fields(19, cells)
    sim, ora = make_pair(n, 0.9, (0, 1, 0))
    sim.set_equilibrium(dev(rho), dev(u))
    ora.set_equilibrium(rho, u)
    rho_o, u_o = ora.read_macros()
    r = torch.empty(cells, device=DEV)
    plb.lbm_read_macros(sim.h, r, None)
    assert np.abs(r.cpu().numpy() - rho_o).max() <= 3e-7
    v = torch.empty(3 * cells, device=DEV)
    plb.lbm_read_macros(sim.h, None, v)
    assert np.abs(v.view(3, -1).cpu().numpy() - u_o).max() <= 3e-7
    plb.lbm_read_macros(sim.h, None, None)


def test_mass_and_momentum_budget_on_gpu():
    """P1/P3 as properties of the CUDA path itself: mass constant, momentum gain = sum g."""
    n = (40, 24, 24)
    cells = n[0] * n[1] * n[2]
    rho, u = wl.random_fields(23, cells)
    sim = plb.Simulation(*n, 0.7, (0, 0, 0))
    sim.set_equilibrium(dev(rho), dev(u))
    rng = np.random.default_rng(29)
    g = 1e-3 * (2 * rng.random((3, cells)) - 1)
    gd = pu.soa_to_forcing(sim, g)
    f0 = sim.read_populations().double()
    sim.step(gd)
    f1 = sim.read_populations().double()
    c, _ = orc.lattice()
    cd = torch.as_tensor(c, dtype=torch.float64, device=DEV)
    assert abs(float(f1.sum() - f0.sum())) / cells <= 2e-8
    dj = (cd.t() @ f1 - cd.t() @ f0).sum(1).cpu().numpy()
    assert np.abs(dj - g.sum(1)).max() / cells <= 2e-8


# ------------------------------------------------------------------ closed forms on the GPU (P4, P5)
def test_couette_profile_on_gpu():
    nx, ny, nz, uw, tau = 8, 16, 8, 0.05, 0.8
    kind = (0, 1, 0)
    u_hi = np.zeros((3, 3)); u_hi[1, 0] = uw
    sim = plb.Simulation(nx, ny, nz, tau, kind, None, u_hi)
    sim.set_equilibrium()
    for _ in range(6000):
        sim.step(None)
    rho, u = sim.read_macros()
    ux = u[0].view(nz, ny, nx).cpu().numpy()
    lin = uw * (np.arange(ny) + 0.5) / ny
    assert np.abs(ux - lin[None, :, None]).max() <= 1e-4 * uw
    assert float((rho - 1).abs().max()) <= 1e-6
    assert float(u[1:].abs().max()) <= 1e-4 * uw


def test_config2_reduced_full_length_parity():
    """C2 shape at 64^3 (same tau, u0, one wavelength per box), all 1000 steps against the
    oracle, plus the closed-form decay u0 exp(-2 nu k^2 t) (P5)."""
    w = wl.config2(n=64, steps=1000)
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, w.steps)
    out = pu.compare(w, sim, ora)
    assert out["dv_rel"] <= 1e-4 and out["drho"] <= 1e-6
    _, u = sim.read_macros()
    u = u.cpu().numpy().astype(np.float64)
    amp = (u[:2] * w.u0[:2]).sum() / (w.u0[:2] ** 2).sum()
    nu, k = (w.tau - 0.5) / 3, 2 * math.pi / 64
    assert amp == pytest.approx(math.exp(-2 * nu * k * k * w.steps), rel=5e-3)


def test_config2_full_size_against_slab_oracle():
    """C2 at the full 256^3, in the launch configuration bench.py times.  The Taylor-Green field
    is uniform in z and the update is translation-invariant, so every z-plane of the 256^3 run
    equals the oracle run on a 256 x 256 x 4 periodic slab of the same seeded field: the oracle
    computes the sampled planes exactly.  200 steps by default, all 1000 with PLB_FULL=1."""
    steps = 1000 if FULL else 200
    w = wl.config2()
    sim = plb.Simulation.from_workload(w)
    for _ in range(steps):
        sim.step(None)
    sim.status()
    ws = wl.config2()
    ws.nz = 4
    ws.u0 = np.ascontiguousarray(w.u0.reshape(3, 256, 256 * 256)[:, :4].reshape(3, -1))
    ora = orc.Oracle.from_workload(ws)
    for _ in range(steps):
        ora.step(None)
    rho_o, u_o = ora.read_macros()
    rho_g, u_g = sim.read_macros()
    rho_g = rho_g.view(256, -1)
    u_g = u_g.view(3, 256, -1)
    plane = 256 * 256
    for kz in (0, 1, 127, 255):                       # sampled planes, incl. the periodic seam
        assert np.abs(rho_g[kz].cpu().numpy() - rho_o[:plane]).max() <= 1e-6
        assert np.abs(u_g[:, kz].cpu().numpy() - u_o[:, :plane]).max() <= 1e-4 * w.u_ref
    # z-invariance of the GPU result (so the sampled planes speak for all of them)
    assert float((rho_g - rho_g[0:1]).abs().max()) == 0.0
    assert float((u_g - u_g[:, 0:1]).abs().max()) == 0.0
    nu, k = (w.tau - 0.5) / 3, 2 * math.pi / 256
    u0 = torch.as_tensor(w.u0[:2], dtype=torch.float64, device=DEV)
    amp = float((u_g.view(3, -1)[:2].double() * u0).sum() / (u0 * u0).sum())
    assert amp == pytest.approx(math.exp(-2 * nu * k * k * steps), rel=1e-3)


def test_maximum_size_grid_against_slab_oracle():
    """Largest grid that fits one B200 beside the test's own buffers: 1024 x 512 x 1280 = 671 M cells
    (ten times config 4; 102 GB of populations, byte offsets far beyond 2^32, cell indices beyond
    2^29).  Same device as the config-2 full-size test: a field uniform in z, so every z-plane must
    equal the oracle run on a 4-plane periodic slab of the same field.  Walls in y with a moving top
    wall, so the bounce-back rows are exercised at this size too."""
    nx, ny, nz, steps = 1024, 512, 1280, 10
    free, _ = torch.cuda.mem_get_info()
    if free < 150e9:
        pytest.skip("needs ~145 GB of free device memory")
    kind = (0, 1, 0)
    u_hi = np.zeros((3, 3)); u_hi[1, 0] = 0.05
    plane_u = wl.taylor_green_field(nx, ny, 1, 0.02)                     # [3, ny*nx], 2-D vortex in x-y
    sim = plb.Simulation(nx, ny, nz, 0.6, kind, None, u_hi)
    u_dev = torch.as_tensor(plane_u, dtype=torch.float32, device=DEV).view(3, 1, ny * nx).expand(3, nz, ny * nx).contiguous()
    sim.set_equilibrium(None, u_dev.view(-1))
    del u_dev
    for _ in range(steps):
        sim.step(None)
    sim.status()
    ora = orc.Oracle(nx, ny, 4, 0.6, kind, None, u_hi)
    ora.set_equilibrium(None, np.ascontiguousarray(np.broadcast_to(plane_u.reshape(3, 1, ny * nx), (3, 4, ny * nx))).reshape(3, -1))
    for _ in range(steps):
        ora.step(None)
    rho_o, u_o = ora.read_macros()
    rho_g, u_g = sim.read_macros()
    rho_g = rho_g.view(nz, -1)
    u_g = u_g.view(3, nz, -1)
    plane = nx * ny
    for kz in (0, 1, nz // 2 + 1, nz - 1):
        assert np.abs(rho_g[kz].cpu().numpy() - rho_o[:plane]).max() <= 1e-6
        assert np.abs(u_g[:, kz].cpu().numpy() - u_o[:, :plane]).max() <= 1e-4 * 0.05
    assert float((rho_g - rho_g[0:1]).abs().max()) == 0.0                 # every plane equals plane 0
    for d in range(3):
        assert float((u_g[d] - u_g[d, 0:1]).abs().max()) == 0.0
    assert abs(float(rho_g.double().sum()) / (nx * ny * nz) - 1.0) <= 1e-9   # mass
    sim.close(); ora.close()


def test_check_finite_counts_broken_cells():
    """debug aid: 0 on a healthy state, the number of poisoned cells otherwise"""
    sim = plb.Simulation(16, 12, 10, 0.7, (0, 1, 0))
    with pytest.raises(plb.PlbError) as e:
        sim.check_finite()                                   # populations not set yet
    assert e.value.code == plb.PLB_ERR_ORDER
    sim.set_equilibrium()
    for _ in range(3):
        sim.step(None)
    assert sim.check_finite() == 0
    clean = sim.read_populations().clone()
    for d, q, value in ((5, 100, float("nan")), (2, 1500, float("inf"))):
        f = clean.clone()
        f[d, q] = value                                     # one population of one cell
        sim.write_populations(f)
        assert sim.check_finite() == 1
    f = clean.clone()
    f[:, 16 * 12 * 5 + 16 * 6 + 8] = -1.0                   # one cell with density -19: that cell, no other
    sim.write_populations(f)
    assert sim.check_finite() == 1
    f = clean.clone()
    f[18, 7] = -2.0                                         # finite populations, density <= 0
    f[18, 16 * 12 * 10 - 1] = -2.0                          # ... also in a wall-row cell
    sim.write_populations(f)
    assert sim.check_finite() == 2
    sim.write_populations(clean)
    assert sim.check_finite() == 0
    sim.close()


# ------------------------------------------------------------------ edge cases
def test_degenerate_grids():
    """1-cell-thick periodic axes (a link wraps onto its own cell) and a 1-layer channel."""
    for n, kind in (((1, 1, 1), (0, 0, 0)), ((5, 1, 3), (0, 0, 0)), ((7, 1, 4), (0, 1, 0)), ((1, 6, 1), (0, 1, 0))):
        cells = n[0] * n[1] * n[2]
        rho, u = wl.random_fields(31, cells)
        u_hi = np.zeros((3, 3)); u_hi[1, 0] = 0.03
        sim, ora = make_pair(n, 0.8, kind, None, u_hi if kind[1] else None)
        sim.set_equilibrium(dev(rho), dev(u))
        ora.set_equilibrium(rho, u)
        for _ in range(3):
            sim.step(None)
            ora.step(None)
        assert np.abs(sim.read_populations().cpu().numpy() - ora.read_populations()).max() <= 3e-7, (n, kind)


def test_call_order_and_argument_errors():
    sim = plb.Simulation(8, 8, 8, 0.8)
    with pytest.raises(plb.PlbError) as e:
        sim.step(None)                                   # populations not set
    assert e.value.code == plb.PLB_ERR_ORDER
    sim.set_equilibrium()
    with pytest.raises(plb.PlbError) as e:
        sim.set_equilibrium(noise_amp=-1.0)
    assert e.value.code == plb.PLB_ERR_ARG
    misaligned = torch.zeros(8 * 8 * 8 * 4 + 1, device=DEV)[1:]
    with pytest.raises(plb.PlbError) as e:
        sim.step(misaligned)
    assert e.value.code == plb.PLB_ERR_ARG
    with pytest.raises(plb.PlbError) as e:
        plb.Simulation(8, 8, 8, 0.5)                     # tau must exceed 1/2
    assert e.value.code == plb.PLB_ERR_ARG
    ws = torch.empty(1024, dtype=torch.uint8, device=DEV)
    with pytest.raises(plb.PlbError) as e:
        plb.lbm_create(8, 8, 8, 0.8, plb.make_boundary((0, 0, 0)), ws, 0, 0, None)
    assert e.value.code == plb.PLB_ERR_WORKSPACE
