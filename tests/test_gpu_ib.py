"""GPU parity tests of the immersed-boundary / membrane part of libplb against the fp64 CPU
oracle, through the C-ABI.  Same seeded inputs on both sides; nothing the oracle consumes or is
compared with comes from the CUDA path.

Tolerances: node positions within 1e-4 lattice units, |dv| <= 1e-4 u_ref, |drho| <= 1e-6 at the
end of a run (BASELINE.json north_star); single calls to fp32 round-off of the quantities
involved (stated at each assert)."""
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
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def dev(a, dtype=torch.float32):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to(DEV).contiguous()


# ------------------------------------------------------------------ O-8 Philox
def test_philox_known_answers_on_device():
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    ctr = np.array([[int(x, 16) for x in r[0:4]] for r in rows], dtype=np.uint32)
    key = np.array([[int(x, 16) for x in r[4:6]] for r in rows], dtype=np.uint32)
    exp = np.array([[int(x, 16) for x in r[6:10]] for r in rows], dtype=np.uint32)
    d_ctr = torch.as_tensor(ctr.view(np.int32)).to(DEV)
    d_key = torch.as_tensor(key.view(np.int32)).to(DEV)
    d_out = torch.zeros_like(d_ctr)
    plb.plb_philox4x32_10(d_ctr, d_key, d_out)
    torch.cuda.synchronize()
    assert (d_out.cpu().numpy().view(np.uint32) == exp).all()


def test_philox_equals_oracle_on_many_counters():
    rng = np.random.default_rng(41)
    n = 100_000
    ctr = rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    d_ctr = torch.as_tensor(ctr.view(np.int32)).to(DEV)
    d_key = torch.as_tensor(key.view(np.int32)).to(DEV)
    d_out = torch.zeros_like(d_ctr)
    plb.plb_philox4x32_10(d_ctr, d_key, d_out)
    out = d_out.cpu().numpy().view(np.uint32)
    for t in rng.integers(0, n, size=2000):
        assert out[t].tolist() == orc.philox4x32_10(ctr[t], key[t])


# ------------------------------------------------------------------ helpers
def mesh_pair(n, kind, xyz, edges, rest, k, tau=0.8, u_hi=None):
    sim = plb.Simulation(*n, tau, kind, None, u_hi, max_nodes=xyz.shape[0], max_edges=max(1, edges.shape[0]))
    ora = orc.Oracle(*n, tau, kind, None, u_hi)
    sim.add_mesh(xyz, edges, rest, k)
    ora.add_mesh(xyz, edges, rest, k)
    return sim, ora


def scattered_nodes(n, kind, count, seed):
    """Seeded node cloud exercising every stencil case: periodic seams, unwrapped coordinates far
    outside the box, exact integers, stencils that cross a wall (dropped cells, G15)."""
    rng = np.random.default_rng(seed)
    X = rng.random((count, 3)) * np.asarray(n, dtype=np.float64)
    X[0] = (0.2, 3.3, n[2] - 0.1)
    X[1] = (4.0, 5.0, 2.0)
    X[2] = (n[0] - 0.01, 4.5, 0.01)
    for a in range(3):
        if kind[a] == 0:
            X[3, a] += 3 * n[a]                # unwrapped, several boxes away
            X[4, a] -= 2 * n[a]
        else:
            X[5, a] = 0.3                      # low wall: two layers of the stencil dropped
            X[6, a] = n[a] - 1.2               # high wall
            X[7, a] = -0.4
            X[8, a] = n[a] - 0.6
    return X


# ------------------------------------------------------------------ O-5 membrane forces
@pytest.mark.parametrize("sigma", [0.0, 1e-4])
def test_membrane_forces_match_oracle(sigma):
    w = wl.config1()
    xyz = np.concatenate([w.mesh_xyz[0], w.mesh_xyz[0] + (300.0, 0.0, 700.0)])   # a far copy: large coordinates
    e = np.concatenate([w.edges, w.edges + w.mesh_xyz.shape[1]])
    rest = np.concatenate([w.rest, w.rest])
    sim, ora = mesh_pair((32, 32, 64), w.kind, xyz, e, rest, w.k_spring)
    sim.compute_membrane_forces(sigma, 99, 17)
    ora.compute_membrane_forces(sigma, 99, 17)
    F_g, F_o = sim.read_forces().astype(np.float64), ora.read_forces()
    scale = np.abs(F_o).max()
    assert scale > 1e-4
    # sums of <= 6 edge terms of size <= scale, each formed with ~4 fp32 roundings
    assert np.abs(F_g - F_o).max() <= 2e-6 * scale
    if sigma == 0.0:
        assert np.abs(F_g.sum(0)).max() <= 1e-7          # P14: springs sum to zero


def test_membrane_force_default_rest_lengths_and_zero_edge():
    rng = np.random.default_rng(43)
    X = rng.random((12, 3)) * 4 + 8
    e = np.array([(a, b) for a in range(12) for b in range(a + 1, 12)][:30], dtype=np.int32)
    sim, ora = mesh_pair((24, 24, 24), (0, 0, 0), X, e, None, 0.05)
    sim.compute_membrane_forces()
    # rest = initial lengths => F = 0 up to the fp32 rounding of the stored rest length (k ulp(L))
    assert np.abs(sim.read_forces()).max() <= 0.05 * 11 * 6e-8 * 7
    Y = X.copy(); Y[1] = Y[0]                             # collapse an edge: |R| = 0 is an error
    sim.write_nodes(Y)
    sim.compute_membrane_forces()
    with pytest.raises(plb.PlbError) as err:
        sim.status()
    assert err.value.code == plb.PLB_ERR_ARG


# ------------------------------------------------------------------ O-6 spread
SPREAD_FORMS = ["scatter", "aggregate", "gather"]


@pytest.mark.parametrize("mode", SPREAD_FORMS)
@pytest.mark.parametrize("kind", [(0, 0, 0), (0, 1, 0), (1, 1, 1)])
def test_spread_matches_oracle(kind, mode):
    n = (37, 19, 23)
    X = scattered_nodes(n, kind, 400, 47)
    F = np.random.default_rng(53).standard_normal((400, 3))
    sim, ora = mesh_pair(n, kind, X, np.zeros((0, 2), dtype=np.int32), None, 0.0)
    sim.set_spread_mode(mode)
    assert sim.spread_mode() == plb.SPREAD_MODES[mode]
    sim.write_forces(F)
    ora.write_forces(F)
    sim.spread()
    g_g = pu.forcing_to_soa(sim)
    g_o = ora.spread()
    assert np.abs(g_o).max() > 0.1
    assert np.abs(g_g - g_o).max() <= 2e-6               # ~10 contributions of O(1) per cell, fp32
    full = np.ones(400, dtype=bool)
    for a in range(3):
        if kind[a] == 1:
            full &= (np.floor(X[:, a]) - 1 >= 0) & (np.floor(X[:, a]) + 2 <= n[a] - 1)
    if full.all():                                        # P10 on the GPU result
        assert np.abs(g_g.sum(1) - F.sum(0)).max() <= 2e-4
    # a second spread on the same buffer first clears what the first one wrote
    X2 = scattered_nodes(n, kind, 400, 59)
    sim.write_nodes(X2)
    ora.write_nodes(X2)
    sim.write_forces(F)
    ora.write_forces(F)
    sim.spread()
    assert np.abs(pu.forcing_to_soa(sim) - ora.spread()).max() <= 2e-6


@pytest.mark.parametrize("mode", SPREAD_FORMS)
def test_spread_dense_meshes_all_forms(mode):
    """Densely sampled tiles (config 5's shape: 2562 nodes on ~2700 tile cells, ~6 nodes per occupied
    base cell): one platelet in the interior, one across the periodic x seam (unwrapped), one
    poking through the y wall (clipped tile, dropped cells G15), one 12-node mesh (fixed-point
    scale bounded by the single product, not by the node count) and one with zero force."""
    n = (40, 24, 36)
    kind = (0, 1, 0)
    v4, e4, _ = wl.icosphere(4)
    v0, e0, _ = wl.icosphere(0)
    rng = np.random.default_rng(83)
    sim = plb.Simulation(*n, 0.8, kind, max_nodes=4 * len(v4) + len(v0), max_edges=1)
    ora = orc.Oracle(*n, 0.8, kind)
    meshes = [v4 * (5.0, 5.0, 1.25) + (20.3, 12.1, 18.7),
              v4 * (5.0, 1.25, 5.0) + (39.6 + 40.0, 11.0, 9.2),
              v4 * (1.25, 5.0, 5.0) + (11.1, 2.2, 27.9),
              v0 * (1.5, 1.5, 1.5) + (30.2, 18.4, 30.1),
              v4 * (5.0, 5.0, 1.25) + (8.0, 17.0, 8.0)]
    edges = np.zeros((0, 2), dtype=np.int32)
    for x in meshes:
        sim.add_mesh(x, edges, None, 0.0)
        ora.add_mesh(x, edges, None, 0.0)
    sim.set_spread_mode(mode)
    F = rng.standard_normal((sim.n_nodes, 3)) * np.array([1.0, 0.3, 2.0])
    F[-len(v4):] = 0.0
    F[3 * len(v4)] *= 50.0                                     # one dominant nodal force in the tiny mesh
    sim.write_forces(F)
    ora.write_forces(F)
    sim.spread()
    g_g, g_o = pu.forcing_to_soa(sim), ora.spread()
    scale = np.abs(g_o).max()
    assert scale > 1.0                                         # the field is not trivially small
    # a cell collects up to ~300 contributions, each rounded to the tile's fixed-point quantum
    # q = (n/8) 2^-30 max|F|: error ~ q sqrt(300/12) ~ 5 q, 40 q allowed;
    # the fp32 products add ~300 x 6e-8 x |F W| on top
    quantum = (len(v4) / 8.0) * 2.0 ** -29 * np.abs(F).max()
    assert np.abs(g_g - g_o).max() <= 40 * quantum + 2e-6 * scale
    # the forms agree with each other to a few quanta: same products, order-independent integer
    # sums (the scatter form rounds a product twice, the binned forms once)
    sim.set_spread_mode("scatter" if mode != "scatter" else "aggregate")
    sim.write_forces(F)
    sim.spread()
    assert np.abs(pu.forcing_to_soa(sim) - g_g).max() <= 20 * quantum
    sim.close(); ora.close()


def test_spread_forms_are_reproducible():
    """integer tile accumulation: the sum a block forms in its tile does not depend on the order
    in which its nodes arrive, so repeated launches agree up to the order of the float adds with
    which OVERLAPPING tiles (patches of one mesh, interpenetrating meshes) meet in the forcing
    field: a few fp32 roundings of the cell value, and nothing at all where one tile owns a cell"""
    w = wl.config5(n=32, grid_xz=4, layers=2, steps=1, subdiv=4)
    sim = plb.Simulation.from_workload(w)
    for mode in SPREAD_FORMS:
        sim.set_spread_mode(mode)
        outs = []
        for _ in range(3):
            sim.compute_membrane_forces(1e-4, 5, 0)
            sim.spread()
            outs.append(sim.forcing.clone())
        scale = float(outs[0].abs().max())
        assert scale > 0.0
        for o in outs[1:]:
            assert float((o - outs[0]).abs().max()) <= 8 * 6e-8 * scale
    sim.close()


def test_node_order_is_hidden():
    """the library stores the nodes of a mesh in its own (Morton) order; every call that names a
    node speaks the caller's indices: positions, forces, velocities round-trip unchanged, and the
    Philox force noise is keyed on the caller's global node index"""
    w = wl.config3(nx=64, ny=32, nz=64, n_meshes=3, steps=1)
    sim = plb.Simulation.from_workload(w)
    X = w.mesh_xyz.reshape(-1, 3)
    assert np.array_equal(sim.read_nodes(), X)
    Y = X + np.random.default_rng(89).random(X.shape)
    sim.write_nodes(Y)
    assert np.array_equal(sim.read_nodes(), Y)
    F = np.random.default_rng(97).standard_normal(X.shape).astype(np.float32)
    sim.write_forces(F)
    assert np.array_equal(sim.read_forces(), F)
    sim.write_nodes(X)
    sim.compute_membrane_forces(0.5, 1234, 7)                  # rest lengths = initial lengths: noise only
    Fn = sim.read_forces().astype(np.float64)
    for m in (0, 1, 641, 642, 1925):
        z = 0.5 * np.asarray(orc.noise_normal3(1234, m, 7, 2))
        assert np.abs(Fn[m] - z).max() <= 1e-5
    sim.close()


def test_spread_requires_forces_and_buffer():
    X = np.full((1, 3), 4.0)
    sim, _ = mesh_pair((8, 8, 8), (0, 0, 0), X, np.zeros((0, 2), dtype=np.int32), None, 0.0)
    with pytest.raises(plb.PlbError) as e:
        sim.spread()
    assert e.value.code == plb.PLB_ERR_ORDER
    sim.compute_membrane_forces()
    with pytest.raises(plb.PlbError) as e:
        plb.ib_spread(sim.h, None)
    assert e.value.code == plb.PLB_ERR_ARG


# ------------------------------------------------------------------ O-7 interpolate + advance
@pytest.mark.parametrize("kind", [(0, 0, 0), (0, 1, 0), (1, 1, 1)])
def test_interpolate_advance_matches_oracle(kind):
    n = (37, 19, 23)
    cells = n[0] * n[1] * n[2]
    X = scattered_nodes(n, kind, 400, 61)
    for a in range(3):                                    # keep every node inside the channel
        if kind[a] == 1:
            X[:, a] = np.clip(X[:, a], -0.3, n[a] - 0.7)
    F = 1e-2 * np.random.default_rng(67).standard_normal((400, 3))
    rho, u = wl.random_fields(71, cells)
    sim, ora = mesh_pair(n, kind, X, np.zeros((0, 2), dtype=np.int32), None, 0.0)
    sim.set_equilibrium(dev(rho), dev(u))
    ora.set_equilibrium(rho, u)
    for s in (sim, ora):
        s.write_forces(F)
    sim.spread(); sim.step(sim.forcing); sim.interpolate_advance()
    g = ora.spread(); ora.step(g); ora.interpolate_advance()
    sim.status()
    U_g, U_o = sim.read_node_velocities().astype(np.float64), ora.read_node_velocities()
    assert np.abs(U_o).max() > 1e-3
    assert np.abs(U_g - U_o).max() <= 1e-6                # 64 products of O(0.03) x O(1) in fp32
    assert np.abs(sim.read_nodes() - ora.read_nodes()).max() <= 1e-6
    # the macros after a forced step carry g/2 (L201)
    rho_g, u_g = sim.read_macros()
    rho_o, u_o = ora.read_macros()
    assert np.abs(u_g.cpu().numpy() - u_o).max() <= 6e-7
    assert np.abs(rho_g.cpu().numpy() - rho_o).max() <= 6e-7


@pytest.mark.parametrize("form", ["tile", "tile-own-box", "direct", "pull"])
@pytest.mark.parametrize("mode", SPREAD_FORMS)
def test_interpolation_forms_cover_forceless_and_weak_nodes(form, mode, monkeypatch):
    """the listed-cells forms ("tile", "direct") rely on ib_spread listing every cell inside some
    node's stencil, whatever its force; the pull form needs no list.  A mesh with NO force, one whose
    forces are 1e-12 of the neighbouring mesh's (they round to zero in the tile's fixed point) and
    nodes sitting exactly on lattice points (zero weights) all get the oracle's velocity from every
    form of the interpolation (PLB_INTERP: measurement knob; default = by sampling density)"""
    monkeypatch.setenv("PLB_INTERP", "tile" if form == "tile-own-box" else form)
    if form == "tile-own-box":
        monkeypatch.setenv("PLB_BOX_CAP", "2")                     # ranges beyond the second compute their own box
    n = (40, 24, 36)
    kind = (0, 1, 0)
    cells = n[0] * n[1] * n[2]
    v2, _, _ = wl.icosphere(2)
    meshes = [v2 * (4.0, 4.0, 1.0) + (20.3, 12.1, 18.7),
              v2 * (4.0, 1.0, 4.0) + (39.6, 11.0, 9.2),            # across the periodic x seam
              v2 * (1.0, 4.0, 4.0) + (11.1, 3.6, 27.9),            # against the y wall (clipped stencils)
              np.round(v2 * (4.0, 4.0, 1.0) + (30.0, 14.0, 30.0))]  # nodes on lattice points
    sim = plb.Simulation(*n, 0.8, kind, max_nodes=4 * len(v2), max_edges=1)
    ora = orc.Oracle(*n, 0.8, kind)
    edges = np.zeros((0, 2), dtype=np.int32)
    for x in meshes:
        sim.add_mesh(x, edges, None, 0.0)
        ora.add_mesh(x, edges, None, 0.0)
    sim.set_spread_mode(mode)
    rng = np.random.default_rng(101)
    F = 1e-2 * rng.standard_normal((sim.n_nodes, 3))
    F[:len(v2)] = 0.0                                              # mesh 0: no force at all
    F[len(v2):len(v2) + len(v2) // 2] *= 1e-12                      # half of mesh 1: far below the tile's quantum
    rho, u = wl.random_fields(103, cells)
    sim.set_equilibrium(dev(rho), dev(u))
    ora.set_equilibrium(rho, u)
    for s_ in (sim, ora):
        s_.write_forces(F)
    sim.spread(); sim.step(sim.forcing); sim.interpolate_advance()
    g = ora.spread(); ora.step(g); ora.interpolate_advance()
    sim.status()
    U_g, U_o = sim.read_node_velocities().astype(np.float64), ora.read_node_velocities()
    assert np.abs(U_o).max() > 1e-3
    assert np.abs(U_g - U_o).max() <= 1e-6
    assert np.abs(sim.read_nodes() - ora.read_nodes()).max() <= 1e-6
    sim.close(); ora.close()


def test_P13_passive_advection_across_the_seam():
    """GPU twin of the oracle pin P13: lbm_step(NULL) -> ib_interpolate_advance with NO spread in
    between (Eq. 33 alone).  A pre-stressed mesh in a uniform periodic flow translates rigidly by u0
    per step, crosses the x seam with unwrapped coordinates, and keeps its spring forces."""
    nx, ny, nz = 12, 10, 9
    v, _, e = wl.icosphere(1)
    x0 = 2.5 * v + np.array([nx - 3.0, 5.0, 4.5])
    u0 = np.array([0.09, -0.02, 0.035])
    rest = 0.9 * wl.edge_lengths(x0, e)
    sim, ora = mesh_pair((nx, ny, nz), (0, 0, 0), x0, e, rest, 0.3)
    uf = np.tile(u0[:, None], (1, nx * ny * nz))
    sim.set_equilibrium(None, dev(uf)); ora.set_equilibrium(None, uf)
    sim.compute_membrane_forces(); ora.compute_membrane_forces()
    F0 = sim.read_forces().astype(np.float64)
    assert np.abs(F0 - ora.read_forces()).max() <= 2e-6 * np.abs(F0).max()
    for n in range(1, 61):
        sim.step(None); sim.interpolate_advance()
        ora.step(None); ora.interpolate_advance()
    sim.status()
    X = sim.read_nodes()
    assert np.abs(X - (x0 + 60 * u0)).max() <= 60 * 2e-7          # fp32 velocities, fp64 positions
    assert np.abs(X - ora.read_nodes()).max() <= 60 * 2e-7
    assert np.abs(sim.read_node_velocities() - u0).max() <= 2e-7
    assert X[:, 0].max() > nx + 2                                 # unwrapped storage (G17)
    sim.compute_membrane_forces()
    assert np.abs(sim.read_forces() - F0).max() <= 1e-5 * np.abs(F0).max()
    sim.close(); ora.close()


def test_release_forcing_forgets_the_buffers():
    """ib_release_forcing clears what the last spread wrote and drops the pointers: the caller may
    free the buffer, the next spread may go to another one, the macros see g = 0"""
    w = wl.config1(steps=3)
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, 3)
    first = sim.forcing
    assert float(first.abs().max()) > 0.0
    plb.ib_release_forcing(sim.h)
    assert float(first.abs().max()) == 0.0
    sim.forcing = torch.zeros_like(first)
    del first
    _, u_g = sim.read_macros()                                   # g = 0 now: plain u = sum c f / rho
    f = sim.read_populations().double()
    c = torch.as_tensor(orc.lattice()[0], dtype=torch.float64, device=f.device)     # [19, 3]
    u_plain = (c.t() @ f) / f.sum(0)
    assert float((u_g.double() - u_plain).abs().max()) <= 2e-7
    sim.coupled_step(); ora.coupled_step()
    out = pu.compare(w, sim, ora)
    assert out["dX"] <= 1e-6
    sim.close(); ora.close()


@pytest.mark.parametrize("mode", SPREAD_FORMS)
def test_spread_alternating_buffers_many_times(mode):
    """ib_spread clears what the previous call wrote -- into whichever buffer that was -- while the
    spread kernel already runs (it is a programmatic dependent launch behind the clear and waits
    just ahead of its flush): 40 spreads alternating between two buffers, the nodes moved in
    between, must each leave the oracle's field in one buffer and exact zeros in the other"""
    w = wl.config3(nx=64, ny=32, nz=64, n_meshes=3, steps=1)
    sim, ora = pu.build_pair(w)
    sim.set_spread_mode(mode)
    A, B = sim.forcing, torch.zeros_like(sim.forcing)
    X0 = w.mesh_xyz.reshape(-1, 3)
    rng = np.random.default_rng(113)
    for it in range(40):
        X = X0 + rng.uniform(-1.5, 1.5, size=(1, 3)) + 0.05 * rng.standard_normal(X0.shape)
        sim.write_nodes(X); ora.write_nodes(X)
        sim.compute_membrane_forces(); ora.compute_membrane_forces()
        tgt, other = (A, B) if it % 2 == 0 else (B, A)
        sim.spread(tgt)
        g_o = ora.spread()
        assert float(other.abs().max()) == 0.0
        g_g = tgt.view(-1, 4)[:, :3].t().cpu().numpy().astype(np.float64)
        # the gather form rounds every single product W F to 2^-22 of max|F|/8 (ib.cu), ~13 of them per
        # cell: a few 1e-6 of the field's maximum; the other forms round once per (node, cell) at 2^-30
        tol = 6e-6 if mode == "gather" else 2e-6
        assert np.abs(g_g - g_o.reshape(3, -1)).max() <= tol * max(np.abs(g_o).max(), 1e-30)
    sim.close(); ora.close()


def test_node_leaving_channel_is_reported():
    n = (8, 8, 8)
    u = np.zeros((3, 512)); u[1] = 0.2                    # fluid moving towards the wall
    X = np.array([[4.0, 7.49, 4.0]])
    sim, ora = mesh_pair(n, (0, 1, 0), X, np.zeros((0, 2), dtype=np.int32), None, 0.0)
    sim.set_equilibrium(None, dev(u))
    ora.set_equilibrium(None, u)
    sim.coupled_step()
    with pytest.raises(orc.OracleError) as eo:
        ora.coupled_step()
    assert eo.value.code == -5
    with pytest.raises(plb.PlbError) as eg:
        sim.status()
    assert eg.value.code == plb.PLB_ERR_NODE_LEFT


def test_no_meshes_is_a_no_op():
    sim = plb.Simulation(8, 8, 8, 0.8)
    sim.set_equilibrium()
    sim.coupled_step()
    sim.status()
    assert sim.n_nodes == 0 and float(sim.forcing.abs().max()) == 0.0


def test_capacity_is_enforced():
    X = np.full((4, 3), 4.0) + np.arange(4)[:, None] * 0.1
    sim = plb.Simulation(8, 8, 8, 0.8, max_nodes=4, max_edges=1)
    sim.add_mesh(X, np.array([[0, 1]], dtype=np.int32))
    with pytest.raises(plb.PlbError) as e:
        sim.add_mesh(X, np.array([[0, 1]], dtype=np.int32))
    assert e.value.code == plb.PLB_ERR_WORKSPACE
    with pytest.raises(plb.PlbError) as e:
        plb.Simulation(8, 8, 8, 0.8, max_nodes=4, max_edges=1).add_mesh(X, np.array([[0, 4]], dtype=np.int32))
    assert e.value.code == plb.PLB_ERR_ARG
