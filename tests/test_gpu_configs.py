"""GPU-vs-oracle parity on the five BASELINE.json configs, through the C-ABI.

* C1 runs whole (200 steps) against the fp64 oracle.
* C3, C4, C5 run (a) scaled down -- same recipe, tau, wall speed, mesh shape and spring constant,
  smaller grid / fewer meshes / fewer steps -- whole against the oracle, and (b) at FULL size in
  the launch configuration bench.py times, where the oracle recomputes the first 20 / 20 / 6 coupled
  steps on a sub-block cut from the seeded inputs alone (parity_utils.Block) and size-independent
  properties (mass, total spread force = total node force, springs sum to zero) are checked.
* C2 is in test_gpu_lbm.py (reduced whole run + full-size slab oracle).
* PLB_FULL=1 adds the full-length, full-size, whole-domain runs of C3 (2000 steps), C4 (500) and
  C5 (200) against the oracle (2, 12 and 25 minutes on the GPU box's 16 host cores; results in
  profiles/r02_full_parity.md).

Tolerances are the north_star's: |dv| <= 1e-4 u_wall, |drho| <= 1e-6, |dX| <= 1e-4."""
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


def run_and_compare(w, steps=None):
    sim, ora = pu.build_pair(w)
    pu.run_pair(w, sim, ora, w.steps if steps is None else steps)
    out = pu.compare(w, sim, ora)
    sim.close(); ora.close()
    return out


def test_config1_whole():
    w = wl.config1()
    assert (w.nx, w.ny, w.nz, w.steps, w.n_nodes, w.n_edges) == (32, 32, 64, 200, 162, 480)
    out = run_and_compare(w)
    print("C1", out)


def test_config3_scaled_whole():
    w = wl.config3(nx=64, ny=32, nz=128, n_meshes=4, steps=400)
    out = run_and_compare(w)
    print("C3 scaled", out)


def test_config4_scaled_whole():
    w = wl.config4(nx=96, ny=48, nz=128, n_meshes=12, steps=150)
    out = run_and_compare(w)
    print("C4 scaled", out)


def test_config5_scaled_whole():
    """contention shape: meshes on a pitch-4 jittered lattice in the bottom slab, per-step Philox
    force noise (sigma = 1e-4)"""
    w = wl.config5(n=64, grid_xz=16, layers=2, steps=40, subdiv=2)
    assert w.force_sigma == 1e-4 and w.n_nodes == 512 * 162
    out = run_and_compare(w)
    print("C5 scaled", out)


# ------------------------------------------------------------------ full size
def full_size_block_parity(w, steps, inner, mesh_id):
    sim = plb.Simulation.from_workload(w)
    centre = w.mesh_xyz[mesh_id].mean(axis=0)
    blk = pu.Block(w, np.floor(centre).astype(int) - inner // 2, inner, steps, 12.5)
    wb, ids = pu.block_workload(w, blk)
    assert mesh_id in ids
    ora = orc.Oracle.from_workload(wb)
    # global node ids of the block's meshes (the force noise is keyed on the global node index)
    nn = w.mesh_xyz.shape[1]
    F_tot = None
    for s in range(steps):
        sim.compute_membrane_forces(w.force_sigma, w.force_seed, s)
        if s == steps - 1:
            F_tot = sim.read_forces().astype(np.float64)
        sim.spread()
        if s == steps - 1:
            g_sum = sim.forcing.view(-1, 4).double().sum(0)[:3].cpu().numpy()
        sim.step(sim.forcing)
        sim.interpolate_advance()
        block_coupled_step(ora, w, ids, nn, s)
    sim.status()
    # --- sampled outputs the oracle computed from the seeded inputs
    rho_g, u_g = sim.read_macros()
    rho_o, u_o = ora.read_macros()
    sl = blk.inner_slices()
    bz, by, bx = blk.size[2], blk.size[1], blk.size[0]
    d_rho = np.abs(blk.take_field(rho_g.view(1, -1))[sl] - rho_o.reshape(1, bz, by, bx)[sl]).max()
    d_u = np.abs(blk.take_field(u_g)[sl] - u_o.reshape(3, bz, by, bx)[sl]).max()
    X_g = sim.read_nodes().reshape(w.n_meshes, nn, 3)[ids]
    X_o = ora.read_nodes().reshape(len(ids), nn, 3)
    Xl = blk.local(X_g)
    clean = blk.near_inner(X_o, -3.0)                      # nodes whose stencil stayed well inside
    assert clean.sum() >= 100
    d_X = np.abs(Xl - X_o)[clean].max()
    moved = np.abs(X_o - wb.mesh_xyz)[clean].max()
    assert moved > 1e-3                                     # the nodes really were advected
    assert d_rho <= pu.TOL_RHO and d_u <= pu.TOL_V_REL * w.u_ref and d_X <= pu.TOL_X, (d_rho, d_u, d_X)
    # --- properties that hold at any size
    cells = w.cells
    assert abs(float(rho_g.double().sum()) / cells - 1.0) <= 1e-7             # P1 mass
    assert np.abs(g_sum - F_tot.sum(0)).max() <= 1e-6 * np.abs(F_tot).sum() + 1e-9          # P10
    if w.force_sigma == 0.0:
        per_mesh = F_tot.reshape(w.n_meshes, nn, 3).sum(1)
        assert np.abs(per_mesh).max() <= 1e-6                                 # P14 springs sum to zero
    sim.close(); ora.close()
    return d_rho, d_u, d_X


def block_coupled_step(ora, w, ids, nn, step):
    """one coupled step of the block oracle; the per-node Philox force noise of C5 is keyed on the
    GLOBAL node index, so it is drawn with the oracle's own generator for the block's nodes"""
    if ora.n_nodes == 0:
        ora.step(None)
        return
    ora.compute_membrane_forces(0.0, 0, step)
    if w.force_sigma > 0:
        F = ora.read_forces()
        glob = (np.asarray(ids)[:, None] * nn + np.arange(nn)[None, :]).ravel()
        F += w.force_sigma * orc.noise_normal3_many(w.force_seed, glob, step, 2)
        ora.write_forces(F)
    g = ora.spread()
    ora.step(g)
    ora.interpolate_advance()


def test_config3_full_size_block_and_invariants():
    w = wl.config3()
    assert (w.nx, w.ny, w.nz, w.n_nodes, w.n_edges) == (128, 64, 512, 10272, 30720)
    print("C3 full-size block", full_size_block_parity(w, steps=20, inner=24, mesh_id=5))


def test_config4_full_size_block_and_invariants():
    w = wl.config4()
    assert (w.nx, w.ny, w.nz, w.n_nodes, w.n_edges) == (512, 128, 1024, 657408, 1966080)
    print("C4 full-size block", full_size_block_parity(w, steps=20, inner=32, mesh_id=100))


def test_config5_full_size_block_and_invariants():
    w = wl.config5()
    assert (w.nx, w.ny, w.nz, w.n_nodes, w.n_edges) == (256, 256, 256, 20987904, 62914560)
    print("C5 full-size block", full_size_block_parity(w, steps=6, inner=8, mesh_id=4000))


def record(name, w, out):
    """print the parity maxima; append them to $PLB_RESULTS (a text file) when set"""
    line = "%s %dx%dx%d nodes=%d steps=%d  max|drho|=%.3g  max|dv|/u_ref=%.3g  max|dX|=%s" % (
        name, w.nx, w.ny, w.nz, w.n_nodes, w.steps, out["drho"], out["dv_rel"],
        ("%.3g" % out["dX"]) if "dX" in out else "-")
    print(line)
    path = os.environ.get("PLB_RESULTS")
    if path:
        with open(path, "a") as fh:
            fh.write(line + "\n")


def full_steps(cfg, configured):
    """PLB_FULL_STEPS="4:250,5:25" caps the full-size runs of those configs (the plain oracle spreads
    config 5's 21 M nodes serially, about a minute per step); default = the configured length"""
    for item in os.environ.get("PLB_FULL_STEPS", "").split(","):
        if ":" in item and int(item.split(":")[0]) == cfg:
            return min(configured, int(item.split(":")[1]))
    return configured


@pytest.mark.slow
@pytest.mark.skipif(not FULL, reason="full-length, full-size oracle runs take minutes to an hour of CPU time (PLB_FULL=1)")
@pytest.mark.parametrize("cfg", [3, 5, 4])
def test_config_full_length_full_size(cfg):
    """the whole configured run (C3: 2000 steps, C5: 200, C4: 500) at full size against the fp64
    oracle, at the north_star tolerances (C4 needs ~25 GB of host memory for the oracle)"""
    w = wl.config(cfg)
    w.steps = full_steps(cfg, w.steps)
    record("C%d full" % cfg, w, run_and_compare(w))
