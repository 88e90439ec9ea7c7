"""Helpers for the GPU-vs-oracle parity tests: build both sides from one Workload, run them in
lock-step through the same calls, compare element by element."""
from __future__ import annotations

import numpy as np

from oracle import orc
from paper_1312_2234_b200 import binding as plb

# north_star tolerances (BASELINE.json): |dv| <= 1e-4 u_ref, |drho| <= 1e-6, |dX| <= 1e-4
TOL_V_REL, TOL_RHO, TOL_X = 1e-4, 1e-6, 1e-4


def forcing_to_soa(sim):
    """float4-per-cell device forcing -> numpy [3, cells] float64"""
    return sim.forcing.view(sim.cells, 4)[:, :3].t().contiguous().cpu().numpy().astype(np.float64)


def soa_to_forcing(sim, g):
    import torch
    t = torch.zeros(sim.cells, 4, dtype=torch.float32, device=sim.device)
    t[:, :3] = torch.as_tensor(np.ascontiguousarray(g.T), dtype=torch.float32, device=sim.device)
    return t.view(-1)


def build_pair(w, fp32_oracle=False):
    sim = plb.Simulation.from_workload(w)
    ora = orc.Oracle.from_workload(w, fp32=fp32_oracle)
    return sim, ora


def run_pair(w, sim, ora, steps):
    for s in range(steps):
        if w.n_meshes:
            sim.coupled_step(w.force_sigma, w.force_seed, s)
            ora.coupled_step(w.force_sigma, w.force_seed, s)
        else:
            sim.step(None)
            ora.step(None)
    sim.status()


def compare(w, sim, ora, check=True):
    rho_g, u_g = sim.read_macros()
    rho_g = rho_g.cpu().numpy().astype(np.float64)
    u_g = u_g.cpu().numpy().astype(np.float64)
    rho_o, u_o = ora.read_macros()
    out = {
        "drho": float(np.abs(rho_g - rho_o).max()),
        "dv": float(np.abs(u_g - u_o).max()),
        "dv_rel": float(np.abs(u_g - u_o).max() / w.u_ref),
    }
    if w.n_meshes:
        out["dX"] = float(np.abs(sim.read_nodes() - ora.read_nodes()).max())
    if check:
        assert np.isfinite(rho_g).all() and np.isfinite(u_g).all()
        assert out["drho"] <= TOL_RHO, out
        assert out["dv_rel"] <= TOL_V_REL, out
        if w.n_meshes:
            assert out["dX"] <= TOL_X, out
    return out


# ---------------------------------------------------------------------------------------------
# Block parity at FULL size: one coupled step of a sub-block of the lattice is recomputed by the
# oracle from the GPU's own pre-step state and compared on the block interior.  One LBM step only
# couples nearest neighbours and a node only touches floor(X)-1 .. floor(X)+2, so with a halo of
# H >= 4 cells on the periodic axes the interior of the block is exact; wall axes are taken whole.
# ---------------------------------------------------------------------------------------------
class BlockSpec:
    def __init__(self, w, origin, width, halo=4):
        self.n = (w.nx, w.ny, w.nz)
        self.kind = tuple(w.kind)
        self.lo, self.size, self.inner = [], [], []
        for a in range(3):
            if self.kind[a] == 1:                       # wall axis: whole extent
                self.lo.append(0); self.size.append(self.n[a]); self.inner.append((0, self.n[a]))
            else:
                bw = min(width, self.n[a])
                if bw == self.n[a]:                     # the block wraps onto itself: exact everywhere
                    self.lo.append(0); self.size.append(bw); self.inner.append((0, bw))
                else:
                    self.lo.append(int(origin[a]) % self.n[a]); self.size.append(bw); self.inner.append((halo, bw - halo))

    def index(self, a, device=None):
        import torch
        return (torch.arange(self.lo[a], self.lo[a] + self.size[a], device=device) % self.n[a])

    def take(self, t):
        """t: device tensor [C, nz, ny, nx] -> numpy [C, bz, by, bx] float64"""
        ix, iy, iz = (self.index(a, t.device) for a in range(3))
        return t.index_select(3, ix).index_select(2, iy).index_select(1, iz).cpu().numpy().astype(np.float64)

    def inner_slices(self):
        (x0, x1), (y0, y1), (z0, z1) = self.inner
        return (slice(None), slice(z0, z1), slice(y0, y1), slice(x0, x1))

    def local_positions(self, X):
        """Unwrapped positions -> block coordinates (nearest periodic image to the block centre)."""
        Y = np.array(X, dtype=np.float64, copy=True)
        for a in range(3):
            if self.kind[a] == 0:
                centre = self.lo[a] + 0.5 * self.size[a]
                Y[:, a] -= self.n[a] * np.round((Y[:, a] - centre) / self.n[a])
            Y[:, a] -= self.lo[a]
        return Y

    def nodes_near(self, Xl, margin=2.5):
        m = np.ones(Xl.shape[0], dtype=bool)
        for a in range(3):
            if self.kind[a] == 0 and self.size[a] < self.n[a]:
                m &= (Xl[:, a] > -margin) & (Xl[:, a] < self.size[a] + margin)
        return m

    def nodes_clean(self, Xl):
        """nodes whose whole 4^3 stencil lies inside the clean interior"""
        m = np.ones(Xl.shape[0], dtype=bool)
        for a in range(3):
            if self.kind[a] == 0 and self.size[a] < self.n[a]:
                fl = np.floor(Xl[:, a])
                m &= (fl - 1 >= self.inner[a][0]) & (fl + 2 < self.inner[a][1])
        return m


def block_oracle_step(w, blk, f_before, g_dev, X_before, F_nodes):
    """Recompute one coupled step on the block with the oracle.  f_before: [19, bz, by, bx] true
    populations; returns dict with the oracle's g, f_after, U, X_after (block-local) and masks."""
    bx, by, bz = blk.size
    ora = orc.Oracle(bx, by, bz, w.tau, w.kind, w.u_lo, w.u_hi)
    ora.write_populations(f_before.reshape(19, -1))
    res = {}
    if X_before is not None and X_before.shape[0]:
        Xl = blk.local_positions(X_before)
        near = blk.nodes_near(Xl)
        ora.add_mesh(Xl[near], np.zeros((0, 2), dtype=np.int32), None, 0.0)
        ora.write_forces(F_nodes[near].astype(np.float64))
        g = ora.spread()
        ora.step(g)
        ora.interpolate_advance_safe = None
        try:
            ora.interpolate_advance()
        except orc.OracleError as e:          # nodes outside the block may "leave" its walls; ignored
            if e.code != -5:
                raise
        res.update(g=g.reshape(3, bz, by, bx), near=near, clean=blk.nodes_clean(Xl[near]),
                   U=ora.read_node_velocities(), X_after=ora.read_nodes(), Xl=Xl[near])
    else:
        g = None if g_dev is None else g_dev
        ora.step(g)
    res["f_after"] = ora.read_populations().reshape(19, bz, by, bx)
    rho, u = ora.read_macros()
    res["rho"] = rho.reshape(1, bz, by, bx)
    res["u"] = u.reshape(3, bz, by, bx)
    return res
