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
# Block parity at FULL size, from the SEEDED INPUTS ONLY (nothing the oracle consumes comes from
# the CUDA path): the oracle runs the first `steps` coupled steps on a sub-block of the workload
# cut out of the generator's own initial state, and the result is compared on the block's inner
# region.  Why the inner region is exact: one LBM step couples nearest neighbours, a node touches
# cells floor(X)-1 .. floor(X)+2 and moves < 0.1 per step, so after `steps` steps a cell only
# knows about cells / nodes within 3*steps of it.  The block is the inner region plus a halo of
# 3*steps + mesh diameter + 1 on the periodic axes (wall axes are taken whole); every mesh with a
# node within 3*steps of the inner region is included whole and lies inside the block, so the
# block's own periodic wrap never reaches the inner region.
# ---------------------------------------------------------------------------------------------
class Block:
    def __init__(self, w, origin, inner, steps, mesh_diameter):
        self.n = (w.nx, w.ny, w.nz)
        self.kind = tuple(w.kind)
        self.reach = 3 * steps
        halo = self.reach + int(np.ceil(mesh_diameter)) + 1
        self.lo, self.size, self.inner = [], [], []
        for a in range(3):
            if self.kind[a] == 1 or inner + 2 * halo >= self.n[a]:      # wall axis / whole periodic axis: exact
                self.lo.append(0); self.size.append(self.n[a]); self.inner.append((0, self.n[a]))
            else:
                self.lo.append(int(origin[a]) - halo); self.size.append(inner + 2 * halo)
                self.inner.append((halo, halo + inner))

    def whole(self, a):
        return self.size[a] == self.n[a]

    def local(self, X):
        """unwrapped positions [..., 3] -> block coordinates; a mesh is shifted as a whole by the
        periodic image that brings its first node nearest to the block centre"""
        Y = np.array(X, dtype=np.float64, copy=True)
        for a in range(3):
            if not self.whole(a):
                centre = self.lo[a] + 0.5 * self.size[a]
                shift = self.n[a] * np.round((Y[..., :1, a] - centre) / self.n[a])
                Y[..., a] -= shift
                Y[..., a] -= self.lo[a]
        return Y

    def cell_index(self, a):
        return (np.arange(self.lo[a], self.lo[a] + self.size[a]) % self.n[a])

    def take_field(self, t):
        """t: torch tensor or ndarray [C, cells] of the full grid -> numpy [C, bz, by, bx] float64"""
        nx, ny, nz = self.n
        if isinstance(t, np.ndarray):
            v = t.reshape(t.shape[0], nz, ny, nx)
            return v[:, self.cell_index(2)][:, :, self.cell_index(1)][:, :, :, self.cell_index(0)].astype(np.float64)
        import torch
        v = t.view(t.shape[0], nz, ny, nx)
        ix = [torch.as_tensor(self.cell_index(a), device=t.device) for a in range(3)]
        return v.index_select(1, ix[2]).index_select(2, ix[1]).index_select(3, ix[0]).cpu().numpy().astype(np.float64)

    def inner_slices(self):
        (x0, x1), (y0, y1), (z0, z1) = self.inner
        return (slice(None), slice(z0, z1), slice(y0, y1), slice(x0, x1))

    def near_inner(self, Xl, margin):
        """mask over [..., n_nodes] positions (block coordinates) within `margin` of the inner region"""
        m = np.ones(Xl.shape[:-1], dtype=bool)
        for a in range(3):
            if not self.whole(a):
                m &= (Xl[..., a] >= self.inner[a][0] - margin) & (Xl[..., a] <= self.inner[a][1] - 1 + margin)
        return m


def block_workload(w, blk):
    """Sub-workload of w on the block, built from the generator's outputs alone.  Returns
    (Workload, mesh_ids): the meshes with a node within blk.reach of the inner region."""
    import copy
    wb = copy.copy(w)
    wb.nx, wb.ny, wb.nz = blk.size
    wb.u0 = None if w.u0 is None else blk.take_field(w.u0).reshape(3, -1)
    assert w.noise_amp == 0.0, "population noise is keyed on the global cell index"
    ids = np.zeros(0, dtype=np.int64)
    if w.n_meshes:
        Xl = blk.local(w.mesh_xyz)                                   # [meshes, nodes, 3]
        ids = np.nonzero(blk.near_inner(Xl, blk.reach).any(axis=1))[0]
        wb.mesh_xyz = np.ascontiguousarray(Xl[ids]) if len(ids) else None
        for a in range(3):                                           # included meshes lie inside the block
            if len(ids) and not blk.whole(a):
                assert wb.mesh_xyz[..., a].min() >= 1.0 and wb.mesh_xyz[..., a].max() <= blk.size[a] - 2.0
    return wb, ids
