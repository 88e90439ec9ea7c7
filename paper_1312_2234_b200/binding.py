"""Thin ctypes binding of libplb (include/plb.h): same names as the C-ABI, argument marshalling
only.  Every step of the path runs in the CUDA kernels; there is no CPU fallback -- if libplb.so
is missing or a call fails, a PlbError is raised.

PyTorch is used here only for device memory (workspace, field buffers) and the stream handle.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libplb.so")

PLB_PERIODIC, PLB_WALL_BB, PLB_WALL_HH = 0, 1, 2
PLB_OK, PLB_ERR_ARG, PLB_ERR_WORKSPACE, PLB_ERR_CUDA, PLB_ERR_ORDER, PLB_ERR_NODE_LEFT = 0, -1, -2, -3, -4, -5

# every symbol include/plb.h declares: name -> (restype, argtypes)
_vp, _i, _l, _f = C.c_void_p, C.c_int, C.c_long, C.c_float
_u64, _sz = C.c_ulonglong, C.c_size_t
SYMBOLS = {
    "plb_last_error": (C.c_char_p, []),
    "lbm_workspace_bytes": (_i, [_vp, _l, _l, C.POINTER(_sz)]),
    "lbm_create": (_i, [_vp, _f, _vp, _vp, _sz, _l, _l, _vp, C.POINTER(_vp)]),
    "lbm_destroy": (_i, [_vp]),
    "lbm_set_equilibrium": (_i, [_vp, _vp, _vp, _f, _u64]),
    "lbm_step": (_i, [_vp, _vp]),
    "lbm_read_macros": (_i, [_vp, _vp, _vp]),
    "ib_add_mesh": (_i, [_vp, _i, _vp, _i, _vp, _vp, _f, C.POINTER(_i)]),
    "ib_add_meshes": (_i, [_vp, _i, _i, _vp, _i, _vp, _vp, _f, C.POINTER(_i)]),
    "ib_set_triangles": (_i, [_vp, _i, _i, _i, _vp, _vp, _f, _f, _f]),
    "ib_compute_membrane_forces": (_i, [_vp, _f, _u64, _u64]),
    "ib_spread": (_i, [_vp, _vp]),
    "ib_release_forcing": (_i, [_vp]),
    "ib_set_spread_mode": (_i, [_vp, _i]),
    "ib_get_spread_mode": (_i, [_vp, C.POINTER(_i)]),
    "ib_interpolate_advance": (_i, [_vp]),
    "ib_n_nodes": (_i, [_vp, C.POINTER(_l)]),
    "ib_read_nodes": (_i, [_vp, _vp]),
    "ib_write_nodes": (_i, [_vp, _vp]),
    "ib_read_forces": (_i, [_vp, _vp]),
    "ib_write_forces": (_i, [_vp, _vp]),
    "ib_read_node_velocities": (_i, [_vp, _vp]),
    "lbm_read_populations": (_i, [_vp, _vp]),
    "lbm_write_populations": (_i, [_vp, _vp]),
    "ib_adhesion_workspace_bytes": (_i, [_vp, _i, _l, C.POINTER(_sz)]),
    "ib_set_receptors": (_i, [_vp, _l, _vp, _vp, _vp, _sz]),
    "ib_adhesion_update": (_i, [_vp, _u64, _u64]),
    "ib_n_receptors": (_i, [_vp, C.POINTER(_l)]),
    "ib_read_bonds": (_i, [_vp, _vp]),
    "ib_write_bonds": (_i, [_vp, _vp]),
    "lbm_check_finite": (_i, [_vp, C.POINTER(_l)]),
    "lbm_check_finite_static": (_i, [_vp, _vp]),
    "plb_status": (_i, [_vp]),
    "plb_launch_count": (_i, [_vp, C.POINTER(_l)]),
    "plb_philox4x32_10": (_i, [_vp, _l, _vp, _vp, _vp]),
}


class PlbGrid(C.Structure):
    _fields_ = [("nx", _i), ("ny", _i), ("nz", _i)]


class PlbBoundary(C.Structure):
    _fields_ = [("kind", _i * 3), ("u_lo", (_f * 3) * 3), ("u_hi", (_f * 3) * 3)]


class PlbAdhesion(C.Structure):
    """plb_adhesion of include/plb.h (NEXT-4), lattice units, rates per step"""
    _fields_ = [("wall_axis", _i), ("max_per_site", _i), ("k_on0", _f), ("k_off0", _f), ("s", _f), ("gamma", _f),
                ("sigma", _f), ("l_b", _f), ("l_max", _f), ("F0", _f), ("tau_rep", _f)]

    @classmethod
    def from_dict(cls, d):
        return cls(int(d.get("wall_axis", 1)), int(d.get("max_per_site", 4)), float(d["k_on0"]), float(d["k_off0"]),
                   float(d["s"]), float(d["gamma"]), float(d["sigma"]), float(d["l_b"]), float(d["l_max"]),
                   float(d.get("F0", 0.0)), float(d.get("tau_rep", 0.0)))


class PlbError(RuntimeError):
    def __init__(self, code, what, msg=""):
        super().__init__("%s failed with code %d: %s" % (what, code, msg))
        self.code = code


_lib = None


def lib():
    """Load libplb.so (fails loudly if it has not been built: run `python -m paper_1312_2234_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PlbError(PLB_ERR_CUDA, "load", "libplb.so not built (python -m paper_1312_2234_b200.build); "
                           "there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(rc, what):
    if rc != 0:
        raise PlbError(rc, what, (lib().plb_last_error() or b"").decode())


def _np_ptr(a):
    return None if a is None else a.ctypes.data


def _dev_ptr(t):
    return None if t is None else t.data_ptr()


# ---------------------------------------------------------------------------------------------
# C-ABI calls, one Python function each (same names)
# ---------------------------------------------------------------------------------------------
def lbm_workspace_bytes(nx, ny, nz, max_nodes, max_edges) -> int:
    g = PlbGrid(nx, ny, nz)
    out = _sz(0)
    _check(lib().lbm_workspace_bytes(C.addressof(g), int(max_nodes), int(max_edges), C.byref(out)), "lbm_workspace_bytes")
    return out.value


def make_boundary(kind, u_lo=None, u_hi=None) -> PlbBoundary:
    b = PlbBoundary()
    for a in range(3):
        b.kind[a] = int(kind[a])
        for d in range(3):
            b.u_lo[a][d] = 0.0 if u_lo is None else float(u_lo[a][d])
            b.u_hi[a][d] = 0.0 if u_hi is None else float(u_hi[a][d])
    return b


def lbm_create(nx, ny, nz, tau, boundary: PlbBoundary, workspace, max_nodes, max_edges, stream_handle):
    g = PlbGrid(nx, ny, nz)
    h = _vp()
    _check(lib().lbm_create(C.addressof(g), float(tau), C.addressof(boundary), workspace.data_ptr(),
                            workspace.numel() * workspace.element_size(), int(max_nodes), int(max_edges),
                            stream_handle, C.byref(h)), "lbm_create")
    return h


def lbm_destroy(h):
    _check(lib().lbm_destroy(h), "lbm_destroy")


def lbm_set_equilibrium(h, d_rho=None, d_u=None, noise_amp=0.0, seed=0):
    _check(lib().lbm_set_equilibrium(h, _dev_ptr(d_rho), _dev_ptr(d_u), float(noise_amp), int(seed)), "lbm_set_equilibrium")


def lbm_step(h, d_forcing=None):
    _check(lib().lbm_step(h, _dev_ptr(d_forcing)), "lbm_step")


def lbm_read_macros(h, d_rho=None, d_u=None):
    _check(lib().lbm_read_macros(h, _dev_ptr(d_rho), _dev_ptr(d_u)), "lbm_read_macros")


def lbm_read_populations(h, d_f):
    _check(lib().lbm_read_populations(h, _dev_ptr(d_f)), "lbm_read_populations")


def lbm_write_populations(h, d_f):
    _check(lib().lbm_write_populations(h, _dev_ptr(d_f)), "lbm_write_populations")


def ib_add_mesh(h, xyz, edges, rest=None, k=0.0) -> int:
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    edges = np.ascontiguousarray(edges, dtype=np.int32).reshape(-1, 2)
    rest = None if rest is None else np.ascontiguousarray(rest, dtype=np.float32)
    mid = _i(-1)
    _check(lib().ib_add_mesh(h, xyz.shape[0], _np_ptr(xyz), edges.shape[0], _np_ptr(edges), _np_ptr(rest), float(k),
                             C.byref(mid)), "ib_add_mesh")
    return mid.value


def ib_add_meshes(h, xyz, edges, rest=None, k=0.0) -> int:
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    assert xyz.ndim == 3 and xyz.shape[2] == 3
    edges = np.ascontiguousarray(edges, dtype=np.int32).reshape(-1, 2)
    rest = None if rest is None else np.ascontiguousarray(rest, dtype=np.float32)
    mid = _i(-1)
    _check(lib().ib_add_meshes(h, xyz.shape[0], xyz.shape[1], _np_ptr(xyz), edges.shape[0], _np_ptr(edges),
                               _np_ptr(rest), float(k), C.byref(mid)), "ib_add_meshes")
    return mid.value


def ib_set_triangles(h, first_mesh_id, n_meshes, tris, ref_xyz=None, k_s=0.0, k_t=0.0, k_v=0.0):
    tris = np.ascontiguousarray(tris, dtype=np.int32)
    ref_xyz = None if ref_xyz is None else np.ascontiguousarray(ref_xyz, dtype=np.float64)
    _check(lib().ib_set_triangles(h, int(first_mesh_id), int(n_meshes), tris.shape[0], _np_ptr(tris), _np_ptr(ref_xyz),
                                  float(k_s), float(k_t), float(k_v)), "ib_set_triangles")


def ib_compute_membrane_forces(h, noise_sigma=0.0, noise_seed=0, step=0):
    _check(lib().ib_compute_membrane_forces(h, float(noise_sigma), int(noise_seed), int(step)), "ib_compute_membrane_forces")


def ib_spread(h, d_forcing):
    _check(lib().ib_spread(h, _dev_ptr(d_forcing)), "ib_spread")


PLB_SPREAD_AUTO, PLB_SPREAD_SCATTER, PLB_SPREAD_AGGREGATE, PLB_SPREAD_GATHER = 0, 1, 2, 3
SPREAD_MODES = {"auto": 0, "scatter": 1, "aggregate": 2, "gather": 3}


def ib_release_forcing(h):
    _check(lib().ib_release_forcing(h), "ib_release_forcing")


def ib_set_spread_mode(h, mode):
    _check(lib().ib_set_spread_mode(h, int(SPREAD_MODES.get(mode, mode))), "ib_set_spread_mode")


def ib_get_spread_mode(h) -> int:
    out = _i(0)
    _check(lib().ib_get_spread_mode(h, C.byref(out)), "ib_get_spread_mode")
    return out.value


def ib_interpolate_advance(h):
    _check(lib().ib_interpolate_advance(h), "ib_interpolate_advance")


def ib_n_nodes(h) -> int:
    out = _l(0)
    _check(lib().ib_n_nodes(h, C.byref(out)), "ib_n_nodes")
    return out.value


def ib_read_nodes(h, out=None):
    n = ib_n_nodes(h)
    out = np.empty((n, 3), dtype=np.float64) if out is None else out
    _check(lib().ib_read_nodes(h, _np_ptr(out)), "ib_read_nodes")
    return out


def ib_write_nodes(h, xyz):
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    assert xyz.shape == (ib_n_nodes(h), 3)
    _check(lib().ib_write_nodes(h, _np_ptr(xyz)), "ib_write_nodes")


def ib_read_forces(h):
    out = np.empty((ib_n_nodes(h), 3), dtype=np.float32)
    _check(lib().ib_read_forces(h, _np_ptr(out)), "ib_read_forces")
    return out


def ib_write_forces(h, F):
    F = np.ascontiguousarray(F, dtype=np.float32)
    assert F.shape == (ib_n_nodes(h), 3)
    _check(lib().ib_write_forces(h, _np_ptr(F)), "ib_write_forces")


def ib_read_node_velocities(h):
    out = np.empty((ib_n_nodes(h), 3), dtype=np.float32)
    _check(lib().ib_read_node_velocities(h, _np_ptr(out)), "ib_read_node_velocities")
    return out


def ib_adhesion_workspace_bytes(nx, ny, nz, wall_axis, n_receptors) -> int:
    g = PlbGrid(nx, ny, nz)
    out = _sz(0)
    _check(lib().ib_adhesion_workspace_bytes(C.addressof(g), int(wall_axis), int(n_receptors), C.byref(out)),
           "ib_adhesion_workspace_bytes")
    return out.value


def ib_set_receptors(h, node, prm: dict, workspace):
    node = np.ascontiguousarray(node, dtype=np.int32)
    a = PlbAdhesion.from_dict(prm)
    _check(lib().ib_set_receptors(h, node.shape[0], _np_ptr(node), C.addressof(a), workspace.data_ptr(),
                                  workspace.numel() * workspace.element_size()), "ib_set_receptors")


def ib_adhesion_update(h, seed=0, step=0):
    _check(lib().ib_adhesion_update(h, int(seed), int(step)), "ib_adhesion_update")


def ib_n_receptors(h) -> int:
    out = _l(0)
    _check(lib().ib_n_receptors(h, C.byref(out)), "ib_n_receptors")
    return out.value


def ib_read_bonds(h):
    out = np.empty((ib_n_receptors(h), 3), dtype=np.int32)
    _check(lib().ib_read_bonds(h, _np_ptr(out)), "ib_read_bonds")
    return out


def ib_write_bonds(h, bonds):
    b = np.ascontiguousarray(bonds, dtype=np.int32)
    assert b.shape == (ib_n_receptors(h), 3)
    _check(lib().ib_write_bonds(h, _np_ptr(b)), "ib_write_bonds")


def lbm_check_finite(h) -> int:
    out = _l(0)
    _check(lib().lbm_check_finite(h, C.byref(out)), "lbm_check_finite")
    return out.value


def lbm_check_finite_static(h, d_out):
    """d_out: a device int32 tensor of one element (written asynchronously on the context's stream)"""
    _check(lib().lbm_check_finite_static(h, None if d_out is None else d_out.data_ptr()), "lbm_check_finite_static")


def plb_status(h):
    _check(lib().plb_status(h), "plb_status")


def plb_launch_count(h) -> int:
    out = _l(0)
    _check(lib().plb_launch_count(h, C.byref(out)), "plb_launch_count")
    return out.value


def plb_philox4x32_10(d_ctr, d_key, d_out, stream_handle=None):
    _check(lib().plb_philox4x32_10(stream_handle, d_ctr.numel() // 4, _dev_ptr(d_ctr), _dev_ptr(d_key), _dev_ptr(d_out)),
           "plb_philox4x32_10")


# ---------------------------------------------------------------------------------------------
# Convenience holder: owns the torch buffers (workspace, forcing) a context needs.  Marshalling
# only: each method is one C-ABI call.
# ---------------------------------------------------------------------------------------------
class Simulation:
    def __init__(self, nx, ny, nz, tau, kind=(0, 0, 0), u_lo=None, u_hi=None, max_nodes=0, max_edges=0, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise PlbError(PLB_ERR_CUDA, "Simulation", "no CUDA device; this library has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.cells = self.nx * self.ny * self.nz
        nbytes = lbm_workspace_bytes(nx, ny, nz, max_nodes, max_edges)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.forcing = torch.zeros(self.cells * 4, dtype=torch.float32, device=self.device)  # float4 per cell
        self.stream = torch.cuda.current_stream(self.device)
        self.boundary = make_boundary(kind, u_lo, u_hi)
        self.h = lbm_create(nx, ny, nz, tau, self.boundary, self.workspace, max_nodes, max_edges, self.stream.cuda_stream)

    @classmethod
    def from_workload(cls, w, device="cuda:0"):
        import torch
        s = cls(w.nx, w.ny, w.nz, w.tau, w.kind, w.u_lo, w.u_hi, max_nodes=w.n_nodes, max_edges=w.n_edges, device=device)
        u = None if w.u0 is None else torch.as_tensor(w.u0, dtype=torch.float32).to(s.device).contiguous()
        s.set_equilibrium(None, u, w.noise_amp, w.noise_seed)
        if w.n_meshes:
            first = s.add_meshes(w.mesh_xyz, w.edges, w.rest, w.k_spring)
            if w.k_area_global or w.k_area_local or w.k_volume:
                s.set_triangles(first, w.n_meshes, w.tris, w.ref_xyz, w.k_area_global, w.k_area_local, w.k_volume)
        if getattr(w, "receptor_node", None) is not None:
            s.set_receptors(w.receptor_node, w.adhesion)
            s.adhesion_seed = w.adhesion_seed
        return s

    def close(self):
        if getattr(self, "h", None):
            lbm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_equilibrium(self, d_rho=None, d_u=None, noise_amp=0.0, seed=0):
        lbm_set_equilibrium(self.h, d_rho, d_u, noise_amp, seed)

    def step(self, d_forcing=None):
        lbm_step(self.h, d_forcing)

    def read_macros(self):
        rho = self.torch.empty(self.cells, dtype=self.torch.float32, device=self.device)
        u = self.torch.empty(3 * self.cells, dtype=self.torch.float32, device=self.device)
        lbm_read_macros(self.h, rho, u)
        return rho, u.view(3, self.cells)

    def check_finite(self) -> int:
        return lbm_check_finite(self.h)

    def read_populations(self):
        f = self.torch.empty(19 * self.cells, dtype=self.torch.float32, device=self.device)
        lbm_read_populations(self.h, f)
        return f.view(19, self.cells)

    def write_populations(self, d_f):
        lbm_write_populations(self.h, d_f.contiguous())

    def add_mesh(self, xyz, edges, rest=None, k=0.0):
        return ib_add_mesh(self.h, xyz, edges, rest, k)

    def add_meshes(self, xyz, edges, rest=None, k=0.0):
        return ib_add_meshes(self.h, xyz, edges, rest, k)

    def set_triangles(self, first_mesh_id, n_meshes, tris, ref_xyz=None, k_s=0.0, k_t=0.0, k_v=0.0):
        ib_set_triangles(self.h, first_mesh_id, n_meshes, tris, ref_xyz, k_s, k_t, k_v)

    def compute_membrane_forces(self, sigma=0.0, seed=0, step=0):
        ib_compute_membrane_forces(self.h, sigma, seed, step)

    def set_receptors(self, node, prm: dict):
        node = np.ascontiguousarray(node, dtype=np.int32)
        nbytes = ib_adhesion_workspace_bytes(self.nx, self.ny, self.nz, int(prm.get("wall_axis", 1)), node.shape[0])
        self.adhesion_workspace = self.torch.empty(nbytes, dtype=self.torch.uint8, device=self.device)
        ib_set_receptors(self.h, node, prm, self.adhesion_workspace)
        self.n_rec = node.shape[0]
        self.adhesion_seed = getattr(self, "adhesion_seed", 0)

    def adhesion_update(self, seed=0, step=0):
        ib_adhesion_update(self.h, seed, step)

    def read_bonds(self):
        return ib_read_bonds(self.h)

    def write_bonds(self, bonds):
        ib_write_bonds(self.h, bonds)

    def spread(self, d_forcing=None):
        ib_spread(self.h, self.forcing if d_forcing is None else d_forcing)

    def set_spread_mode(self, mode):
        ib_set_spread_mode(self.h, mode)

    def spread_mode(self) -> int:
        return ib_get_spread_mode(self.h)

    def interpolate_advance(self):
        ib_interpolate_advance(self.h)

    def coupled_step(self, sigma=0.0, seed=0, step=0):
        """The four calls of one coupled step, in the paper's order (L75, L276, Fig. 1)."""
        ib_compute_membrane_forces(self.h, sigma, seed, step)
        ib_spread(self.h, self.forcing)
        lbm_step(self.h, self.forcing)
        ib_interpolate_advance(self.h)
        if getattr(self, "n_rec", 0):               # L276: "Finally, the MC computations are performed"
            ib_adhesion_update(self.h, self.adhesion_seed, step)

    @property
    def n_nodes(self):
        return ib_n_nodes(self.h)

    def read_nodes(self, out=None):
        return ib_read_nodes(self.h, out)

    def write_nodes(self, xyz):
        ib_write_nodes(self.h, xyz)

    def read_forces(self):
        return ib_read_forces(self.h)

    def write_forces(self, F):
        ib_write_forces(self.h, F)

    def read_node_velocities(self):
        return ib_read_node_velocities(self.h)

    def status(self):
        plb_status(self.h)

    def launch_count(self):
        return plb_launch_count(self.h)
