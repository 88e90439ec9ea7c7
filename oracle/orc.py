"""ctypes wrapper around the CPU oracle (oracle/orc.c) -- TEST INFRASTRUCTURE ONLY.

`Oracle(..., fp32=False)` drives one orc_ctx with numpy float64 arrays.  Names follow orc.h.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_libs = {}


class Adhesion(C.Structure):
    """orc_adhesion of orc.h (NEXT-4: PAPER.md section 3.2 / 3.4.1), lattice units, rates per step"""
    _fields_ = [("wall_axis", C.c_int), ("max_per_site", C.c_int), ("k_on0", C.c_double), ("k_off0", C.c_double),
                ("s", C.c_double), ("gamma", C.c_double), ("sigma", C.c_double), ("l_b", C.c_double),
                ("l_max", C.c_double), ("F0", C.c_double), ("tau_rep", C.c_double)]

    @classmethod
    def from_dict(cls, d):
        return cls(int(d.get("wall_axis", 1)), int(d.get("max_per_site", 4)), float(d["k_on0"]), float(d["k_off0"]),
                   float(d["s"]), float(d["gamma"]), float(d["sigma"]), float(d["l_b"]), float(d["l_max"]),
                   float(d.get("F0", 0.0)), float(d.get("tau_rep", 0.0)))


def adhesion_probabilities(prm: dict, x_b: float):
    """(P_f, P_r) of Eq. 12-13 / L151 at bond length x_b"""
    a = Adhesion.from_dict(prm)
    pf, pr = C.c_double(), C.c_double()
    lib().orc_adhesion_probabilities(C.byref(a), float(x_b), C.byref(pf), C.byref(pr))
    return pf.value, pr.value


def lib(fp32: bool = False):
    if fp32 not in _libs:
        _build.build()
        L = C.CDLL(_build.LIB32 if fp32 else _build.LIB64)
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        vp = C.c_void_p
        u64, u32 = C.c_uint64, C.c_uint32
        sig = {
            "orc_lattice": (None, [ip, dp]),
            "orc_real_bytes": (C.c_int, []),
            "orc_phi": (C.c_double, [C.c_double]),
            "orc_feq": (C.c_double, [C.c_int, C.c_double, dp]),
            "orc_philox4x32_10": (None, [C.POINTER(u32), C.POINTER(u32), C.POINTER(u32)]),
            "orc_uniform01": (C.c_double, [u32]),
            "orc_noise_uniform": (None, [u64, u64, u32, u32, dp]),
            "orc_noise_normal3": (None, [u64, u64, u32, u32, dp]),
            "orc_noise_normal3_many": (None, [u64, C.POINTER(u64), C.c_long, u32, u32, dp]),
            "orc_create": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_double, ip, dp, dp, C.POINTER(vp)]),
            "orc_destroy": (C.c_int, [vp]),
            "orc_set_equilibrium": (C.c_int, [vp, dp, dp, C.c_double, u64]),
            "orc_step": (C.c_int, [vp, dp]),
            "orc_read_macros": (C.c_int, [vp, dp, dp]),
            "orc_read_populations": (C.c_int, [vp, dp]),
            "orc_write_populations": (C.c_int, [vp, dp]),
            "orc_add_mesh": (C.c_int, [vp, C.c_int, dp, C.c_int, ip, dp, C.c_double, ip]),
            "orc_compute_membrane_forces": (C.c_int, [vp, C.c_double, u64, u64]),
            "orc_set_triangles": (C.c_int, [vp, C.c_int, C.c_int, ip, dp, C.c_double, C.c_double, C.c_double]),
            "orc_mesh_area_volume": (C.c_int, [vp, C.c_int, dp, dp]),
            "orc_area_volume_energy": (C.c_double, [vp]),
            "orc_spread": (C.c_int, [vp, dp]),
            "orc_interpolate_advance": (C.c_int, [vp]),
            "orc_n_nodes": (C.c_int, [vp]),
            "orc_read_nodes": (C.c_int, [vp, dp]),
            "orc_write_nodes": (C.c_int, [vp, dp]),
            "orc_read_forces": (C.c_int, [vp, dp]),
            "orc_write_forces": (C.c_int, [vp, dp]),
            "orc_read_node_velocities": (C.c_int, [vp, dp]),
            "orc_spring_energy": (C.c_double, [vp]),
            "orc_interpolate_field": (C.c_int, [vp, dp, dp]),
            "orc_set_receptors": (C.c_int, [vp, C.c_int, ip, C.POINTER(Adhesion)]),
            "orc_adhesion_update": (C.c_int, [vp, u64, u64]),
            "orc_read_bonds": (C.c_int, [vp, ip]),
            "orc_write_bonds": (C.c_int, [vp, ip]),
            "orc_adhesion_energy": (C.c_double, [vp]),
            "orc_adhesion_probabilities": (None, [C.POINTER(Adhesion), C.c_double, dp, dp]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _libs[fp32] = L
    return _libs[fp32]


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def lattice():
    c = np.zeros((19, 3), dtype=np.int32)
    w = np.zeros(19, dtype=np.float64)
    lib().orc_lattice(_ip(c), _dp(w))
    return c, w


def phi(r: float) -> float:
    return lib().orc_phi(float(r))


def feq(i0: int, rho: float, v) -> float:
    v = _f64(v)
    return lib().orc_feq(int(i0), float(rho), _dp(v))


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def noise_uniform(seed, index, step, tag):
    out = np.zeros(4)
    lib().orc_noise_uniform(int(seed), int(index), int(step), int(tag), _dp(out))
    return out


def noise_normal3(seed, index, step, tag):
    out = np.zeros(3)
    lib().orc_noise_normal3(int(seed), int(index), int(step), int(tag), _dp(out))
    return out


def noise_normal3_many(seed, index, step, tag):
    """[n, 3] normals of the n counters `index` (orc_noise_normal3 in a loop)"""
    idx = np.ascontiguousarray(index, dtype=np.uint64)
    out = np.zeros((idx.shape[0], 3))
    lib().orc_noise_normal3_many(int(seed), idx.ctypes.data_as(C.POINTER(C.c_uint64)), idx.shape[0], int(step), int(tag), _dp(out))
    return out


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__("%s returned %d" % (what, code))
        self.code = code


class Oracle:
    def __init__(self, nx, ny, nz, tau, kind=(0, 0, 0), u_lo=None, u_hi=None, fp32=False):
        self.L = lib(fp32)
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.cells = self.nx * self.ny * self.nz
        kind = np.ascontiguousarray(kind, dtype=np.int32)
        u_lo = _f64(np.zeros((3, 3)) if u_lo is None else u_lo)
        u_hi = _f64(np.zeros((3, 3)) if u_hi is None else u_hi)
        h = C.c_void_p()
        self._chk(self.L.orc_create(self.nx, self.ny, self.nz, float(tau), _ip(kind), _dp(u_lo), _dp(u_hi),
                                    C.byref(h)), "orc_create")
        self.h = h

    @classmethod
    def from_workload(cls, w, fp32=False):
        o = cls(w.nx, w.ny, w.nz, w.tau, w.kind, w.u_lo, w.u_hi, fp32=fp32)
        o.set_equilibrium(None, w.u0, w.noise_amp, w.noise_seed)
        for m in range(w.n_meshes):
            o.add_mesh(w.mesh_xyz[m], w.edges, w.rest, w.k_spring)
            if w.k_area_global or w.k_area_local or w.k_volume:
                o.set_triangles(m, w.tris, w.ref_xyz, w.k_area_global, w.k_area_local, w.k_volume)
        if getattr(w, "receptor_node", None) is not None:
            o.set_receptors(w.receptor_node, w.adhesion)
            o.adhesion_seed = w.adhesion_seed
        return o

    def _chk(self, rc, what):
        if rc != 0:
            raise OracleError(rc, what)

    def close(self):
        if getattr(self, "h", None):
            self.L.orc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- lattice ----
    def set_equilibrium(self, rho=None, u=None, noise_amp=0.0, seed=0):
        rho, u = _f64(rho), _f64(u)
        self._chk(self.L.orc_set_equilibrium(self.h, _dp(rho), _dp(u), float(noise_amp), int(seed)),
                  "orc_set_equilibrium")

    def step(self, g=None):
        g = _f64(g)
        self._chk(self.L.orc_step(self.h, _dp(g)), "orc_step")

    def read_macros(self):
        rho = np.empty(self.cells)
        u = np.empty((3, self.cells))
        self._chk(self.L.orc_read_macros(self.h, _dp(rho), _dp(u)), "orc_read_macros")
        return rho, u

    def read_populations(self):
        f = np.empty((19, self.cells))
        self._chk(self.L.orc_read_populations(self.h, _dp(f)), "orc_read_populations")
        return f

    def write_populations(self, f):
        f = _f64(f)
        assert f.size == 19 * self.cells
        self._chk(self.L.orc_write_populations(self.h, _dp(f)), "orc_write_populations")

    # ---- meshes ----
    def add_mesh(self, xyz, edges, rest=None, k=0.0):
        xyz = _f64(xyz)
        edges = np.ascontiguousarray(edges, dtype=np.int32)
        rest = _f64(rest)
        mid = C.c_int(-1)
        self._chk(self.L.orc_add_mesh(self.h, xyz.shape[0], _dp(xyz), edges.shape[0], _ip(edges), _dp(rest),
                                      float(k), C.byref(mid)), "orc_add_mesh")
        return mid.value

    def set_triangles(self, mesh_id, tris, ref_xyz=None, k_s=0.0, k_t=0.0, k_v=0.0):
        tris = np.ascontiguousarray(tris, dtype=np.int32)
        ref_xyz = _f64(ref_xyz)
        self._chk(self.L.orc_set_triangles(self.h, int(mesh_id), tris.shape[0], _ip(tris), _dp(ref_xyz),
                                           float(k_s), float(k_t), float(k_v)), "orc_set_triangles")

    def mesh_area_volume(self, mesh_id):
        S, V = C.c_double(), C.c_double()
        self._chk(self.L.orc_mesh_area_volume(self.h, int(mesh_id), C.byref(S), C.byref(V)), "orc_mesh_area_volume")
        return S.value, V.value

    def area_volume_energy(self):
        return self.L.orc_area_volume_energy(self.h)

    @property
    def n_nodes(self):
        return self.L.orc_n_nodes(self.h)

    def compute_membrane_forces(self, sigma=0.0, seed=0, step=0):
        self._chk(self.L.orc_compute_membrane_forces(self.h, float(sigma), int(seed), int(step)),
                  "orc_compute_membrane_forces")

    def spread(self):
        g = np.empty((3, self.cells))
        self._chk(self.L.orc_spread(self.h, _dp(g)), "orc_spread")
        return g

    def interpolate_advance(self):
        self._chk(self.L.orc_interpolate_advance(self.h), "orc_interpolate_advance")

    def interpolate_field(self, w):
        w = _f64(w)
        U = np.empty((self.n_nodes, 3))
        self._chk(self.L.orc_interpolate_field(self.h, _dp(w), _dp(U)), "orc_interpolate_field")
        return U

    def read_nodes(self):
        x = np.empty((self.n_nodes, 3))
        self._chk(self.L.orc_read_nodes(self.h, _dp(x)), "orc_read_nodes")
        return x

    def write_nodes(self, xyz):
        xyz = _f64(xyz)
        assert xyz.shape == (self.n_nodes, 3)
        self._chk(self.L.orc_write_nodes(self.h, _dp(xyz)), "orc_write_nodes")

    def read_forces(self):
        F = np.empty((self.n_nodes, 3))
        self._chk(self.L.orc_read_forces(self.h, _dp(F)), "orc_read_forces")
        return F

    def write_forces(self, F):
        F = _f64(F)
        assert F.shape == (self.n_nodes, 3)
        self._chk(self.L.orc_write_forces(self.h, _dp(F)), "orc_write_forces")

    def read_node_velocities(self):
        U = np.empty((self.n_nodes, 3))
        self._chk(self.L.orc_read_node_velocities(self.h, _dp(U)), "orc_read_node_velocities")
        return U

    def spring_energy(self):
        return self.L.orc_spring_energy(self.h)

    # ---- NEXT-4: adhesion (section 3.2) and wall repulsion (section 3.4.1)
    def set_receptors(self, node, prm: dict):
        node = np.ascontiguousarray(node, dtype=np.int32)
        self.n_rec = node.shape[0]
        self.adhesion_seed = getattr(self, "adhesion_seed", 0)
        a = Adhesion.from_dict(prm)
        self._chk(self.L.orc_set_receptors(self.h, node.shape[0], _ip(node), C.byref(a)), "orc_set_receptors")

    def adhesion_update(self, seed=0, step=0):
        self._chk(self.L.orc_adhesion_update(self.h, int(seed), int(step)), "orc_adhesion_update")

    def read_bonds(self):
        b = np.empty((self.n_rec, 3), dtype=np.int32)
        self._chk(self.L.orc_read_bonds(self.h, _ip(b)), "orc_read_bonds")
        return b

    def write_bonds(self, bonds):
        b = np.ascontiguousarray(bonds, dtype=np.int32)
        assert b.shape == (self.n_rec, 3)
        self._chk(self.L.orc_write_bonds(self.h, _ip(b)), "orc_write_bonds")

    def adhesion_energy(self):
        return self.L.orc_adhesion_energy(self.h)

    def coupled_step(self, sigma=0.0, seed=0, step=0):
        """forces -> spread -> LBM step -> interpolate + advance (Fig. 1)."""
        if self.n_nodes:
            self.compute_membrane_forces(sigma, seed, step)
            g = self.spread()
            self.step(g)
            self.interpolate_advance()
            if getattr(self, "n_rec", 0):          # L276: "Finally, the MC computations are performed"
                self.adhesion_update(self.adhesion_seed, step)
        else:
            self.step(None)
