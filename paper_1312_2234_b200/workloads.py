"""Seeded synthetic input generators for the five BASELINE.json configs and
for the two workloads of the widened rows: `flipping_platelet` (NEXT-3, section 4.1) and
`adhering_platelets` (NEXT-4, section 3.2).

This module is INPUT ONLY.  It is the one module the oracle tests and the CUDA path share, and it
holds none of the method's arithmetic: no lattice-Boltzmann update, no delta kernel, no spring
force, no Philox.  It builds meshes (icospheres scaled to oblate ellipsoids, as the platelet shape
of PAPER.md:L81, x^2/a^2 + y^2/a^2 + z^2/(lambda a)^2 = 1), initial macroscopic fields (linear
shear, Taylor-Green) and placements with ``numpy.random.Generator(PCG64(seed))``.

The paper measures on no public dataset; its workload is one or two 958-node platelets in a sheared
channel.  The configs are synthetic stand-ins "shaped like the paper's".

Layout conventions (shared by the oracle and the CUDA library):
  * linear cell index  q = i + nx*(j + ny*k)  (x fastest), lattice node (i,j,k) at the integer point
  * macroscopic fields as SoA: rho[cells], u[3, cells]
  * mesh nodes AoS float64 [n_nodes, 3]; edges int32 [n_edges, 2], mesh-local, (low, high) sorted
"""
from __future__ import annotations

from dataclasses import dataclass, field
import math

import numpy as np

SEED_BASE = 131222340  # seeds are SEED_BASE + config number

PERIODIC = 0
WALL = 1        # halfway bounce-back + moving-wall term (the BASELINE configs)
WALL_HH = 2     # Hecht-Harting on-site velocity wall (the paper's own, Eq. 23-30)


# --------------------------------------------------------------------------------------
# meshes
# --------------------------------------------------------------------------------------
def icosphere(subdiv: int):
    """Unit icosphere: 12-vertex icosahedron, each triangle split in four `subdiv` times, new
    vertices normalised, vertices in creation order, triangles oriented outwards.  Returns (verts[n,3] f64, tris[m,3] i32,
    edges[e,2] i32 sorted unique (low, high)).  n = 10*4^s + 2, e = 30*4^s, m = 20*4^s."""
    t = (1.0 + math.sqrt(5.0)) / 2.0
    verts = [(-1, t, 0), (1, t, 0), (-1, -t, 0), (1, -t, 0),
             (0, -1, t), (0, 1, t), (0, -1, -t), (0, 1, -t),
             (t, 0, -1), (t, 0, 1), (-t, 0, -1), (-t, 0, 1)]
    verts = [np.asarray(v, dtype=np.float64) / math.sqrt(1.0 + t * t) for v in verts]
    tris = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11),
            (1, 5, 9), (5, 11, 4), (11, 10, 2), (10, 7, 6), (7, 1, 8),
            (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9),
            (4, 9, 5), (2, 4, 11), (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    for _ in range(subdiv):
        mid = {}

        def midpoint(a, b):
            key = (a, b) if a < b else (b, a)
            if key not in mid:
                m = verts[a] + verts[b]
                verts.append(m / np.linalg.norm(m))
                mid[key] = len(verts) - 1
            return mid[key]

        new = []
        for a, b, c in tris:
            ab, bc, ca = midpoint(a, b), midpoint(b, c), midpoint(c, a)
            new += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        tris = new
    tris = np.asarray(tris, dtype=np.int32)
    e = np.concatenate([tris[:, [0, 1]], tris[:, [1, 2]], tris[:, [2, 0]]], axis=0)
    e = np.sort(e, axis=1)
    e = np.unique(e, axis=0).astype(np.int32)
    return np.asarray(verts, dtype=np.float64), tris, e


def rot_x(theta: float) -> np.ndarray:
    c, s = math.cos(theta), math.sin(theta)
    return np.array([[1, 0, 0], [0, c, -s], [0, s, c]], dtype=np.float64)


def random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    """n uniform random rotation matrices from normalised Gaussian quaternions.  [n,3,3]"""
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3), dtype=np.float64)
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def edge_lengths(xyz: np.ndarray, edges: np.ndarray) -> np.ndarray:
    d = xyz[edges[:, 1]] - xyz[edges[:, 0]]
    return np.sqrt((d * d).sum(axis=1))


def place_centres(rng, n, lo, hi, min_dist, periodic_len=(None, None, None), max_tries=2_000_000):
    """Rejection sampling of n centres uniform in [lo, hi) with pairwise distance >= min_dist,
    minimum-image on the axes whose periodic_len is not None."""
    lo = np.asarray(lo, dtype=np.float64); hi = np.asarray(hi, dtype=np.float64)
    out = np.empty((n, 3), dtype=np.float64)
    m = 0
    tries = 0
    while m < n:
        tries += 1
        if tries > max_tries:
            raise RuntimeError("placement failed: domain too crowded for min_dist")
        c = lo + (hi - lo) * rng.random(3)
        if m:
            d = out[:m] - c
            for a in range(3):
                L = periodic_len[a]
                if L is not None:
                    d[:, a] -= L * np.round(d[:, a] / L)
            if ((d * d).sum(axis=1) < min_dist * min_dist).any():
                continue
        out[m] = c
        m += 1
    return out


# --------------------------------------------------------------------------------------
# macroscopic initial fields (SoA, x fastest)
# --------------------------------------------------------------------------------------
def shear_field(nx, ny, nz, u_wall):
    """rho = 1, u_x(j) = u_wall (j + 1/2)/ny (the Couette steady state with walls at y = -1/2 and
    ny - 1/2), u_y = u_z = 0.  Returns u[3, cells] float64."""
    u = np.zeros((3, nz, ny, nx), dtype=np.float64)
    j = np.arange(ny, dtype=np.float64)
    u[0] = (u_wall * (j + 0.5) / ny)[None, :, None]
    return u.reshape(3, -1)


def taylor_green_field(nx, ny, nz, u0):
    """2-D Taylor-Green vortex in the x-y plane, uniform in z:
    u_x = -u0 cos(kx x) sin(ky y), u_y = u0 (kx/ky) sin(kx x) cos(ky y) with kx = 2pi/nx, ky = 2pi/ny."""
    kx, ky = 2 * math.pi / nx, 2 * math.pi / ny
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    u = np.zeros((3, nz, ny, nx), dtype=np.float64)
    u[0] = -u0 * np.cos(kx * x) * np.sin(ky * y)
    u[1] = u0 * (kx / ky) * np.sin(kx * x) * np.cos(ky * y)
    return u.reshape(3, -1)


# --------------------------------------------------------------------------------------
# workload description
# --------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    tau: float
    kind: tuple                       # per axis PERIODIC / WALL
    u_lo: np.ndarray                  # [3 axes, 3 comps] wall velocity at the low face of axis a
    u_hi: np.ndarray                  # [3 axes, 3 comps] wall velocity at the high face of axis a
    steps: int
    u0: np.ndarray | None = None      # [3, cells] f64 initial velocity (None = rest); rho0 = 1 always
    noise_amp: float = 0.0            # population noise amplitude (C1)
    noise_seed: int = 0
    mesh_xyz: np.ndarray | None = None  # [n_meshes, n_nodes, 3] f64, unwrapped positions
    edges: np.ndarray | None = None     # [n_edges, 2] i32, mesh-local, shared topology
    rest: np.ndarray | None = None      # [n_edges] f64, shared rest lengths
    k_spring: float = 0.0
    tris: np.ndarray | None = None      # [n_tris, 3] i32, mesh-local, outward oriented (shared topology)
    ref_xyz: np.ndarray | None = None   # [n_nodes, 3] f64 unstressed body-frame shape (defines S_0, S0_tot, V_0)
    k_area_global: float = 0.0        # k_s of Eq. 4 (0 = area / volume constraints off: the BASELINE configs)
    k_area_local: float = 0.0         # k_t of Eq. 4
    k_volume: float = 0.0             # k_v of Eq. 5
    force_sigma: float = 0.0          # per-step Philox normal force noise (C5)
    force_seed: int = 0
    receptor_node: np.ndarray | None = None   # [n_receptors] i32 global node of each receptor (NEXT-4)
    adhesion: dict | None = None      # DAM + wall-repulsion parameters (include/plb.h plb_adhesion), lattice units
    adhesion_seed: int = 0
    shear_rate: float = 0.0           # du_x/dy of the initial flow (flipping workload)
    u_ref: float = 1.0                # velocity scale for the |du| <= 1e-4 u_ref tolerance (u_wall, or u0 for C2)
    notes: list = field(default_factory=list)

    @property
    def cells(self):
        return self.nx * self.ny * self.nz

    @property
    def n_meshes(self):
        return 0 if self.mesh_xyz is None else self.mesh_xyz.shape[0]

    @property
    def n_nodes(self):
        return 0 if self.mesh_xyz is None else self.mesh_xyz.shape[0] * self.mesh_xyz.shape[1]

    @property
    def n_edges(self):
        return 0 if self.mesh_xyz is None else self.mesh_xyz.shape[0] * self.edges.shape[0]


def _walls_y(u_wall):
    u_lo = np.zeros((3, 3)); u_hi = np.zeros((3, 3))
    u_hi[1, 0] = u_wall
    return (PERIODIC, WALL, PERIODIC), u_lo, u_hi


class MeshSet:
    def __init__(self, xyz, edges, rest, tris, ref_xyz):
        self.xyz, self.edges, self.rest, self.tris, self.ref_xyz = xyz, edges, rest, tris, ref_xyz

    def fields(self):
        return dict(mesh_xyz=self.xyz, edges=self.edges, rest=self.rest, tris=self.tris, ref_xyz=self.ref_xyz)


def ellipsoid_meshes(subdiv, semi_axes, rotations, centres, radial_scale=None):
    """Common mesh recipe: unit icosphere -> scale by semi-axes (a, a, c) along
    body (x, y, z) -> rest lengths from this shape -> [optional] multiply each node's radius
    vector by radial_scale[m] -> rotate -> translate.  Returns a MeshSet: xyz[n_meshes,n,3],
    edges, rest lengths, triangles and the unstressed body-frame shape ref_xyz[n,3]."""
    v, tris, e = icosphere(subdiv)
    body = v * np.asarray(semi_axes, dtype=np.float64)[None, :]
    ref = body.copy()
    rest = edge_lengths(body, e)
    if radial_scale is not None:
        body = body * np.asarray(radial_scale, dtype=np.float64)[:, None]
    xyz = np.einsum("mab,nb->mna", np.asarray(rotations, dtype=np.float64), body)
    xyz += np.asarray(centres, dtype=np.float64)[:, None, :]
    return MeshSet(np.ascontiguousarray(xyz), e, rest, tris, ref)


def shear_channel(name, nx, ny, nz, tau, u_wall, n_meshes, subdiv, semi_axes, k_spring, y_range,
                  min_dist, steps, seed, notes=()):
    """C3/C4-shaped workload: walls in y, top wall moving at u_wall along x, n_meshes randomly
    oriented ellipsoids at rejection-sampled centres (minimum image in x and z)."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    kind, u_lo, u_hi = _walls_y(u_wall)
    centres = place_centres(rng, n_meshes, (0.0, y_range[0], 0.0), (float(nx), y_range[1], float(nz)),
                            min_dist, periodic_len=(float(nx), None, float(nz)))
    R = random_rotations(rng, n_meshes)
    ms = ellipsoid_meshes(subdiv, semi_axes, R, centres)
    return Workload(name=name, nx=nx, ny=ny, nz=nz, tau=tau, kind=kind, u_lo=u_lo, u_hi=u_hi, steps=steps,
                    u0=shear_field(nx, ny, nz, u_wall), k_spring=k_spring, u_ref=u_wall, notes=list(notes),
                    **ms.fields())


def config1(nx=32, ny=32, nz=64, steps=200, subdiv=2, seed=SEED_BASE + 1):
    """C1 tiny coupled: one compressed, tilted s=2 ellipsoid (4,4,1) in a 32x32x64 Couette cell."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    kind, u_lo, u_hi = _walls_y(0.05)
    theta = 0.5 * math.pi * rng.random()            # tilt about the world x axis, [0, pi/2)
    n_nodes = 10 * 4 ** subdiv + 2
    xi = rng.random(n_nodes)                         # 5 % seeded radial compression
    ms = ellipsoid_meshes(subdiv, (4.0, 4.0, 1.0), rot_x(theta)[None], [(nx / 2, ny / 2, nz / 2)],
                          radial_scale=1.0 - 0.05 * xi)
    return Workload(name="C1", nx=nx, ny=ny, nz=nz, tau=0.8, kind=kind, u_lo=u_lo, u_hi=u_hi, steps=steps,
                    u0=shear_field(nx, ny, nz, 0.05), noise_amp=1e-4, noise_seed=seed,
                    k_spring=0.01, u_ref=0.05,
                    notes=["tilt = rotation about world x by (pi/2)*xi"], **ms.fields())


def config2(n=256, steps=1000, u0=0.02):
    """C2 pure LBM: fully periodic n^3 box, 2-D Taylor-Green vortex (wavelength n), rho = 1."""
    z = np.zeros((3, 3))
    return Workload(name="C2", nx=n, ny=n, nz=n, tau=0.6, kind=(PERIODIC,) * 3, u_lo=z, u_hi=z.copy(),
                    steps=steps, u0=taylor_green_field(n, n, n, u0), u_ref=u0,
                    notes=["2-D vortex in the x-y plane (decay rate 2 nu k^2 is the 2-D one)"])


def config3(nx=128, ny=64, nz=512, n_meshes=16, steps=2000, subdiv=3, seed=SEED_BASE + 3):
    return shear_channel("C3", nx, ny, nz, 0.7, 0.08, n_meshes, subdiv, (6.0, 6.0, 1.5), 0.02,
                         (8.5, min(26.0, ny / 2 - 6.0)), 14.0, steps, seed,
                         notes=["centre height in [8.5, 26] (lower half, full stencil inside at t=0)"])


def config4(nx=512, ny=128, nz=1024, n_meshes=1024, steps=500, subdiv=3, seed=SEED_BASE + 4):
    return shear_channel("C4", nx, ny, nz, 0.65, 0.05, n_meshes, subdiv, (6.0, 6.0, 1.5), 0.02,
                         (8.5, min(64.0, ny - 8.5)), 14.0, steps, seed,
                         notes=["centre height in [8.5, 64] instead of the config's [4, 64]: with semi-axis 6 "
                                "a centre at y=4 would put nodes outside the channel"])


def config5(n=256, grid_xz=64, layers=2, steps=200, subdiv=4, seed=SEED_BASE + 5):
    """C5 contention stress: grid_xz x layers x grid_xz meshes on a jittered lattice inside the
    bottom 20-cell slab (the config's spacing of 11 is geometrically infeasible)."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    kind, u_lo, u_hi = _walls_y(0.05)
    pitch = n / grid_xz
    p, q, r = np.meshgrid(np.arange(grid_xz), np.arange(layers), np.arange(grid_xz), indexing="ij")
    centres = np.stack([pitch * (p.ravel() + 0.5), 8.0 + 8.0 * q.ravel(), pitch * (r.ravel() + 0.5)], axis=1)
    centres = centres + (rng.random(centres.shape) - 0.5)
    R = random_rotations(rng, centres.shape[0])
    ms = ellipsoid_meshes(subdiv, (5.0, 5.0, 1.25), R, centres)
    return Workload(name="C5", nx=n, ny=n, nz=n, tau=0.7, kind=kind, u_lo=u_lo, u_hi=u_hi, steps=steps,
                    u0=shear_field(n, n, n, 0.05), k_spring=0.02, **ms.fields(),
                    force_sigma=1e-4, force_seed=seed, u_ref=0.05,
                    notes=["centres on a jittered %dx%dx%d lattice (spacing >= 3): the config's minimum centre "
                           "spacing of 11 cannot hold 8192 platelets in a 256x20x256 slab; meshes interpenetrate"
                           % (grid_xz, layers, grid_xz)])


def with_onsite_walls(w: Workload) -> Workload:
    """The same workload closed with the paper's own wall (Hecht-Harting on-site velocity
    condition, walls ON layers 0 and n_y - 1) instead of the configs' halfway bounce-back; the
    initial shear is the matching Couette steady state u_x(j) = u_wall j/(n_y - 1)."""
    import copy
    v = copy.copy(w)
    assert tuple(w.kind) == (PERIODIC, WALL, PERIODIC)
    v.kind = (PERIODIC, WALL_HH, PERIODIC)
    u_wall = float(w.u_hi[1, 0])
    u = np.zeros((3, w.nz, w.ny, w.nx), dtype=np.float64)
    u[0] = (u_wall * np.arange(w.ny, dtype=np.float64) / (w.ny - 1))[None, :, None]
    v.u0 = u.reshape(3, -1)
    v.name = w.name + "-onsite"
    v.notes = list(w.notes) + ["walls: Hecht-Harting on-site velocity condition (PAPER.md Eq. 23-30)"]
    return v


def with_area_volume_constraints(w: Workload, ratio=4.4) -> Workload:
    """The same workload with the paper's area and volume constraints switched on (Eq. 4-5;
    SURVEY.md NEXT-2).  Table 2 gives k_s = k_t = 6000 k_B T/l_0^2 = 4.4e-3 N/m against the spring
    stiffness k = 2 E dx/5 = 1e-3 N/m (L94), i.e. k_s/k = k_t/k = 4.4; k_v (an energy per volume)
    is taken as k_s per lattice spacing."""
    import copy
    v = copy.copy(w)
    assert w.tris is not None
    v.k_area_global = v.k_area_local = ratio * w.k_spring
    v.k_volume = ratio * w.k_spring
    v.name = w.name + "-constrained"
    v.notes = list(w.notes) + ["area / volume constraints on (PAPER.md Eq. 4-5): k_s = k_t = k_v = %.3g" % v.k_volume]
    return v


def rot_z(theta: float) -> np.ndarray:
    c, s = math.cos(theta), math.sin(theta)
    return np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]], dtype=np.float64)


def flipping_platelet(nx=64, ny=200, nz=64, a=5.0, lam=0.25, height=None, u_wall=0.1, tau=1.379, k_spring=0.1,
                      subdiv=3, theta0=0.0, steps=1000, constraints=4.4):
    """SURVEY.md NEXT-3, the paper's validation case (section 4.1, Fig. 5-6): ONE
    stiff platelet, oblate spheroid of major radius `a` cells and aspect ratio `lam` (L81), tau =
    1.379 (L215), flipping in a linear shear flow.
      height=None : far from any wall ("H/a > 20", the Jeffery-orbit case): the two walls move in
                    opposite directions (-u_wall, +u_wall) so the centre, at mid-height, does not
                    drift; shear rate 2 u_wall/ny.
      height=H    : near-wall case (the paper's H = 2.4 a): bottom wall at rest, top wall at u_wall,
                    centre H above the bottom WALL (which lies at y = -1/2); shear rate u_wall/ny.
    The symmetry axis of the disc starts in the shear plane (x-y), `theta0` away from the gradient
    direction y towards the flow direction x.  The membrane is the hot path's springs plus the
    area / volume constraints of NEXT-2 (`constraints` = k_s/k, 0 = off); no seed: nothing is random."""
    kind = (PERIODIC, WALL, PERIODIC)
    u_lo = np.zeros((3, 3)); u_hi = np.zeros((3, 3))
    j = np.arange(ny, dtype=np.float64)
    if height is None:
        u_lo[1, 0], u_hi[1, 0] = -u_wall, u_wall
        prof = u_wall * (2.0 * (j + 0.5) / ny - 1.0)
        centre = (nx / 2.0, (ny - 1) / 2.0, nz / 2.0)
        shear = 2.0 * u_wall / ny
        name = "flip-far"
    else:
        u_hi[1, 0] = u_wall
        prof = u_wall * (j + 0.5) / ny
        centre = (nx / 2.0, height - 0.5, nz / 2.0)
        shear = u_wall / ny
        name = "flip-wall"
    u = np.zeros((3, nz, ny, nx), dtype=np.float64)
    u[0] = prof[None, :, None]
    # body z (the short axis) -> world y, then tilt by theta0 about world z towards +x
    R = rot_z(-theta0) @ rot_x(-0.5 * math.pi)
    ms = ellipsoid_meshes(subdiv, (a, a, lam * a), R[None], [centre])
    w = Workload(name=name, nx=nx, ny=ny, nz=nz, tau=tau, kind=kind, u_lo=u_lo, u_hi=u_hi, steps=steps,
                 u0=u.reshape(3, -1), k_spring=k_spring, u_ref=u_wall,
                 notes=["one platelet a=%g lambda=%g, shear rate %.4g per step, Jeffery period %.0f steps"
                        % (a, lam, shear, 2 * math.pi * (lam + 1.0 / lam) / shear)], shear_rate=shear,
                 **ms.fields())
    if constraints:
        w = with_area_volume_constraints(w, ratio=constraints)
    return w


def adhering_platelets(nx=48, ny=32, nz=48, n_side=1, a=5.0, lam=0.25, gap=0.25, u_wall=0.04, tau=1.0, k_spring=0.05,
                       subdiv=3, receptors_per_platelet=5344, steps=200, seed=SEED_BASE + 14, adhesion=None):
    """SURVEY.md NEXT-4 workload: n_side x n_side platelets lying flat just above the resting bottom
    wall (lowest point `gap` above the wall plane y = -1/2) under a shear flow, each carrying
    `receptors_per_platelet` receptor points (5344 per platelet) assigned to uniformly
    drawn nodes of its mesh.  vWF sites are the lattice points of the wall plane (one per h^2 =
    25 per um^2 at h = 0.2 um, L145/L173).  The DAM parameters sigma, gamma, l_b are not in Table 2;
    the defaults below are synthetic values in lattice units chosen so that bonds form, stretch and
    break within a few hundred steps (capture distance 128 nm = 0.64 h is the paper's, L149)."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    kind, u_lo, u_hi = _walls_y(u_wall)
    c = lam * a
    px, pz = nx / n_side, nz / n_side
    p, r = np.meshgrid(np.arange(n_side), np.arange(n_side), indexing="ij")
    centres = np.stack([px * (p.ravel() + 0.5), np.full(p.size, -0.5 + gap + c), pz * (r.ravel() + 0.5)], axis=1)
    centres[:, [0, 2]] += rng.random((p.size, 2)) - 0.5
    R = np.repeat(rot_x(-0.5 * math.pi)[None], p.size, axis=0)          # body z (short axis) -> world y
    ms = ellipsoid_meshes(subdiv, (a, a, c), R, centres)
    n_nodes = ms.xyz.shape[1]
    rec = (rng.integers(0, n_nodes, size=(p.size, receptors_per_platelet)) + n_nodes * np.arange(p.size)[:, None])
    prm = dict(wall_axis=1, max_per_site=4, k_on0=0.1, k_off0=0.002, s=4.0, gamma=0.2, sigma=0.05, l_b=0.3,
               l_max=0.64, F0=2e-5, tau_rep=4.0)
    if adhesion:
        prm.update(adhesion)
    w = Workload(name="adhesion", nx=nx, ny=ny, nz=nz, tau=tau, kind=kind, u_lo=u_lo, u_hi=u_hi, steps=steps,
                 u0=shear_field(nx, ny, nz, u_wall), k_spring=k_spring, u_ref=u_wall,
                 receptor_node=np.ascontiguousarray(rec.ravel(), dtype=np.int32), adhesion=prm, adhesion_seed=seed,
                 notes=["%d platelets flat on the bottom wall, %d receptors each; DAM parameters synthetic (not in Table 2)"
                        % (p.size, receptors_per_platelet)], **ms.fields())
    return with_area_volume_constraints(w)


def disc_axis(xyz: np.ndarray) -> np.ndarray:
    """Unit symmetry axis of a disc-like node cloud [n,3]: the eigenvector of the smallest
    eigenvalue of the gyration tensor (measurement helper for the flipping workload)."""
    d = xyz - xyz.mean(axis=0)
    w, v = np.linalg.eigh(d.T @ d)
    return v[:, 0]


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def config(n: int, **kw) -> Workload:
    return CONFIGS[n](**kw)


def random_fields(seed, cells, rho_amp=0.02, u_amp=0.03):
    """Seeded smooth-free random rho in 1 +- rho_amp and u in +- u_amp (test input only)."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    rho = 1.0 + rho_amp * (2 * rng.random(cells) - 1)
    u = u_amp * (2 * rng.random((3, cells)) - 1)
    return rho, u
