"""The seeded input generators (input only, no method arithmetic): sizes, determinism, geometry."""
import numpy as np
import pytest

from paper_1312_2234_b200 import workloads as wl


@pytest.mark.parametrize("s", [0, 1, 2, 3])
def test_icosphere_counts_and_topology(s):
    v, t, e = wl.icosphere(s)
    assert v.shape[0] == 10 * 4 ** s + 2 and e.shape[0] == 30 * 4 ** s and t.shape[0] == 20 * 4 ** s
    assert v.shape[0] - e.shape[0] + t.shape[0] == 2                      # Euler characteristic of a sphere
    assert np.allclose(np.linalg.norm(v, axis=1), 1.0, atol=1e-15)
    assert (e[:, 0] < e[:, 1]).all() and len({tuple(x) for x in e.tolist()}) == e.shape[0]
    deg = np.bincount(e.ravel())
    assert (deg == 5).sum() == 12 and set(deg.tolist()) <= {5, 6}


def test_configs_shapes_and_determinism():
    w1 = wl.config1(); w1b = wl.config1()
    assert (w1.nx, w1.ny, w1.nz, w1.steps) == (32, 32, 64, 200) and w1.n_nodes == 162 and w1.n_edges == 480
    assert np.array_equal(w1.mesh_xyz, w1b.mesh_xyz)
    r = np.linalg.norm(w1.mesh_xyz[0] - [16, 16, 32], axis=1)
    assert r.max() <= 4.0 + 1e-12 and r.min() >= 0.95 * 1.0 - 1e-12
    assert wl.edge_lengths(w1.mesh_xyz[0], w1.edges).sum() < w1.rest.sum()   # compressed
    u = w1.u0.reshape(3, 64, 32, 32)
    assert u[0, 5, 31, 7] == pytest.approx(0.05 * 31.5 / 32) and u[0, 0, 0, 0] == pytest.approx(0.05 * 0.5 / 32)
    w2 = wl.config2(n=16, steps=3)
    assert w2.kind == (0, 0, 0) and w2.n_nodes == 0 and np.abs(w2.u0[2]).max() == 0
    w3 = wl.config3()
    assert (w3.nx, w3.ny, w3.nz, w3.steps) == (128, 64, 512, 2000) and w3.n_nodes == 10272 and w3.n_edges == 30720
    y = w3.mesh_xyz[..., 1]
    assert y.min() >= 2.5 and y.max() <= 32.0
    c = w3.mesh_xyz.mean(1)
    d = c[:, None, :] - c[None, :, :]
    d[..., 0] -= 128 * np.round(d[..., 0] / 128); d[..., 2] -= 512 * np.round(d[..., 2] / 512)
    dist = np.sqrt((d ** 2).sum(-1)) + 1e9 * np.eye(16)
    assert dist.min() >= 14.0 - 1e-9


def test_scaled_configs_keep_nodes_inside_channel():
    w4 = wl.config4(nx=64, ny=32, nz=64, n_meshes=4, steps=5)
    assert w4.mesh_xyz[..., 1].min() >= 2.5 and w4.mesh_xyz[..., 1].max() <= 32 - 2.5
    w5 = wl.config5(n=32, grid_xz=8, subdiv=2, steps=5)
    assert w5.n_meshes == 8 * 2 * 8 and w5.force_sigma == 1e-4
    y = w5.mesh_xyz[..., 1]
    assert y.min() >= 2.0 and y.max() <= 22.0
    assert any("infeasible" in n or "cannot hold" in n for n in w5.notes)


def test_random_rotations_are_rotations():
    R = wl.random_rotations(np.random.default_rng(1), 50)
    assert np.allclose(np.einsum("nab,ncb->nac", R, R), np.eye(3)[None], atol=1e-14)
    assert np.allclose(np.linalg.det(R), 1.0, atol=1e-14)
