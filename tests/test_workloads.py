"""Seeded input generators: reproducible, correctly shaped, pack/unpack round trip. CPU only."""
import numpy as np

from workloads import make_config


def test_config_shapes_and_reproducibility():
    a = make_config(3, n_cells=44)
    b = make_config(3, n_cells=44)
    assert a.n_cells == 44 and [ct.n_vertices for ct in a.types] == [642, 162]
    assert int(np.sum(a.type_of_cell == 1)) == 4                      # every 11th cell a platelet
    for t in range(2):
        assert np.array_equal(a.positions[t], b.positions[t])
        assert np.array_equal(a.forces(3)[t], b.forces(3)[t])
        assert not np.array_equal(a.forces(3)[t], a.forces(4)[t])     # noise redrawn every step
        assert np.array_equal(a.forces(3)[t], a.forces(3)[t])
    # shear term: mean x-force follows gamma * z
    f = a.forces(0)[0]
    z = a.positions[0][..., 2] - 0.5 * a.box[2]
    slope = np.sum(f[..., 0] * z) / np.sum(z * z)
    assert abs(slope - 0.02) < 2e-3


def test_prefix_property_and_subset():
    big = make_config(4, n_cells=60)
    small = make_config(4, n_cells=30)
    # bucket prefixes agree: a shrunken config is a prefix of the full one, per type
    for t in range(2):
        k = small.positions[t].shape[0]
        assert np.array_equal(big.positions[t][:k], small.positions[t])
    ids = np.array([3, 9, 19, 42])
    sub = big.subset(ids)
    assert sub.n_cells == 4 and list(sub.type_of_cell) == [0, 1, 1, 0]
    flat = big.packed(big.positions, ids)
    per_type = big.unpack(flat, ids)
    for t in range(2):
        assert np.array_equal(per_type[t], sub.positions[t])
        assert np.array_equal(sub.forces(0)[t].shape, sub.positions[t].shape)


def test_pack_unpack_round_trip_all_cells():
    pop = make_config(3, n_cells=23)
    flat = pop.packed(pop.positions)
    assert flat.shape[0] == 3 * int(pop.vertex_counts().sum())
    back = pop.unpack(flat)
    for t in range(2):
        assert np.array_equal(back[t], pop.positions[t])
    # cell 10 is the first platelet: its block sits after ten RBC blocks, in [n][3] order
    off = 10 * 642 * 3
    assert np.array_equal(flat[off:off + 162 * 3].reshape(162, 3), pop.positions[1][0])


def test_rigid_placement_preserves_shape():
    pop = make_config(2, n_cells=5)
    rest = pop.types[0].rest_positions
    d_rest = np.linalg.norm(rest[1:] - rest[:-1], axis=1)
    for c in range(5):
        x = pop.positions[0][c]
        assert np.allclose(np.linalg.norm(x[1:] - x[:-1], axis=1), d_rest, rtol=1e-12)
    assert np.all(pop.positions[0].mean(axis=1) >= -1e-9)


def test_octahedral_meshes_of_the_paper():
    """RBC 258 / platelet 66 surface vertices = octahedron subdivided 3 / 2 times."""
    import numpy as np
    from workloads import make_config, octasphere
    for level, n in ((2, 66), (3, 258)):
        v, f = octasphere(level)
        assert v.shape == (n, 3) and f.shape == (8 * 4 ** level, 3)
        assert np.allclose(np.linalg.norm(v, axis=1), 1.0)
        val = np.bincount(f.ravel())
        assert sorted(set(val)) == [4, 6] and np.sum(val == 4) == 6
        # closed and consistently oriented: every directed edge once, its twin present
        edges = {(a, b) for t in f for a, b in ((t[0], t[1]), (t[1], t[2]), (t[2], t[0]))}
        assert len(edges) == 3 * len(f) and all((b, a) in edges for a, b in edges)
        nrm = np.cross(v[f[:, 1]] - v[f[:, 0]], v[f[:, 2]] - v[f[:, 0]])
        assert np.all(np.sum(nrm * (v[f[:, 0]] + v[f[:, 1]] + v[f[:, 2]]), axis=1) > 0)      # outward
    pop = make_config(6)
    assert pop.n_cells == 114 and int(np.sum(pop.type_of_cell == 1)) == 19
