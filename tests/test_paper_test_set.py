"""The regenerated test set of PAPER.md:388-450 (gn_inputs/paper_test_set.py): what the paper fixes about it."""
import os

import numpy as np
import pytest

from gn_inputs import paper_test_set as ts


def _golden():
    out = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_printed_values.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = line[1]
    return out


def test_generator_against_the_values_the_paper_prints():
    g = _golden()
    assert ts.d_min(100.0, 1000, 3) == pytest.approx(float(g["d_min_L100_N1000_D3"]), rel=1e-12)
    assert len(ts.table1()) == int(g["table1_networks"])
    assert list(ts.SIZES) == [int(x) for x in g["table1_sizes"].split(",")]
    assert list(ts._PARAM["lattice"]) == [int(x) for x in g["lattice_neighbours"].split(",")]
    assert list(ts._PARAM["small_world"]) == [float(x) for x in g["small_world_rewiring"].split(",")]
    assert list(ts._PARAM["random"]) == [float(x) for x in g["random_density"].split(",")]


def test_d_min_worked_example():
    """L = 100, N = 1000, D = 3 'implies a minimum distance of 10'."""
    assert ts.d_min(100.0, 1000, 3) == pytest.approx(10.0, rel=1e-12)
    assert ts.d_min(100.0, 100, 2) == pytest.approx(10.0, rel=1e-12)
    assert ts.d_min(100.0, 1000, 2.5) == pytest.approx(100.0 * 1000 ** -0.4)       # fractional dimensions (:423)


def test_table1_is_eighty_networks():
    """PAPER.md:441-450 Table 1: 2 dimensions x 5 sizes x 4 classes x 2 densities."""
    nets = ts.table1()
    assert len(nets) == 80
    combos = {(n.dim, n.n_vertices, n.meta["cls"], n.meta["density"]) for n in nets}
    assert len(combos) == 80
    assert {c[1] for c in combos} == {10, 30, 100, 300, 1000} and {c[0] for c in combos} == {2, 3}


@pytest.mark.parametrize("n,dim", [(100, 2), (300, 3), (1000, 2)])
def test_placement_respects_the_minimum_distance_and_numbering(n, dim):
    net = ts.make_test_network(7, n, dim, "lattice", "low")
    p = net.positions.astype(np.float64)
    d2 = np.sum((p[:, None, :] - p[None, :, :]) ** 2, axis=2)
    d2[np.arange(n), np.arange(n)] = np.inf
    assert np.sqrt(d2.min()) >= net.meta["d_min"] * (1 - 1e-6)                  # rejection loop
    assert (p >= 0).all() and (p <= ts.SPACE).all()
    r = np.sum((p - ts.SPACE / 2) ** 2, axis=1)
    assert (np.diff(r) >= -1e-3).all()                                          # numbered from the centre outwards (:423)


def test_connectivity_classes_have_the_stated_parameters():
    n = 300
    for dens, k in (("low", 3), ("high", 8)):                                   # lattice: 3 / 8 closest neighbours
        net = ts.make_test_network(1, n, 2, "lattice", dens)
        deg = np.diff(net.row_offsets.astype(np.int64))
        assert (deg == k).all()
        p = net.positions.astype(np.float64)
        src = np.repeat(np.arange(n), deg)
        d_edge = np.linalg.norm(p[src] - p[net.targets], axis=1)
        d_all = np.sort(np.linalg.norm(p[:, None] - p[None], axis=2), axis=1)[:, k]      # k-th nearest (0 = self)
        assert (d_edge <= d_all[src] + 1e-9).all()
    for dens, frac in (("low", 0.05), ("high", 0.15)):                          # small world: 5 % / 15 % rewired
        sw = ts.make_test_network(1, n, 2, "small_world", dens)
        lat = ts.make_test_network(1, n, 2, "lattice", "high")
        same_pos = np.array_equal(sw.positions, lat.positions)
        assert sw.n_edges == 8 * n
        if same_pos:
            a = set(zip(np.repeat(np.arange(n), 8).tolist(), lat.targets.tolist()))
            b = set(zip(np.repeat(np.arange(n), 8).tolist(), sw.targets.tolist()))
            assert abs(len(b - a) / (8 * n) - frac) < 0.03
    for dens, dns in (("low", 0.10), ("high", 0.20)):                           # random: 0.1 N^2 / 0.2 N^2 edges
        net = ts.make_test_network(1, n, 3, "random", dens)
        assert net.n_edges == round(dns * n * n)
    for dens, m in (("low", 2), ("high", 4)):                                   # scale free: heavy-tailed degrees
        net = ts.make_test_network(1, 1000, 2, "scale_free", dens)
        deg = np.diff(net.row_offsets.astype(np.int64))
        assert deg.min() >= m and deg.max() > 8 * np.median(deg)
        assert abs(net.n_edges - 2 * m * 1000) < 4 * m * m


def test_batch_is_block_diagonal():
    nets = [ts.make_test_network(3, n, d, "random", "high") for n, d in ((10, 2), (30, 3), (100, 2))]
    b = ts.batch(nets)
    assert b.n_networks == 3 and b.dim == 3 and list(b.net_offsets) == [0, 10, 40, 140]
    assert b.n_edges == sum(x.n_edges for x in nets)
    src = np.repeat(np.arange(b.n_vertices), np.diff(b.row_offsets.astype(np.int64)))
    blk = np.searchsorted(b.net_offsets, src, side="right")
    assert (blk == np.searchsorted(b.net_offsets, b.targets, side="right")).all()
    assert (b.positions[:10, 2] == 0).all()                                     # a 2D network lies in the plane z = 0
