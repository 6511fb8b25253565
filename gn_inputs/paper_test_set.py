"""The paper's standardized test set (section 3.5, Table 1), regenerated: INPUTS ONLY.

The authors' 80 network files are on their website and not in this container, so this module rebuilds the recipe the
paper states: vertices placed at random with a minimum-distance constraint (the rejection loop of PAPER.md:398-415,
d_min proportional to L N^(-1/D)), numbered from the centre outwards (:423), and connected by one of
four classes at two densities each (:427-433): lattice (3 / 8 nearest neighbours), small world (the lattice with 5 % /
15 % of the edges rewired at random), scale free (preferential attachment, m = 2 / 4 edges per new vertex) and random
(0.1 N^2 / 0.2 N^2 edges).  Sizes N = 10, 30, 100, 300, 1000 in 2 and 3 dimensions: 2 x 5 x 4 x 2 = 80 networks (:441-450).

Where the paper leaves a number open the reading is stated at the function that takes it (and in DESIGN.md):
the fraction of the cubic-packing distance used as d_min, the base lattice of the small-world class, the attachment
rule of the scale-free class, edge direction, weights.  Randomness is numpy's PCG64 seeded per network from the master
seed; nothing here computes a delay, quantises a weight or steps a vertex.
"""
from __future__ import annotations

import numpy as np

from .generate import Network

SIZES = (10, 30, 100, 300, 1000)
DIMS = (2, 3)
CLASSES = ("lattice", "small_world", "scale_free", "random")
DENSITIES = ("low", "high")
_PARAM = {"lattice": (3, 8), "small_world": (0.05, 0.15), "scale_free": (2, 4), "random": (0.10, 0.20)}
SPACE = 100.0          # side L of the square / cube ("non-dimensional and can be scaled")
SMALL_WORLD_K = 8      # reading: the small-world class rewires the 8-nearest-neighbour lattice


def d_min(L: float, n: int, dim: float, fraction: float = 1.0) -> float:
    """d_min proportional to L N^(-1/D); fraction = 1 is the cubic-packing distance the paper's
    worked example prints (L = 100, N = 1000, D = 3 gives 10); random placement needs a smaller fraction."""
    return fraction * L * float(n) ** (-1.0 / dim)


def place_min_distance(rng: np.random.Generator, n: int, dim: int, L: float, d: float) -> np.ndarray:
    """The paper's rejection loop verbatim: draw a uniform position, accept it iff it is at least d
    from every vertex accepted so far.  Returned in acceptance order."""
    pos = np.empty((n, dim), dtype=np.float64)
    i = 0
    while i < n:
        x = rng.uniform(0.0, L, size=dim)
        if i == 0 or np.min(np.sum((pos[:i] - x) ** 2, axis=1)) >= d * d:
            pos[i] = x
            i += 1
    return pos


def centre_outwards(pos: np.ndarray, L: float) -> np.ndarray:
    """vertices are numbered from the centre outwards."""
    order = np.argsort(np.sum((pos - L / 2.0) ** 2, axis=1), kind="stable")
    return pos[order]


def _nearest(pos: np.ndarray, k: int) -> np.ndarray:
    """[n][k] indices of every vertex's k nearest other vertices (ties by index)."""
    n = len(pos)
    d2 = np.sum((pos[:, None, :] - pos[None, :, :]) ** 2, axis=2)
    d2[np.arange(n), np.arange(n)] = np.inf
    return np.argsort(d2, axis=1, kind="stable")[:, :min(k, n - 1)]


def lattice_edges(pos: np.ndarray, k: int) -> np.ndarray:
    """every vertex connects to its k closest neighbours (directed i -> neighbour)."""
    nb = _nearest(pos, k)
    src = np.repeat(np.arange(len(pos)), nb.shape[1])
    return np.stack([src, nb.ravel()], axis=1)


def small_world_edges(rng: np.random.Generator, pos: np.ndarray, p: float, k: int = SMALL_WORLD_K) -> np.ndarray:
    """a lattice in which each edge is, with probability p, re-wired to a random target (Watts-Strogatz
    on the k-nearest-neighbour lattice; no self-edges, no duplicate edges)."""
    e = lattice_edges(pos, k)
    n = len(pos)
    have = set(map(tuple, e.tolist()))
    for idx in np.nonzero(rng.random(len(e)) < p)[0]:
        i = int(e[idx, 0])
        for _ in range(64):
            j = int(rng.integers(0, n))
            if j != i and (i, j) not in have:
                have.discard((i, int(e[idx, 1])))
                have.add((i, j))
                e[idx, 1] = j
                break
    return e


def scale_free_edges(rng: np.random.Generator, n: int, m: int) -> np.ndarray:
    """power-law degree distribution.  Reading: preferential attachment in the centre-outwards vertex
    order -- vertex v (v >= m) sends m edges to distinct earlier vertices chosen with probability proportional to
    degree + 1; each connection is reciprocal (two directed edges), the first m vertices form a clique."""
    m = min(m, n - 1)
    deg = np.zeros(n, dtype=np.float64)
    pairs = []
    for a in range(m):
        for b in range(a):
            pairs.append((a, b))
            deg[a] += 1
            deg[b] += 1
    for v in range(max(m, 1), n):
        w = deg[:v] + 1.0
        tg = rng.choice(v, size=min(m, v), replace=False, p=w / w.sum())
        for t in tg:
            pairs.append((v, int(t)))
            deg[v] += 1
            deg[int(t)] += 1
    pr = np.array(pairs, dtype=np.int64).reshape(-1, 2)
    return np.concatenate([pr, pr[:, ::-1]], axis=0)


def random_edges(rng: np.random.Generator, n: int, density: float) -> np.ndarray:
    """round(density * N^2) directed edges between randomly chosen distinct vertices, position ignored
    (capped at the N (N - 1) ordered pairs that exist)."""
    want = min(int(round(density * n * n)), n * (n - 1))
    codes = rng.choice(n * (n - 1), size=want, replace=False)       # ordered pairs i != j, enumerated
    i = codes // (n - 1)
    j = codes % (n - 1)
    j = j + (j >= i)
    return np.stack([i, j], axis=1)


def _csr(n: int, edges: np.ndarray):
    """Directed edge list -> CSR by source, targets ascending, duplicates and self-edges dropped."""
    e = np.unique(edges[edges[:, 0] != edges[:, 1]].astype(np.int64), axis=0)
    order = np.lexsort((e[:, 1], e[:, 0]))
    e = e[order]
    row = np.zeros(n + 1, dtype=np.uint64)
    np.add.at(row, e[:, 0] + 1, 1)
    return np.cumsum(row).astype(np.uint64), e[:, 1].astype(np.uint32)


def make_test_network(seed: int, n: int, dim: int, cls: str, density: str, *, min_dist_fraction: float = 0.5,
                 frac_inh: float = 0.2, w_range=(0.0, 8.0), L: float = SPACE) -> Network:
    """One network of Table 1.  min_dist_fraction: the paper says the cubic-packing d_min "is reduced to allow for some
    variability in placement" without giving the factor; reading: one half.  Weights are "left to the user" (:392):
    U(w_range), negated for the out-edges of a Bernoulli(frac_inh) subset of vertices (as BASELINE config 5)."""
    assert cls in CLASSES and density in DENSITIES and dim in DIMS
    key = [seed, n, dim, CLASSES.index(cls), DENSITIES.index(density)]
    rng = np.random.default_rng(np.random.SeedSequence(key))
    pos = centre_outwards(place_min_distance(rng, n, dim, L, d_min(L, n, dim, min_dist_fraction)), L)
    par = _PARAM[cls][DENSITIES.index(density)]
    if cls == "lattice":
        edges = lattice_edges(pos, int(par))
    elif cls == "small_world":
        edges = small_world_edges(rng, pos, float(par))
    elif cls == "scale_free":
        edges = scale_free_edges(rng, n, int(par))
    else:
        edges = random_edges(rng, n, float(par))
    row, tgt = _csr(n, edges)
    inh = rng.random(n) < frac_inh
    w = rng.uniform(w_range[0], w_range[1], size=len(tgt)).astype(np.float32)
    src = np.repeat(np.arange(n), np.diff(row.astype(np.int64)))
    w[inh[src]] *= -1.0
    return Network(n, dim, 1, pos.astype(np.float32), row, tgt, w, inh.astype(np.uint8),
                   meta=dict(cls=cls, density=density, parameter=par, d_min=d_min(L, n, dim, min_dist_fraction), L=L))


def table1(seed: int = 0x09083934, **kw) -> list[Network]:
    """The 80 networks of Table 1: 2 dimensions x 5 sizes x 4 connectivity classes x 2 densities."""
    return [make_test_network(seed, n, dim, cls, dens, **kw)
            for dim in DIMS for n in SIZES for cls in CLASSES for dens in DENSITIES]


def batch(networks: list[Network]) -> Network:
    """Concatenate independent networks into one block-diagonal Network with net_offsets (batched mode).  Positions are
    padded to the largest dimension (a 2D network lies in the plane z = 0 of a 3D batch)."""
    dim = max(nw.dim for nw in networks)
    off = np.r_[0, np.cumsum([nw.n_vertices for nw in networks])].astype(np.uint32)
    pos = np.zeros((int(off[-1]), dim), dtype=np.float32)
    rows, tgts, ws, vcs, e0 = [np.zeros(1, np.uint64)], [], [], [], 0
    for b, nw in enumerate(networks):
        pos[off[b]:off[b + 1], :nw.dim] = nw.positions
        rows.append(nw.row_offsets[1:] + np.uint64(e0))
        tgts.append(nw.targets + np.uint32(off[b]))
        ws.append(nw.weights)
        vcs.append(nw.vertex_class)
        e0 += nw.n_edges
    return Network(int(off[-1]), dim, len(networks), pos, np.concatenate(rows).astype(np.uint64),
                   np.concatenate(tgts).astype(np.uint32), np.concatenate(ws).astype(np.float32),
                   np.concatenate(vcs).astype(np.uint8), net_offsets=off,
                   meta=dict(members=[nw.meta for nw in networks]))
