"""Small hand-built networks and default parameter tables for the tests (inputs only)."""
from __future__ import annotations

import numpy as np

from gn_inputs import Network


def rs_class(**over):
    c = dict(a=0.02, b=0.2, c_reset=-65.0, d=8.0, k2=0.04, k1=5.0, k0=140.0, v_peak=30.0,
             tau_syn_ms=2.0, refractory_ms=2.0, drive_rate_hz=0.0, drive_kick=10.0)
    c.update(over)
    return c


def base_cfg(classes=None, **over):
    cfg = dict(dt_ms=0.1, speed=0.1, ring_slots=16, classes=classes or [rs_class()],
               tau_ca_ms=500.0, ca_jump=1.0, obs_gain=1.0, obs_offset=0.0, obs_sigma=0.0,
               obs_stride=0, seed=1234, name="hand", steps=0)
    cfg.update(over)
    return cfg


def hand_net(n, edges, vertex_class=None, positions=None, dim=2):
    """edges: iterable of (source, target, weight, delay).  Returns (Network, delays uint8[E])."""
    edges = sorted(edges, key=lambda e: (e[0], e[1]))
    row = np.zeros(n + 1, dtype=np.uint64)
    for e in edges:
        row[e[0] + 1] += 1
    row = np.cumsum(row).astype(np.uint64)
    tgt = np.array([e[1] for e in edges], dtype=np.uint32)
    w = np.array([e[2] for e in edges], dtype=np.float32)
    dl = np.array([e[3] for e in edges], dtype=np.uint8)
    pos = np.zeros((n, dim), dtype=np.float32) if positions is None else np.asarray(positions, dtype=np.float32)
    vc = np.zeros(n, dtype=np.uint8) if vertex_class is None else np.asarray(vertex_class, dtype=np.uint8)
    return Network(n, pos.shape[1], 1, pos, row, tgt, w, vc), dl


def random_digraph(rng, n, p, D, w_lo=-6.0, w_hi=8.0):
    edges = []
    for i in range(n):
        for j in range(n):
            if i != j and rng.random() < p:
                edges.append((i, j, float(rng.uniform(w_lo, w_hi)), int(rng.integers(1, D))))
    return edges


def unpack_raster(words, n):
    bits = np.unpackbits(np.ascontiguousarray(words).view(np.uint8), axis=1, bitorder="little")
    return bits[:, :n].astype(bool)
