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


class Fp64Gate:
    """The fp32 path (CUDA kernels, or the oracle's fp32-faithful mode) against the fp64 DEFINITION
    (north_star: state within 1e-4 relative / 1e-5 absolute).

    A sample is (vertex, checkpoint, variable in V/W/r) at a checkpoint not later than the first raster
    divergence t*.  Every sample is put in exactly one class, from the two rasters and the fp64 state alone:

      upstroke   the vertex fires (in either run) within the next `pre` steps.  The Euler map's gain
                 dV'/dV = 1 + dt (2 k2 V + k1) exceeds 1 above V_exp = -k1 / (2 k2) and reaches 1.7 per step at the
                 peak, so a rounding difference is amplified by orders of magnitude before the reset discards it:
                 no bound is asserted, the count and the largest error are reported.
      recovery   not upstroke, and within the last `post` steps the vertex either fired or was seen (at a
                 checkpoint) at V >= V_exp, the expanding zone: the amplified difference was integrated into W
                 through b V and decays with 1/a (500 steps for a = 0.02/ms): within `loose` x the tolerance.
      quiet      everything else: within the tolerance, strictly.

    check() asserts the two bounds and that upstroke + recovery violators stay below `frac` of all samples."""

    REL, ABS = 1e-4, 1e-5

    def __init__(self, n_vertices, v_exp=-62.5, pre=30, post=1000, loose=20.0, frac=1e-3):
        self.n, self.v_exp, self.pre, self.post, self.loose, self.frac = n_vertices, v_exp, pre, post, loose, frac
        self.snaps = []

    def add(self, t, fp32_state, fp64_state):
        """State BEFORE step t runs: two dicts name -> array (fp64_state must hold 'V')."""
        self.snaps.append((int(t), {k: np.asarray(v, np.float64) for k, v in fp32_state.items()},
                           {k: np.asarray(v, np.float64) for k, v in fp64_state.items()}))

    def check(self, raster32, raster64, label=""):
        """Rasters as bool [steps][n] covering every checkpoint plus `pre` steps beyond the last one."""
        diff = (raster32 != raster64).any(axis=1)
        t_star = int(np.flatnonzero(diff)[0]) if diff.any() else None
        either = raster32 | raster64
        steps = either.shape[0]
        # last[t][j] / nxt[t][j] as running arrays over time would be steps x n; walk the checkpoints instead
        stats = dict(samples=0, upstroke=0, recovery=0, quiet=0, upstroke_viol=0, recovery_viol=0, quiet_viol=0,
                     upstroke_max=0.0, recovery_max=0.0, quiet_max=0.0)
        for t, s32, s64 in self.snaps:
            if t_star is not None and t > t_star:
                continue
            assert t + self.pre <= steps, "rasters must cover `pre` steps beyond the last checkpoint"
            soon = either[t:t + self.pre].any(axis=0)
            recent = either[max(0, t - self.post):t].any(axis=0)
            for t2, _, z64 in self.snaps:                     # excursions into the expanding zone, spike or not
                if t - self.post <= t2 <= t:
                    recent = recent | (z64["V"] >= self.v_exp)
            up = soon
            rec = ~up & recent
            quiet = ~up & ~rec
            for name in s32:
                err = np.abs(s32[name] - s64[name])
                ratio = err / (self.ABS + self.REL * np.abs(s64[name]))
                for cls, mask in (("upstroke", up), ("recovery", rec), ("quiet", quiet)):
                    stats[cls] += int(mask.sum())
                    if mask.any():
                        stats[cls + "_viol"] += int((ratio[mask] > 1.0).sum())
                        stats[cls + "_max"] = max(stats[cls + "_max"], float(ratio[mask].max()))
                stats["samples"] += ratio.size
        print(f"[fp64 gate{' ' + label if label else ''}] t* = {t_star}; samples {stats['samples']}: quiet {stats['quiet']} "
              f"(violators {stats['quiet_viol']}, worst {stats['quiet_max']:.3g} x tol), recovery {stats['recovery']} "
              f"(violators {stats['recovery_viol']}, worst {stats['recovery_max']:.3g} x tol), upstroke {stats['upstroke']} "
              f"(violators {stats['upstroke_viol']}, worst {stats['upstroke_max']:.3g} x tol)")
        assert stats["samples"] > 0
        assert stats["quiet_viol"] == 0, stats
        assert stats["recovery_max"] <= self.loose, stats
        assert stats["upstroke_viol"] + stats["recovery_viol"] <= self.frac * stats["samples"], stats
        if t_star is not None:
            assert np.array_equal(raster32[:t_star], raster64[:t_star])
        return t_star, stats


# The gate's windows for Hodgkin-Huxley vertices at dt = 0.03 ms: the sodium current regenerates
# above about -58 mV; an action potential is ~3 ms from threshold to the end of its fall (100 steps before its detection
# at 0 mV, V moving at up to 300 mV/ms so that a timing difference of 1e-4 ms is already 0.03 mV); the after-
# hyperpolarisation and the slow gate n forget it over ~45 ms (1,500 steps).  There is no reset that discards the
# difference, so the recovery bound is 50 x the tolerance and, the network firing at 44 Hz, up to 0.5 % of the samples
# may exceed the plain tolerance; quiet samples meet it strictly.
HH_GATE = dict(v_exp=-58.0, pre=100, post=1500, loose=50.0, frac=5e-3)
