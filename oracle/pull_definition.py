"""O1 -- the step written as the paper's DEFINITION, in pure Python.  TEST INFRASTRUCTURE.

Independent of gn_oracle.c (different language, different algorithm, no ring buffer): the input of
vertex j at step t is PAPER.md:311 eq. 30's sum, verbatim,

    I_j(t) = sum over k != j of  w_kj * spd(V_k(t - tau_kj)),

evaluated by scanning every in-edge of j against the stored raster history ("pull").  The vertex
update follows PAPER.md:227-229 eq. 24 with eq. 28's +r(t), eq. 26's PSC and H_c in
plain Python floats (IEEE double, no fused multiply-add).  Pure loops -- small graphs only.

It exists to pin the scalable ring simulator: tests/test_oracle_pull.py requires orc_step (O2) to
reproduce O1's rasters, consumed inputs and state on every directed graph family it tries with
<= 10 nodes, and on configs 1-2.
"""
from __future__ import annotations

import math

_M32 = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    """Philox4x32-10 (Salmon et al., SC'11) from its published description."""
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0 = 0xD2511F53 * c0
        p1 = 0xCD9E8D57 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & _M32, p1 & _M32, ((p0 >> 32) ^ c3 ^ k1) & _M32, p0 & _M32
        k0 = (k0 + 0x9E3779B9) & _M32
        k1 = (k1 + 0xBB67AE85) & _M32
    return c0, c1, c2, c3


def word(seed, stream, j, idx):
    out = philox4x32_10((j >> 2, idx & _M32, (idx >> 32) & _M32, stream), (seed & _M32, (seed >> 32) & _M32))
    return out[j & 3]


def f32(x):
    """Round a Python float to binary32 and back (the boundary types are fp32)."""
    import struct
    return struct.unpack("f", struct.pack("f", x))[0]


def quantise(w):
    """rint(w * 2^16), ties to even; Python's round() on a float is round-half-even."""
    return int(round(f32(w) * 65536.0))


def delay_steps(xi, xj, speed, dt_ms):
    """PAPER.md:251 eq. 25 in whole steps, at least 1."""
    d2 = 0.0
    for a, b in zip(xi, xj):
        d = f32(a) - f32(b)
        d2 = d2 + d * d
    return max(1, math.ceil(math.sqrt(d2) / (f32(speed) * f32(dt_ms))))


class PullSimulator:
    def __init__(self, net, cfg, delays=None, bias=None):
        self.n = n = int(net.n_vertices)
        self.D = int(cfg["ring_slots"])
        self.dt = f32(cfg["dt_ms"])
        self.seed = int(cfg["seed"])
        self.classes = [{k: f32(v) for k, v in c.items()} for c in cfg["classes"]]
        self.cls = [int(x) for x in net.vertex_class]
        self.bias = None if bias is None else [f32(float(x)) for x in bias]
        self.in_edges = [[] for _ in range(n)]      # per target: (source, w_fx, delay)
        row = [int(x) for x in net.row_offsets]
        for i in range(n):
            for e in range(row[i], row[i + 1]):
                m = int(net.targets[e])
                dl = int(delays[e]) if delays is not None else delay_steps(
                    net.positions[i], net.positions[m], cfg["speed"], cfg["dt_ms"])
                assert 1 <= dl <= self.D - 1
                self.in_edges[m].append((i, quantise(float(net.weights[e])), dl))
        self.V = [-70.0] * n
        self.W = [self.classes[self.cls[j]]["b"] * -70.0 for j in range(n)]
        self.r = [0.0] * n
        self.p = [0.0] * n          # second PSC state of the alpha-function (eq. 27)
        self.c = [0.0] * n
        self.refr = [0] * n
        self.raster = []            # raster[t][j]
        self.consumed = []          # consumed[t][j], kick included, fixed point
        self.tau_ca = f32(cfg["tau_ca_ms"])
        self.ca_jump = f32(cfg["ca_jump"])

    def _arrivals(self, j, t):
        """eq. 30: sum of w_kj * spd(V_k(t - tau_kj)) over the in-edges of j, from the raster history (fixed point)."""
        I_fx = 0
        for (k, w_fx, dl) in self.in_edges[j]:
            if t - dl >= 0 and self.raster[t - dl][k]:
                I_fx += w_fx
        return I_fx

    def _after_step(self, t, fired_now):
        """Hook for transition functions beyond the vertex states (oracle/stdp_definition.py)."""

    def step(self, n_steps=1):
        for _ in range(n_steps):
            t = len(self.raster)
            fired_now = [False] * self.n
            consumed = [0] * self.n
            V2, W2, r2, c2, refr2 = self.V[:], self.W[:], self.r[:], self.c[:], self.refr[:]
            p2 = self.p[:]
            for j in range(self.n):
                q = self.classes[self.cls[j]]
                I_fx = self._arrivals(j, t)
                thr = math.floor(q["drive_rate_hz"] * self.dt * 1e-3 * 4294967296.0)
                if thr > 0 and word(self.seed, 5, j, t) < thr:
                    I_fx += quantise(q["drive_kick"])
                consumed[j] = I_fx
                I = I_fx / 65536.0
                U = 0.0 if self.bias is None else self.bias[j]     # U_j(t) of eq. 28
                V, W, r = self.V[j], self.W[j], self.r[j]
                direct = not (q["tau_syn_ms"] > 0.0)
                R = int(round(q["refractory_ms"] / self.dt))
                fired = self.refr[j] == 0 and V >= q["v_peak"]
                W_euler = W + self.dt * (q["a"] * (q["b"] * V - W))
                if fired:
                    V2[j], W2[j], refr2[j] = q["c_reset"], W + q["d"], R
                elif self.refr[j] > 0:
                    V2[j], W2[j], refr2[j] = q["c_reset"], W_euler, self.refr[j] - 1
                else:
                    dV = q["k2"] * V * V + q["k1"] * V + q["k0"] - W + (0.0 if direct else r) + U
                    V2[j] = V + self.dt * dV + (I if direct else 0.0)
                    W2[j] = W_euler
                if not direct and q.get("psc_alpha", 0.0) != 0.0:
                    a = 1.0 / q["tau_syn_ms"]                      # eq. 29: H_r = r + dt p; eq. 30: H_p with the impulse reading
                    r2[j] = r + self.dt * self.p[j]
                    p2[j] = self.p[j] + self.dt * (-a * a * r - 2.0 * a * self.p[j]) + I
                elif not direct:
                    r2[j] = r * (1.0 - self.dt / q["tau_syn_ms"]) + I
                c2[j] = self.c[j] * (1.0 - self.dt / self.tau_ca) + (self.ca_jump if fired else 0.0)
                fired_now[j] = fired
            self.V, self.W, self.r, self.c, self.refr = V2, W2, r2, c2, refr2
            self.p = p2
            self.raster.append(fired_now)
            self.consumed.append(consumed)
            self._after_step(t, fired_now)
