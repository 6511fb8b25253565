"""Spike-time dependent plasticity as the paper writes it (eq. 32-33; eq. 9-10), in pure
Python on top of the pull definition (oracle/pull_definition.py).  TEST INFRASTRUCTURE: the definition that plastic mode
of the CUDA path is compared with in tests/test_parity_gpu.py::test_plastic_* -- at the sizes pure Python
reaches (tens of vertices); it shares nothing with that path.

State added to the framework:
  s_j(t)      time since the last spike of vertex j, transition function eq. 32 verbatim,
                  s_j(t + dt) = (1 - spd(V_j(t))) * (s_j(t) + dt);          +infinity until j has fired once
  w_ij(t)     one weight per edge, now a state of its own (eq. 9), transition function eq. 33 verbatim,
                  q_ij(t) = (s_i(t - tau_ij) - s_j(t)) * max(spd(V_i(t - tau_ij)), spd(V_j(t)))
                  w_ij(t + dt) = w_ij(t) + dt * alpha * sign(q_ij(t)) * exp(-beta * |q_ij(t)|)
The input of vertex j stays eq. 30, sum_k w_kj(t) spd(V_k(t - tau_kj)), with the weight AT THE ARRIVAL step t.

Readings (readings #22, #23):
  #22  The ages inside q are taken after eq. 32's reset factor: a vertex that spikes at the step counts with age 0,
       s~_j(t) = (1 - spd(V_j(t))) s_j(t), likewise the delayed s~_i(t - tau_ij).  Only then does the text hold that a
       post-synaptic spike right after a pre-synaptic arrival strengthens (q = age of the arrival > 0), an arrival
       after a post-synaptic spike weakens (q = -age of that spike < 0) and a coincidence does nothing (q = 0, sign 0):
       with the ages of eq. 32 untouched, q at a spike would compare the two vertices' PREVIOUS inter-spike intervals.
  #23  A vertex that has not fired yet has no age: a q that involves it changes nothing.
By eq. 32 the age one step after a spike is 0 as well, so a pairing k steps apart counts with |q| = (|k| - 1) dt for
|k| >= 2 and, like a coincidence, not at all for |k| = 1 (q = 0, sign 0).
Weights are plain doubles here (no fixed point); with alpha = 0 and weights that are multiples of 2^-16 the run is the
pull definition's, bit for bit (tests/test_oracle_stdp.py).
"""
from __future__ import annotations

import math

from .pull_definition import PullSimulator

INF = float("inf")


class StdpSimulator(PullSimulator):
    def __init__(self, net, cfg, alpha, beta, delays=None, bias=None):
        super().__init__(net, cfg, delays=delays, bias=bias)
        self.alpha, self.beta = float(alpha), float(beta)
        # per target j: [source, weight (double), delay]; the fixed-point value of the static definition / 2^16
        self.w_edges = [[[k, w_fx / 65536.0, dl] for (k, w_fx, dl) in self.in_edges[j]] for j in range(self.n)]
        self.s = [INF] * self.n          # s_j(t)
        self.s_hist = []                 # s_hist[t][j] = s_j(t): the delayed s_i(t - tau_ij) is read from here

    def _arrivals(self, j, t):
        """eq. 30 with the weight at the arrival step; returned in the fixed-point scale of the base class (a float)."""
        total = 0.0
        for (k, w, dl) in self.w_edges[j]:
            if t - dl >= 0 and self.raster[t - dl][k]:
                total += w
        return total * 65536.0

    def _after_step(self, t, fired_now):
        self.s_hist.append(self.s[:])
        for j in range(self.n):                               # eq. 33 for every edge i -> j
            post = fired_now[j]
            s_post = 0.0 if post else self.s[j]               # reading #22
            for edge in self.w_edges[j]:
                i, _, dl = edge
                pre = t - dl >= 0 and self.raster[t - dl][i]
                if not (pre or post):
                    continue                                  # max(spd, spd) = 0
                s_pre = 0.0 if pre else (self.s_hist[t - dl][i] if t - dl >= 0 else INF)
                if s_pre == INF or s_post == INF:
                    continue                                  # reading #23
                q = s_pre - s_post
                if q != 0.0:
                    edge[1] += self.dt * (self.alpha * math.copysign(1.0, q) * math.exp(-self.beta * abs(q)))
        for j in range(self.n):                               # eq. 32
            self.s[j] = 0.0 if fired_now[j] else self.s[j] + self.dt

    def weight(self, i, j):
        for (k, w, _) in self.w_edges[j]:
            if k == i:
                return w
        raise KeyError((i, j))
