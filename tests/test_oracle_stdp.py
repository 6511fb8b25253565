"""Pins of the STDP definition (oracle/stdp_definition.py; eq. 32-33) against what the paper and the
mathematics fix: eq. 32's age recurrence, the closed form of eq. 33 for one pre/post pairing (the two-exponential window
of the model the paper cites), its antisymmetry, no change at coincidence or before both vertices have fired, the
event-by-event sum recomputed from the raster in a different form, eq. 30 with the weight at the ARRIVAL step, and -- with
alpha = 0 -- the static pull definition bit for bit."""
import math

import numpy as np
import pytest

from helpers import base_cfg, hand_net, random_digraph, rs_class
from oracle.pull_definition import PullSimulator
from oracle.stdp_definition import INF, StdpSimulator

DT = 0.1
ALPHA, BETA = 0.5, 0.05          # per ms and 1/ms: a change of alpha*dt = 0.05 at zero age, e-folding over 20 ms


def _pair(delay, w=0.0):
    """Two vertices, one edge 0 -> 1; no drive; weight 0 unless said, so the spikes are the test's alone."""
    net, dl = hand_net(2, [(0, 1, w, delay)])
    cfg = base_cfg([rs_class(drive_rate_hz=0.0, refractory_ms=0.0)], ring_slots=64, dt_ms=DT)
    return StdpSimulator(net, cfg, ALPHA, BETA, delays=dl)


def _run_forced(sim, steps, spikes):
    """spikes: {step: [vertices]} -- V is lifted to the peak just before that step, so the vertex fires AT it (eq. 31)."""
    for t in range(steps):
        for j in spikes.get(t, ()):
            sim.V[j] = 30.0
        sim.step(1)
    return np.array(sim.raster, dtype=bool)


def test_age_recurrence_is_eq_32():
    """s(t + dt) = (1 - spd(V(t))) (s(t) + dt): infinite before the first spike, 0 one step after a spike, then k dt."""
    sim = _pair(5)
    r = _run_forced(sim, 60, {10: [0], 40: [0], 25: [1]})
    assert r[10, 0] and r[40, 0] and r[25, 1] and r.sum() == 3
    s0 = [row[0] for row in sim.s_hist]
    assert all(x == INF for x in s0[:11])                       # s(t) for t <= 10: no spike before
    assert s0[11] == 0.0
    np.testing.assert_allclose(s0[11:41], [k * sim.dt for k in range(30)], rtol=1e-12)
    assert s0[41] == 0.0 and sim.s_hist[26][1] == 0.0 and sim.s_hist[25][1] == INF


@pytest.mark.parametrize("delay", [1, 7])
@pytest.mark.parametrize("k", [-30, -5, -2, -1, 0, 1, 2, 5, 30])
def test_single_pairing_is_the_two_exponential_window(delay, k):
    """Pre-synaptic spike ARRIVES at step a, post-synaptic spike at a + k.  Both vertices have fired once before (ages
    finite: 400 steps earlier, far outside the window's reach at beta * 40 ms = 2 ... so those pairings are subtracted
    exactly, not neglected).  Closed form of eq. 33 with eq. 32's ages: the later of the two events sees the earlier one
    at age (|k| - 1) dt, so  dw = sign(k) dt alpha exp(-beta (|k| - 1) dt)  for |k| >= 2; at coincidence AND one step apart
    q = 0 (eq. 32 resets the age to 0 for the step after a spike) and sign(0) = 0: no change."""
    a = 500
    sim = _pair(delay)
    pre0, post0 = 60 - delay, 100               # warm-up spikes: arrival at 60, post at 100
    _run_forced(sim, 460, {pre0: [0], post0: [1]})
    w_before = sim.weight(0, 1)
    # the warm-up pairing itself, by the same closed form (arrival 60, post 100: k = 40)
    assert w_before == pytest.approx(sim.dt * ALPHA * math.exp(-BETA * 39 * sim.dt), rel=1e-12)
    spikes = {a - delay: [0]}
    spikes.setdefault(a + k, []).append(1)
    for t in range(460, 560):
        for j in spikes.get(t, ()):
            sim.V[j] = 30.0
        sim.step(1)
    dw = sim.weight(0, 1) - w_before
    near = 0.0 if abs(k) == 1 else 1.0             # one step apart: q = 0
    if k == 0:
        expect = 0.0
    elif k > 0:       # post after the arrival: strengthened; the arrival itself saw the warm-up post spike (LTD, age a - 100 - 1)
        expect = sim.dt * ALPHA * (near * math.exp(-BETA * (k - 1) * sim.dt) - math.exp(-BETA * (a - post0 - 1) * sim.dt))
    else:             # post before the arrival: weakened; that post spike saw the warm-up arrival (LTP, age a + k - 60 - 1)
        expect = sim.dt * ALPHA * (-near * math.exp(-BETA * (-k - 1) * sim.dt) + math.exp(-BETA * (a + k - 60 - 1) * sim.dt))
    assert dw == pytest.approx(expect, rel=1e-9, abs=1e-15)


def test_window_is_antisymmetric_and_decays():
    def dw(k):
        sim = _pair(3)
        _run_forced(sim, 2300, {100 - 3: [0], 100: [1]})       # ages finite; 2,200 steps later their trace is e^-11
        w0 = sim.weight(0, 1)
        spikes = {2500 - 3: [0]}
        spikes.setdefault(2500 + k, []).append(1)
        for t in range(2300, 2700):
            for j in spikes.get(t, ()):
                sim.V[j] = 30.0
            sim.step(1)
        return sim.weight(0, 1) - w0
    for k in (2, 4, 20, 100):
        assert dw(k) > 0 > dw(-k)
        assert dw(k) == pytest.approx(-dw(-k), rel=1e-3)          # up to the e^-11 trace of the warm-up spikes
    assert dw(2) > dw(4) > dw(20) > dw(100) > 0 and dw(1) == pytest.approx(0.0, abs=1e-6)
    assert dw(20) / dw(4) == pytest.approx(math.exp(-BETA * 16 * DT), rel=1e-3)


def test_nothing_changes_before_both_vertices_have_fired():
    sim = _pair(4, w=1.5)
    _run_forced(sim, 200, {10: [0], 50: [0], 120: [0]})           # the target never fires (weight too small to make it)
    assert not np.array(sim.raster)[:, 1].any()
    assert sim.weight(0, 1) == 1.5


def test_sum_over_events_recomputed_from_the_raster():
    """A random small network with plastic weights and kicks: every final weight must equal the initial one plus the
    event-by-event sum -- for every post-synaptic spike the most recent earlier arrival, for every arrival the most recent
    earlier post-synaptic spike, ages by eq. 32 -- recomputed here from the raster alone (numpy, event-based: a second
    writing of eq. 33 in another form)."""
    rng = np.random.default_rng(7)
    net, dl = hand_net(8, random_digraph(rng, 8, 0.5, 16, w_lo=0.0, w_hi=9.0))
    cfg = base_cfg([rs_class(drive_rate_hz=400.0)], ring_slots=16, dt_ms=DT)
    sim = StdpSimulator(net, cfg, ALPHA, BETA, delays=dl)
    w0 = {(e[0], j): e[1] for j in range(sim.n) for e in sim.w_edges[j]}
    steps = 3000
    sim.step(steps)
    r = np.array(sim.raster, dtype=bool)
    assert r.sum() > 40
    spike_steps = [np.flatnonzero(r[:, j]) for j in range(sim.n)]
    checked = 0
    for j in range(sim.n):
        for (i, w_final, d) in sim.w_edges[j]:
            arrivals = spike_steps[i] + d
            arrivals = arrivals[arrivals < steps]
            posts = spike_steps[j]
            total = 0.0
            set_a, set_p = set(arrivals.tolist()), set(posts.tolist())
            for t in sorted(set_a | set_p):
                if t in set_a and t in set_p:
                    continue                                             # coincidence
                if t in set_p:                                           # most recent arrival strictly before t
                    prev = arrivals[arrivals < t]
                    if len(prev) and t - prev[-1] > 1:                   # (one step apart: age 0, q = 0)
                        total += sim.dt * ALPHA * math.exp(-BETA * (t - prev[-1] - 1) * sim.dt)
                else:                                                    # most recent post spike strictly before t
                    prev = posts[posts < t]
                    if len(prev) and t - prev[-1] > 1:
                        total -= sim.dt * ALPHA * math.exp(-BETA * (t - prev[-1] - 1) * sim.dt)
            assert w_final == pytest.approx(w0[(i, j)] + total, rel=1e-9, abs=1e-12), (i, j)
            checked += abs(total) > 0
    assert checked >= 5


def test_input_uses_the_weight_at_the_arrival_step():
    """eq. 30 with a plastic weight: a spike emitted at step 0 over a delay of 20 is weighed with w(20), which a post-synaptic
    spike at step 10 (after an earlier arrival) has changed in the meantime."""
    net, dl = hand_net(2, [(0, 1, 2.0, 20)])
    cfg = base_cfg([rs_class(drive_rate_hz=0.0, refractory_ms=0.0)], ring_slots=64, dt_ms=DT)
    sim = StdpSimulator(net, cfg, ALPHA, BETA, delays=dl)
    _run_forced(sim, 200, {100 - 20: [0], 130: [1]})             # arrival 100 (nothing: target never fired), post 130: LTP
    w1 = sim.weight(0, 1)
    assert w1 == pytest.approx(2.0 + sim.dt * ALPHA * math.exp(-BETA * 29 * sim.dt), rel=1e-12)
    spikes = {200: [0], 210: [1]}                                # emitted at 200 (arrives 220); post spike at 210 changes w
    for t in range(200, 230):
        for j in spikes.get(t, ()):
            sim.V[j] = 30.0
        sim.step(1)
    w_at_210 = w1 + sim.dt * ALPHA * math.exp(-BETA * (210 - 100 - 1) * sim.dt)    # LTP against the arrival at 100
    assert sim.consumed[220][1] / 65536.0 == pytest.approx(w_at_210, rel=1e-12)
    assert sim.consumed[220][1] / 65536.0 != pytest.approx(w1, rel=1e-6)


@pytest.mark.parametrize("seed", range(3))
def test_alpha_zero_is_the_static_pull_definition(seed):
    rng = np.random.default_rng(40 + seed)
    n = int(rng.integers(3, 9))
    net, dl = hand_net(n, random_digraph(rng, n, 0.5, 16, w_lo=-6.0, w_hi=8.0))
    cfg = base_cfg([rs_class(drive_rate_hz=50.0)], ring_slots=16, dt_ms=DT)
    a = StdpSimulator(net, cfg, 0.0, BETA, delays=dl)
    b = PullSimulator(net, cfg, delays=dl)
    a.step(1500)
    b.step(1500)
    assert a.raster == b.raster and np.array(a.raster).sum() > 0
    assert [[int(x) for x in row] for row in a.consumed] == b.consumed
    assert a.V == b.V and a.W == b.W and a.r == b.r
