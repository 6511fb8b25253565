"""Pins of the C oracle's plastic mode (oracle/gn_oracle.c orc_enable_stdp / orc_step_plastic; eq. 32-33) --
the oracle that reaches the sizes the CUDA path's plastic kernels are tested at.  It is pinned, before any kernel is compared
with it, against things other than itself: eq. 33's closed form for one pairing (18 cases, both modes), the pure-Python
definition (oracle/stdp_definition.py, a separate writing of the same equations on top of the pull definition) on random
digraphs, an event-by-event sum recomputed from the raster in numpy on a network of a few hundred vertices, eq. 30's "weight
at the arrival step", and -- with alpha = 0 -- the static push/ring oracle bit for bit (pull at arrival time against push
at firing time: two different orders of the same sum)."""
import math

import numpy as np
import pytest

from gn_inputs import Network, make_config
from helpers import base_cfg, hand_net, random_digraph, rs_class
from oracle import Oracle
from oracle import binding as ob
from oracle.stdp_definition import StdpSimulator

DT, ALPHA, BETA = 0.1, 0.5, 0.05
MODES = ["fp64", "fp32"]


def _force(o, vertices):
    v = o.state(ob.V)
    v[list(vertices)] = 30.0
    o.set_state(ob.V, v)


def _run_forced(o, t0, t1, spikes):
    for t in range(t0, t1):
        if t in spikes:
            _force(o, spikes[t])
        o.step(1)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("delay", [1, 7])
@pytest.mark.parametrize("k", [-30, -5, -2, -1, 0, 1, 2, 5, 30])
def test_single_pairing_closed_form(mode, delay, k):
    """Arrival at step a, post-synaptic spike at a + k, after a warm-up pairing (arrival 60, post 100) whose own trace is
    written out exactly: dw = sign(k) dt alpha exp(-beta (|k| - 1) dt) for |k| >= 2, nothing for |k| <= 1 (reading #22)."""
    net, dl = hand_net(2, [(0, 1, 0.0, delay)])
    cfg = base_cfg([rs_class(drive_rate_hz=0.0, refractory_ms=0.0)], ring_slots=64, dt_ms=DT)
    o = Oracle(net, cfg, mode, delays=dl, stdp=(ALPHA, BETA))
    a, post0 = 500, 100
    spikes = {60 - delay: [0], post0: [1], a - delay: [0]}
    spikes.setdefault(a + k, []).append(1)
    _run_forced(o, 0, 560, spikes)
    assert o.raster_bool().sum() == 4
    near = 0.0 if abs(k) == 1 else 1.0
    warm = DT * ALPHA * math.exp(-BETA * 39 * DT)
    if k == 0:
        expect = warm
    elif k > 0:
        expect = warm + DT * ALPHA * (near * math.exp(-BETA * (k - 1) * DT) - math.exp(-BETA * (a - post0 - 1) * DT))
    else:
        expect = warm + DT * ALPHA * (-near * math.exp(-BETA * (-k - 1) * DT) + math.exp(-BETA * (a + k - 60 - 1) * DT))
    # (dt = 0.1f is not 0.1: the oracle takes dt as the binary32 the boundary carries)
    assert o.weights()[0] == pytest.approx(expect, rel=1e-7 if mode == "fp64" else 2e-6, abs=1e-9)


@pytest.mark.parametrize("seed", range(4))
def test_tracks_the_python_definition_on_small_digraphs(seed):
    """Random digraphs of 4..10 vertices, both weight signs, kicks: the C oracle (fp64 mode) and oracle/stdp_definition.py
    have identical rasters up to the first divergence t* -- the definition sums unquantised weights, the oracle rint(w 2^16),
    so chaos separates them eventually; t* must lie beyond 1,000 steps -- and while the rasters agree every weight agrees to
    1e-9: eq. 33 depends on the spike times alone."""
    rng = np.random.default_rng(100 + seed)
    n = int(rng.integers(4, 11))
    net, dl = hand_net(n, random_digraph(rng, n, 0.4, 16, w_lo=-4.0, w_hi=8.0))
    cfg = base_cfg([rs_class(drive_rate_hz=300.0)], ring_slots=16, dt_ms=DT)
    o = Oracle(net, cfg, "fp64", delays=dl, stdp=(ALPHA, BETA))
    sim = StdpSimulator(net, cfg, ALPHA, BETA, delays=dl)
    row = net.row_offsets.astype(np.int64)
    edges = [(i, int(net.targets[e])) for i in range(n) for e in range(row[i], row[i + 1])]
    w0 = o.weights().copy()
    steps, chunk, t_star, moved = 2000, 100, None, 0.0
    for done in range(chunk, steps + 1, chunk):
        o.step(chunk)
        sim.step(chunk)
        ro, rs = o.raster_bool(done - chunk, chunk), np.array(sim.raster[done - chunk:done], dtype=bool)
        if not np.array_equal(ro, rs):
            t_star = done - chunk + int(np.flatnonzero((ro != rs).any(axis=1))[0])
            break
        wo, ws = o.weights(), np.array([sim.weight(i, j) for (i, j) in edges])
        np.testing.assert_allclose(wo, ws, rtol=1e-9, atol=1e-9)
        moved = float(np.abs(wo - w0).max())
    assert t_star is None or t_star > 1000, t_star
    assert moved > 0.05 and o.counters()["spikes"] > 30


@pytest.mark.parametrize("mode", MODES)
def test_event_sum_recomputed_from_the_raster_at_a_few_hundred_vertices(mode):
    """Two classes (excitatory / inhibitory, negative weights), 300 vertices, ~4,500 edges, kicks: every final weight = the
    initial one + the sum over its events, recomputed here from the raster alone in event form (numpy; for every post-synaptic
    spike the most recent earlier arrival, for every arrival the most recent earlier post-synaptic spike, ages by eq. 32) --
    a second writing of eq. 33 that shares nothing with the oracle's per-step edge loop."""
    rng = np.random.default_rng(5)
    n, D = 300, 32
    vc = (rng.random(n) < 0.2).astype(np.uint8)
    edges = [(i, j, float(rng.uniform(-9.0, -2.0) if vc[i] else rng.uniform(0.5, 6.0)), int(rng.integers(1, D)))
             for i in range(n) for j in range(n) if i != j and rng.random() < 0.05]
    net, dl = hand_net(n, edges, vertex_class=vc)
    cfg = base_cfg([rs_class(drive_rate_hz=150.0), rs_class(a=0.1, d=2.0, drive_rate_hz=150.0)], ring_slots=D, dt_ms=DT)
    o = Oracle(net, cfg, mode, delays=dl, stdp=(ALPHA, BETA), threads=4)
    w0 = o.weights().copy()
    steps = 3000
    o.step(steps)
    r = o.raster_bool()
    assert r.sum() > 1000 and r[:, vc == 1].any() and r[:, vc == 0].any()
    spike_steps = [np.flatnonzero(r[:, j]) for j in range(n)]
    row = net.row_offsets.astype(np.int64)
    w1, worst, changed = o.weights(), 0.0, 0
    dt, beta = float(np.float32(DT)), float(np.float32(BETA))   # the boundary carries binary32 parameters
    for i in range(n):
        for e in range(row[i], row[i + 1]):
            j, d = int(net.targets[e]), int(dl[e])
            arr = spike_steps[i] + d
            arr = arr[arr < steps]
            post = spike_steps[j]
            total = 0.0
            both = np.intersect1d(arr, post)
            for t in np.setdiff1d(post, both):                  # strengthening: most recent arrival strictly before t
                k = np.searchsorted(arr, t) - 1
                if k >= 0 and t - arr[k] > 1:
                    total += dt * ALPHA * math.exp(-beta * (t - arr[k] - 1) * dt)
            for t in np.setdiff1d(arr, both):                   # weakening: most recent post spike strictly before t
                k = np.searchsorted(post, t) - 1
                if k >= 0 and t - post[k] > 1:
                    total -= dt * ALPHA * math.exp(-beta * (t - post[k] - 1) * dt)
            worst = max(worst, abs(w1[e] - (w0[e] + total)))
            changed += abs(total) > 1e-3
    assert worst < (1e-9 if mode == "fp64" else 2e-5), worst     # fp32: a few hundred rounded updates of weights up to 9
    assert changed > 1000


def test_input_uses_the_weight_at_the_arrival_step():
    """eq. 30: a spike emitted at step 200 over a delay of 20 is weighed with w(220), which a post-synaptic spike at 210 has
    changed while it was in flight (a delay ring filled at firing time would deliver w(200))."""
    net, dl = hand_net(2, [(0, 1, 2.0, 20)])
    cfg = base_cfg([rs_class(drive_rate_hz=0.0, refractory_ms=0.0)], ring_slots=64, dt_ms=DT)
    o = Oracle(net, cfg, "fp64", delays=dl, stdp=(ALPHA, BETA))
    dt, beta = float(np.float32(DT)), float(np.float32(BETA))   # the boundary carries binary32 parameters
    _run_forced(o, 0, 200, {100 - 20: [0], 130: [1]})
    w1 = o.weights()[0]
    assert w1 == pytest.approx(2.0 + dt * ALPHA * math.exp(-beta * 29 * dt), rel=1e-12)
    _run_forced(o, 200, 221, {200: [0], 210: [1]})               # step 220 is the last one taken: its input is still readable
    w_at_210 = w1 + dt * ALPHA * math.exp(-beta * (210 - 100 - 1) * dt)
    assert o.consumed()[1] == int(np.rint(w_at_210 * 65536.0))
    assert o.consumed()[1] != int(np.rint(w1 * 65536.0))


@pytest.mark.parametrize("mode", MODES)
def test_alpha_zero_is_the_static_ring_oracle_bit_for_bit(mode):
    """With alpha = 0 the plastic mode's pull at arrival time must give what the static oracle's push into the delay ring
    gives: rasters, every state word, consumed inputs and counters identical, on a slice of config 3 (D = 64, two classes)
    and on a batch of config 5's small networks with observation."""
    for k, n, nb in ((3, 600, None), (5, 150, 3)):
        net, cfg = make_config(k, n=n, n_networks=nb)
        a = Oracle(net, cfg, mode, stdp=(0.0, BETA), threads=4)
        b = Oracle(net, cfg, mode, threads=4)
        for _ in range(4):
            a.step(250)
            b.step(250)
            np.testing.assert_array_equal(a.consumed(), b.consumed())
        np.testing.assert_array_equal(a.raster(), b.raster())
        for w in (ob.V, ob.W, ob.R, ob.CA):
            np.testing.assert_array_equal(a.state(w), b.state(w))
        ca, cb = a.counters(), b.counters()
        assert ca["spikes"] == cb["spikes"] > 0 and ca["kicks"] == cb["kicks"]
        assert ca["mass_consumed"] == cb["mass_consumed"] and ca["delivered"] > 0
        np.testing.assert_array_equal(a.weights(), b.weights())
        if cfg["obs_stride"]:
            np.testing.assert_array_equal(a.trace(), b.trace())


def test_enable_refuses_bad_arguments():
    net, dl = hand_net(2, [(0, 1, 1.0, 3)])
    cfg = base_cfg([rs_class()], ring_slots=16)
    with pytest.raises(ValueError):
        Oracle(net, cfg, "fp64", delays=dl, stdp=(0.5, -1.0))
