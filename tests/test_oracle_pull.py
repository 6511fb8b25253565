"""BASELINE invariant 4: the ring simulator (gn_oracle.c, "push") equals the paper's definition
(eq. 30 evaluated by scanning in-edges against the raster history, pure Python,
oracle/pull_definition.py) -- rasters and consumed fixed-point inputs exactly, state to rounding
(O1 uses no fused multiply-add)."""
import numpy as np
import pytest

from gn_inputs import make_config
from helpers import base_cfg, hand_net, random_digraph, rs_class
from oracle import Oracle
from oracle import binding as ob
from oracle.pull_definition import PullSimulator


def _compare(net, cfg, steps, delays=None, bias=None, v0=None):
    o2 = Oracle(net, cfg, "fp64", delays=delays, bias=bias)
    o1 = PullSimulator(net, cfg, delays=delays, bias=bias)
    if v0 is not None:
        o2.set_state(ob.V, v0)
        o1.V = [float(x) for x in v0]
    for t in range(steps):
        o2.step(1)
        o1.step(1)
        assert [int(x) for x in o2.consumed()] == o1.consumed[t], t
    assert np.array_equal(o2.raster_bool(), np.array(o1.raster, dtype=bool).reshape(steps, net.n_vertices))
    for which, ref in ((ob.V, o1.V), (ob.W, o1.W), (ob.R, o1.r)):
        x = o2.state(which)
        assert np.allclose(x, np.array(ref), rtol=1e-9, atol=1e-9)
    if cfg["obs_stride"]:
        assert np.allclose(o2.state(ob.CA), np.array(o1.c), rtol=1e-9, atol=1e-12)
    return o2


@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("direct", (False, True))
def test_all_small_digraphs_match_pull_definition(seed, direct):
    """Random directed graphs on 2..10 nodes (dense enough to include reciprocal pairs and cycles),
    random delays in [1, D-1], mixed-sign weights, two classes, kicks on, a bias on some vertices."""
    rng = np.random.default_rng(100 + seed)
    n = int(rng.integers(2, 11))
    D = int(rng.choice([2, 3, 8, 16]))
    edges = random_digraph(rng, n, 0.6, D, w_lo=-20.0, w_hi=60.0)
    cls = [rs_class(drive_rate_hz=300.0, drive_kick=25.0, tau_syn_ms=0.0 if direct else 2.0),
           rs_class(a=0.1, d=2.0, drive_rate_hz=150.0, drive_kick=40.0, refractory_ms=0.5,
                    tau_syn_ms=0.0 if direct else 1.0)]
    vc = rng.integers(0, 2, size=n)
    net, dl = hand_net(n, edges, vertex_class=vc)
    bias = np.where(rng.random(n) < 0.5, 6.0, 0.0).astype(np.float32)
    cfg = base_cfg(cls, ring_slots=D, seed=1000 + seed, obs_stride=1)
    o = _compare(net, cfg, 1200, delays=dl, bias=bias)
    c = o.counters()
    assert c["spikes"] > 5 and c["delivered"] > 5


def test_all_pairs_complete_graph():
    """Every ordered pair connected (the 'all-pairs' case), delays from positions (eq. 25)."""
    rng = np.random.default_rng(7)
    n = 9
    pos = rng.uniform(0, 0.1, size=(n, 3)).astype(np.float32)
    edges = [(i, j, float(rng.uniform(-5, 30)), 0) for i in range(n) for j in range(n) if i != j]
    net, _ = hand_net(n, edges, positions=pos)
    cfg = base_cfg([rs_class(drive_rate_hz=200.0, drive_kick=30.0)], ring_slots=32, speed=0.06, seed=3)
    o = _compare(net, cfg, 1500)
    assert o.counters()["delivered"] > 50
    assert o.delays().max() <= 31 and o.delays().min() >= 1 and len(set(o.delays())) > 4


@pytest.mark.parametrize("k,n,steps", [(1, None, 1500), (2, 250, 400)])
def test_configs_match_pull_definition(k, n, steps):
    net, cfg = make_config(k, n=n)
    cfg = dict(cfg, obs_stride=1, obs_sigma=0.0,
               classes=[dict(c, drive_rate_hz=40.0) for c in cfg["classes"]])
    o = _compare(net, cfg, steps)
    assert o.counters()["delivered"] > 100
