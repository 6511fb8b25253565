"""Pins of the oracle's Hodgkin-Huxley vertex class.  The paper prints no equations for it, so
the pins are what the textbook model fixes: the rate functions' closed-form values, the gating steady states and the
resting fixed point, one action potential per supra-threshold pulse, the classical firing rate under a constant
current, and -- for the fp32-faithful mode -- its own exp against libm.  All -m "not gpu"."""
import math

import numpy as np
import pytest

from gn_inputs import hh_class
from helpers import HH_GATE, Fp64Gate, base_cfg, hand_net
from oracle import Oracle, lib
from oracle import binding as ob

DT = 0.03
MODES = ["fp64", "fp32"]
P = hh_class()


def _rate(f, V):
    name = ob.HH_RATES[f]
    return lib().orc_hh_rate(f, P[f"hh_{name}_a"], P[f"hh_{name}_v"], P[f"hh_{name}_k"], V)


def test_rate_functions_textbook_values_at_rest():
    """alpha / beta at V = -65 mV written out from the 1952 formulas (not through the oracle's code path):
    alpha_m = 0.1 * (-25) / (1 - e^2.5), beta_m = 4, alpha_h = 0.07, beta_h = 1 / (1 + e^3),
    alpha_n = 0.01 * (-10) / (1 - e), beta_n = 0.125."""
    expect = [2.5 / (math.e ** 2.5 - 1.0), 4.0, 0.07, 1.0 / (1.0 + math.e ** 3), 0.1 / (math.e - 1.0), 0.125]
    for f, e in enumerate(expect):
        assert _rate(f, -65.0) == pytest.approx(e, rel=1e-12), ob.HH_RATES[f]
    # the printed steady states of every textbook: m_inf = 0.0529, h_inf = 0.5961, n_inf = 0.3177
    inf = [_rate(2 * x, -65.0) / (_rate(2 * x, -65.0) + _rate(2 * x + 1, -65.0)) for x in range(3)]
    assert [round(v, 4) for v in inf] == [0.0529, 0.5961, 0.3177]


def test_rate_function_shapes():
    # linoid: removable singularity at V_half, value A k there; continuous across the series / quotient switch
    assert _rate(0, -40.0) == pytest.approx(0.1 * 10.0, rel=1e-12)
    assert _rate(4, -55.0) == pytest.approx(0.01 * 10.0, rel=1e-12)
    for f, vh, k in ((0, -40.0, 10.0), (4, -55.0, 10.0)):
        for u in (-0.0500001, -0.0499999, 0.0499999, 0.0500001, 1e-9, -1e-9):
            V = vh + u * k
            exact = P[f"hh_{ob.HH_RATES[f]}_a"] * k * (u / -math.expm1(-u))
            assert _rate(f, V) == pytest.approx(exact, rel=2e-8)
    # exponential: ratio over one e-fold; sigmoid: half its amplitude at V_half, complement symmetry
    assert _rate(1, -65.0 - 18.0) / _rate(1, -65.0) == pytest.approx(math.e, rel=1e-12)
    assert _rate(3, -35.0) == pytest.approx(0.5, rel=1e-12)
    assert _rate(3, -35.0 + 7.0) + _rate(3, -35.0 - 7.0) == pytest.approx(1.0, rel=1e-12)
    # monotone the right way round: m and n activate, h inactivates with depolarisation
    V = np.linspace(-100, 50, 301)
    m_inf = np.array([_rate(0, v) / (_rate(0, v) + _rate(1, v)) for v in V])
    h_inf = np.array([_rate(2, v) / (_rate(2, v) + _rate(3, v)) for v in V])
    n_inf = np.array([_rate(4, v) / (_rate(4, v) + _rate(5, v)) for v in V])
    assert (np.diff(m_inf) > 0).all() and (np.diff(n_inf) > 0).all() and (np.diff(h_inf) < 0).all()


def test_exp32_against_libm():
    """The fp32-faithful mode's exp (one rounded binary32 operation per step) is within 2 ulp of the real exponential
    over the whole range the rate functions use, exact at 0, monotone, and saturates at its clamp."""
    L = lib()
    x = np.concatenate([np.linspace(-87.0, 88.0, 200_001), np.linspace(-1.0, 1.0, 50_001)]).astype(np.float32)
    got = np.array([L.orc_exp32(float(v)) for v in x], dtype=np.float64)
    ref = np.exp(x.astype(np.float64))
    rel = np.abs(got - ref) / ref
    assert rel.max() < 2.4e-7, rel.max()           # 2 ulp of binary32
    assert L.orc_exp32(0.0) == 1.0
    xs = np.sort(x[:200_001])
    gs = np.array([L.orc_exp32(float(v)) for v in xs[::50]])
    assert (np.diff(gs) >= 0).all()
    assert L.orc_exp32(200.0) == L.orc_exp32(88.0) and L.orc_exp32(-200.0) == L.orc_exp32(-87.0)
    # and the fp32 rate functions track the definition
    for f in range(6):
        name = ob.HH_RATES[f]
        A, vh, k = P[f"hh_{name}_a"], P[f"hh_{name}_v"], P[f"hh_{name}_k"]
        ak = np.float32(A * k) if f in (0, 4) else np.float32(A)
        for V in np.linspace(-95.0, 45.0, 281):
            r32 = L.orc_hh_rate32(f, float(ak), vh, float(np.float32(1.0 / k)), float(np.float32(V)))
            r64 = L.orc_hh_rate(f, A, vh, k, float(np.float32(V)))
            assert r32 == pytest.approx(r64, rel=3e-6), (name, V)


def _one(mode, **cfg_over):
    net, dl = hand_net(1, [])
    cfg = base_cfg([hh_class()], dt_ms=DT, **cfg_over)
    return Oracle(net, cfg, mode, delays=dl)


@pytest.mark.parametrize("mode", MODES)
def test_resting_state_is_a_fixed_point(mode):
    """e_l = -54.387 is the value that makes -65 mV the resting point: with the gates at m_inf, h_inf, n_inf of -65 mV the
    three currents cancel (-1.22 + 4.40 - 3.18 uA/cm^2, residual 3e-3), so an undriven vertex stays put: |V + 65| < 0.01 mV, gates
    within 5e-4 of their steady states, for a whole simulated 300 ms, and never fires."""
    o = _one(mode)
    assert o.state(ob.V)[0] == -65.0
    g0 = [o.state(w)[0] for w in (ob.HM, ob.HH, ob.W)]
    assert [round(v, 4) for v in g0] == [0.0529, 0.5961, 0.3177]
    o.step(10_000)
    assert abs(o.state(ob.V)[0] + 65.0) < 0.01
    for w, g in zip((ob.HM, ob.HH, ob.W), g0):
        assert abs(o.state(w)[0] - g) < 5e-4
    assert o.counters()["spikes"] == 0
    # the current balance itself, from the printed parameters
    m, h, n = g0
    i_ion = 120.0 * m ** 3 * h * (-65.0 - 50.0) + 36.0 * n ** 4 * (-65.0 + 77.0) + 0.3 * (-65.0 + 54.387)
    assert abs(i_ion) < 5e-3


@pytest.mark.parametrize("mode", MODES)
def test_one_pulse_one_action_potential(mode):
    """A brief supra-threshold current (the PSC state set to 20 uA/cm^2, tau_s = 2 ms: 40 nC/cm^2) fires exactly one action
    potential: one detected event, peak between +30 and +50 mV (textbook overshoot ~ +40), after-hyperpolarisation below
    rest towards e_k, back within 1 mV of rest after 25 ms; the gates stay inside [0, 1] throughout.  A sub-threshold
    pulse (2 uA/cm^2) fires none."""
    o = _one(mode)
    o.set_state(ob.R, np.array([20.0]))
    vs, gates = [], []
    for _ in range(1000):                     # 30 ms, step by step
        o.step(1)
        vs.append(o.state(ob.V)[0])
        gates.append([o.state(w)[0] for w in (ob.HM, ob.HH, ob.W)])
    vs, gates = np.array(vs), np.array(gates)
    assert o.counters()["spikes"] == 1
    assert 30.0 < vs.max() < 50.0
    assert -77.0 < vs.min() < -70.0
    assert abs(vs[-1] + 65.0) < 1.0
    assert gates.min() >= 0.0 and gates.max() <= 1.0
    t_peak = int(vs.argmax())
    assert 20 < t_peak < 120                  # 0.6 .. 3.6 ms after the pulse
    assert (vs >= 0.0).sum() * DT < 1.5       # the spike is about a millisecond wide
    o2 = _one(mode)
    o2.set_state(ob.R, np.array([2.0]))
    o2.step(1000)
    assert o2.counters()["spikes"] == 0


@pytest.mark.parametrize("mode", MODES)
def test_constant_current_fires_at_the_textbook_rate(mode):
    """The squid-axon model under a constant 10 uA/cm^2 fires periodically at ~68-70 Hz (every textbook's f-I curve);
    below rheobase (2 uA/cm^2) it stays silent.  User control U_j enters the current balance (eq. 7)."""
    net, dl = hand_net(2, [])
    cfg = base_cfg([hh_class()], dt_ms=DT)
    o = Oracle(net, cfg, mode, delays=dl, bias=np.array([10.0, 2.0], np.float32))
    o.step(20_000)                            # 600 ms
    r = o.raster_bool()
    t = np.flatnonzero(r[:, 0])
    assert r[:, 1].sum() == 0
    isi = np.diff(t[3:]) * DT                 # after the onset transient
    assert len(isi) > 25
    assert 1000.0 / isi.mean() == pytest.approx(68.5, abs=3.0)
    assert isi.std() < 0.1                    # periodic


def test_hh_synaptic_chain_and_mixed_classes():
    """Delivery is the same for every vertex class: a chain of Hodgkin-Huxley vertices with one Izhikevich vertex in the
    middle relays a spike hop by hop; every hop arrives exactly delay steps after its source fired (ring, eq. 30), and
    O2 equals the pull definition's consumed input."""
    from helpers import rs_class
    delays = [5, 9, 3, 12]
    edges = [(h, h + 1, 400.0, d) for h, d in enumerate(delays)]
    net, dl = hand_net(5, edges, vertex_class=[0, 0, 1, 0, 0])
    cfg = base_cfg([hh_class(tau_syn_ms=0.5), rs_class(tau_syn_ms=0.5)], dt_ms=DT, ring_slots=16)
    o = Oracle(net, cfg, "fp64", delays=dl)
    o.set_state(ob.R, np.array([40.0, 0, 0, 0, 0]))
    fire, seen = {}, {}
    for t in range(3000):
        o.step(1)
        c = o.consumed()
        for j in range(5):
            if c[j] != 0 and j not in seen:
                seen[j] = t
        r = o.raster(t, 1)[0, 0]
        for j in range(5):
            if (r >> j) & 1 and j not in fire:
                fire[j] = t
    assert sorted(fire) == [0, 1, 2, 3, 4]
    for h, d in enumerate(delays):
        assert seen[h + 1] == fire[h] + d


@pytest.mark.parametrize("n", [400])
def test_hh_fp32_mode_tracks_fp64(n):
    """The fp32-faithful Hodgkin-Huxley mode against the definition on a driven recurrent network (44 Hz mean rate):
    rasters identical up to t*, state (V, n, r and the gates m, h) through the gate of the Izhikevich classes with the
    windows of this model (helpers.HH_GATE): quiet samples within 1e-4 rel / 1e-5 abs strictly."""
    from gn_inputs import as_hodgkin_huxley, make_config
    net, cfg = make_config(5, n=n, n_networks=1)
    cfg = dict(as_hodgkin_huxley(cfg), obs_stride=0)
    a, b = Oracle(net, cfg, "fp32"), Oracle(net, cfg, "fp64")
    gate, chunk, steps = Fp64Gate(net.n_vertices, **HH_GATE), 50, 6000
    names = (("V", ob.V), ("W", ob.W), ("R", ob.R), ("M", ob.HM), ("H", ob.HH))
    for done in range(chunk, steps + 1, chunk):
        a.step(chunk)
        b.step(chunk)
        gate.add(done, {w: a.state(i) for w, i in names}, {w: b.state(i) for w, i in names})
    a.step(gate.pre)
    b.step(gate.pre)
    t_star, stats = gate.check(a.raster_bool(), b.raster_bool(), "oracle HH fp32 vs fp64")
    assert b.counters()["spikes"] > 50
    assert t_star is None or t_star > 1000


@pytest.mark.parametrize("mode", MODES)
def test_hh_direct_injection_jumps_v_by_the_weight(mode):
    """tau_syn_ms <= 0 (reading #4; gn.h: "the arriving weight jumps V itself") holds for Hodgkin-Huxley
    vertices as for Izhikevich ones: there is no synaptic current state, and V of the target is higher by exactly the
    weight after the step at which the event arrives.  Two runs that differ only in the weight of the one edge 0 -> 1
    (w against 0) are identical at vertex 1 up to the arrival step f + delay and differ by w right after it; a drive
    kick (reading #12: injected like an arriving event) does the same; r stays 0 throughout; a weight large enough
    relays the spike."""
    w, d = 3.0, 7
    cfg = base_cfg([hh_class(tau_syn_ms=0.0)], dt_ms=DT, ring_slots=16)
    runs = []
    for weight in (w, 0.0):
        net, dl = hand_net(2, [(0, 1, weight, d)])
        o = Oracle(net, cfg, mode, delays=dl, bias=np.array([10.0, 0.0], np.float32))
        v1 = []
        for _ in range(400):
            o.step(1)
            v1.append(o.state(ob.V)[1])
            assert o.state(ob.R)[1] == 0.0
        runs.append((np.array(v1), np.flatnonzero(o.raster_bool()[:, 0])))
    (va, fa), (vb, fb) = runs
    assert len(fa) >= 1 and np.array_equal(fa, fb)
    arrive = int(fa[0]) + d                                   # the step that consumes the event; v1[t] is V after step t
    assert np.array_equal(va[:arrive], vb[:arrive])
    tol = 1e-12 if mode == "fp64" else 4e-6                   # one rounding of a number of magnitude ~65
    assert abs((va[arrive] - vb[arrive]) - w) <= tol
    # strong enough an edge relays the spike: 0 fires, 1 fires shortly after the arrival
    net, dl = hand_net(2, [(0, 1, 30.0, d)])
    o = Oracle(net, cfg, mode, delays=dl, bias=np.array([10.0, 0.0], np.float32))
    o.step(400)
    r = o.raster_bool()
    f0, f1 = np.flatnonzero(r[:, 0]), np.flatnonzero(r[:, 1])
    assert len(f1) >= 1 and f0[0] + d < f1[0] < f0[0] + d + 100
    # drive kicks enter the same way: a lone vertex with a 2,000 Hz drive of +2 mV kicks depolarises by 2 per kick
    cfgk = base_cfg([hh_class(tau_syn_ms=0.0, drive_rate_hz=2000.0, drive_kick=2.0)], dt_ms=DT, ring_slots=16)
    cfgq = base_cfg([hh_class(tau_syn_ms=0.0, drive_rate_hz=2000.0, drive_kick=0.0)], dt_ms=DT, ring_slots=16)
    net, dl = hand_net(1, [])
    ok, oq = Oracle(net, cfgk, mode, delays=dl), Oracle(net, cfgq, mode, delays=dl)
    for _ in range(200):
        before = ok.counters()["kicks"]
        ok.step(1)
        oq.step(1)
        if ok.counters()["kicks"] > before:
            assert abs((ok.state(ob.V)[0] - oq.state(ob.V)[0]) - 2.0) <= tol
            break
        assert ok.state(ob.V)[0] == oq.state(ob.V)[0]
    else:
        raise AssertionError("no kick in 200 steps at 2 kHz")
