"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage or DESIGN.md reading it pins.  None of them re-types the oracle's own
update formula as the expected value: expectations are known-answer vectors, fixed points, closed
forms of linear recurrences (matrix powers), exact integer arrival steps, conservation laws, and
statistics.
"""
import math
import os

import numpy as np
import pytest
from scipy import stats

from gn_inputs import make_config
from helpers import Fp64Gate, base_cfg, hand_net, rs_class
from oracle import Oracle, lib
from oracle import binding as ob
from oracle import pull_definition as pd

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
MODES = ("fp64", "fp32")


def _philox_c(ctr, key):
    c = np.array(ctr, dtype=np.uint32)
    k = np.array(key, dtype=np.uint32)
    o = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(c.ctypes.data, k.ctypes.data, o.ctypes.data)
    return tuple(int(x) for x in o)


def _kat_rows():
    rows = []
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(x, 16) for x in line.split()]
        rows.append((v[0:4], v[4:6], tuple(v[6:10])))
    return rows


# ---- generator (reading #13) -------------------------------------------------------------------
def test_philox_known_answers():
    rows = _kat_rows()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert _philox_c(ctr, key) == out
        assert pd.philox4x32_10(ctr, key) == out


def test_word_layout_counter_and_lane():
    # word(seed, stream, j, idx) = Philox({j/4, idx_lo, idx_hi, stream}, {seed_lo, seed_hi})[j%4]
    seed, idx = 0x1234567890ABCDEF, (7 << 32) | 99
    for j in (0, 1, 2, 3, 4, 1023, 123457):
        blk = _philox_c([j >> 2, idx & 0xFFFFFFFF, idx >> 32, 5], [seed & 0xFFFFFFFF, seed >> 32])
        assert lib().orc_word(seed, 5, j, idx) == blk[j & 3]
        assert pd.word(seed, 5, j, idx) == blk[j & 3]


def test_drive_threshold_and_kick_rate():
    L = lib()
    # floor(rate * dt * 1e-3 * 2^32): 10 Hz at dt = 0.1 ms is p = 1e-3 -> 4294967 (float dt is a hair above 0.1)
    thr = L.orc_drive_threshold(10.0, 0.1)
    assert thr in (4294967, 4294968)
    assert L.orc_drive_threshold(0.0, 0.1) == 0
    # realised kick count within 4 sigma of N*T*p (binomial)
    net, _ = hand_net(4000, [])
    cfg = base_cfg([rs_class(drive_rate_hz=10.0, drive_kick=0.0)], seed=77)
    o = Oracle(net, cfg, "fp32")
    o.step(500)
    k = o.counters()["kicks"]
    mean = 4000 * 500 * 1e-3
    assert abs(k - mean) < 4 * math.sqrt(mean)


def test_drive_words_uniform_chi_square():
    L = lib()
    w = np.array([L.orc_word(42, 5, j, t) for j in range(2000) for t in range(10)], dtype=np.uint64)
    counts = np.bincount((w >> 28).astype(np.int64), minlength=16)
    chi2 = ((counts - len(w) / 16) ** 2 / (len(w) / 16)).sum()
    assert chi2 < stats.chi2.ppf(0.9999, 15)


# ---- create-time quantities ---------------------------------------------------------------------
def test_quantise_ties_to_even_and_scale():
    L = lib()
    assert L.orc_quantise(1.0) == 65536
    assert L.orc_quantise(-12.0) == -786432
    assert L.orc_quantise(0.5 / 65536) == 0      # tie -> even
    assert L.orc_quantise(1.5 / 65536) == 2      # tie -> even
    assert L.orc_quantise(2.5 / 65536) == 2
    assert L.orc_quantise(-0.5 / 65536) == 0
    assert L.orc_quantise(0.75 / 65536) == 1
    assert pd.quantise(1.5 / 65536) == 2 and pd.quantise(2.5 / 65536) == 2


def test_delay_is_distance_over_speed_in_steps():
    """PAPER.md:251 eq. 25 on a 3-4-5 triangle and the ceil / floor-at-1 edges."""
    L = lib()

    def dl(a, b, speed, dt):
        a = np.array(a, dtype=np.float32)
        b = np.array(b, dtype=np.float32)
        return L.orc_delay_steps(a.ctypes.data, b.ctypes.data, len(a), speed, dt)

    assert dl([0, 0], [3, 4], 1.0, 1.0) == 5               # |x| = 5, speed*dt = 1
    assert dl([0, 0], [3, 4], 2.0, 1.0) == 3               # 2.5 -> ceil 3
    assert dl([0, 0, 0], [1, 2, 2], 1.0, 0.5) == 6         # |x| = 3, 0.5 per step
    assert dl([1, 1], [1, 1], 1.0, 1.0) == 1               # coincident points -> 1 (reading #7)
    assert dl([0, 0], [0.25, 0], 1.0, 1.0) == 1
    assert dl([0, 0], [4, 3], 1.0, 1.0) == dl([4, 3], [0, 0], 1.0, 1.0)   # symmetric
    assert pd.delay_steps([0, 0], [3, 4], 2.0, 1.0) == 3


def test_refractory_steps_and_keep():
    L = lib()
    assert L.orc_refractory_steps(2.0, 0.1) == 20
    assert L.orc_refractory_steps(0.0, 0.1) == 0
    assert abs(L.orc_keep(0.1, 2.0) - 0.95) < 1e-8
    assert abs(L.orc_keep(0.1, 500.0) - 0.9998) < 1e-8


# ---- vertex update: fixed points and closed forms -----------------------------------------------
@pytest.mark.parametrize("mode", MODES)
def test_resting_fixed_point(mode):
    """V=-70, W=-14 solves 0.04 V^2 + 5 V + 140 - W = 0 and W = 0.2 V (reading #15).  The class
    parameters are binary32 at the boundary (0.04f, 0.2f are not 0.04, 0.2), which moves the root by
    ~5e-6; a dropped term or a wrong sign moves it by O(1).  A model whose constants are exact in
    binary32 (k2 = 2^-5, b = 1/4, k0 = 176: root V = -64, W = -16) must not move at all."""
    net, _ = hand_net(3, [])
    o = Oracle(net, base_cfg(), mode)
    o.step(1000)
    tol = 2e-5 if mode == "fp64" else 1e-3
    assert np.abs(o.state(ob.V) + 70.0).max() < tol
    assert np.abs(o.state(ob.W) + 14.0).max() < tol
    assert o.counters()["spikes"] == 0
    x = Oracle(net, base_cfg([rs_class(k2=0.03125, k1=5.0, k0=176.0, b=0.25)]), mode)
    x.set_state(ob.V, -64.0)
    x.set_state(ob.W, -16.0)
    x.step(500)
    assert np.all(x.state(ob.V) == -64.0) and np.all(x.state(ob.W) == -16.0)


def test_threshold_fixed_point_is_stationary_and_unstable():
    """V=-50, W=-10 is the second root (V^2 + 120 V + 3500 = 0): one step leaves it in place; a
    nudge above it runs away to a spike, a nudge below relaxes to rest."""
    net, _ = hand_net(1, [])
    o = Oracle(net, base_cfg(), "fp64")
    o.set_state(ob.V, -50.0)
    o.set_state(ob.W, -10.0)
    o.step(1)
    assert abs(o.state(ob.V)[0] + 50.0) < 1e-6 and abs(o.state(ob.W)[0] + 10.0) < 1e-6   # 0.04f, 0.2f
    up = Oracle(net, base_cfg(), "fp64")
    up.set_state(ob.V, -49.0)
    up.set_state(ob.W, -10.0)
    up.step(3000)
    assert up.counters()["spikes"] >= 1
    dn = Oracle(net, base_cfg(), "fp64")
    dn.set_state(ob.V, -51.0)
    dn.set_state(ob.W, -10.0)
    dn.step(20000)
    assert dn.counters()["spikes"] == 0 and abs(dn.state(ob.V)[0] + 70.0) < 1e-3


def test_one_step_quadratic_value():
    """Hand arithmetic: V=-60, W=0, r=0: 0.04*3600 - 300 + 140 = -16, so V' = -60 + 0.1*(-16) = -61.6;
    W' = 0 + 0.1*0.02*(0.2*-60 - 0) = -0.024."""
    net, _ = hand_net(1, [])
    o = Oracle(net, base_cfg(), "fp64")
    o.set_state(ob.V, -60.0)
    o.set_state(ob.W, 0.0)
    o.step(1)
    assert abs(o.state(ob.V)[0] + 61.6) < 1e-6
    assert abs(o.state(ob.W)[0] + 0.024) < 1e-8


@pytest.mark.parametrize("mode", MODES)
def test_linear_model_matches_matrix_power(mode):
    """With k2 = 0 the Euler map is affine, y' = M y + f, M = I + dt [[k1, -1], [a b, -a]],
    f = dt [k0 + bias, 0]; its n-th iterate has the textbook closed form
    y_n = M^n y_0 + (M^n - I)(M - I)^-1 f.  Pins dt, k1, k0, the -W coupling, a, b and the bias."""
    k1, k0, a, b, bias = -0.3, 2.0, 0.05, 0.4, 1.5
    cls = rs_class(k2=0.0, k1=k1, k0=k0, a=a, b=b, v_peak=1e9)
    net, _ = hand_net(2, [])
    o = Oracle(net, base_cfg([cls]), mode, bias=np.array([bias, 0.0], dtype=np.float32))
    y0 = np.array([3.0, -1.0])
    o.set_state(ob.V, y0[0])
    o.set_state(ob.W, y0[1])
    n = 400
    o.step(n)
    dt = float(np.float32(0.1))
    for j, bj in enumerate((bias, 0.0)):
        A = np.array([[np.float32(k1), -1.0], [float(np.float32(a)) * float(np.float32(b)), -float(np.float32(a))]], dtype=np.float64)
        M = np.eye(2) + dt * A
        f = dt * np.array([float(np.float32(k0)) + bj, 0.0])
        Mn = np.linalg.matrix_power(M, n)
        yn = Mn @ y0 + (Mn - np.eye(2)) @ np.linalg.solve(M - np.eye(2), f)
        tol = 1e-9 if mode == "fp64" else 2e-4
        assert abs(o.state(ob.V)[j] - yn[0]) < tol * max(1, abs(yn[0]))
        assert abs(o.state(ob.W)[j] - yn[1]) < tol * max(1, abs(yn[1]))


@pytest.mark.parametrize("mode", MODES)
def test_spike_threshold_is_geq_and_reset(mode):
    """PAPER.md:316 eq. 31 (>=) on the state at the start of the step; eq. 24 reset V <- c, W <- W + d."""
    net, _ = hand_net(2, [])
    o = Oracle(net, base_cfg(), mode)
    o.set_state(ob.V, np.array([30.0, np.nextafter(np.float32(30.0), np.float32(0.0))], dtype=np.float64))
    o.set_state(ob.W, np.array([-3.0, -3.0]))
    o.step(1)
    r = o.raster_bool()
    assert r[0, 0] and not r[0, 1]
    assert o.state(ob.V)[0] == -65.0
    assert o.state(ob.W)[0] == 5.0           # -3 + d, exact in both modes
    assert o.refr()[0] == 20 and o.refr()[1] == 0


@pytest.mark.parametrize("mode", MODES)
def test_refractory_hold(mode):
    """Reading #6: after a spike at t the vertex sits at c_reset for steps t+1 .. t+1+R whatever
    arrives, W and r keep evolving, and the next spike is later than t+1+R."""
    net, _ = hand_net(1, [])
    o = Oracle(net, base_cfg(), mode, bias=np.array([400.0], dtype=np.float32))
    o.set_state(ob.V, 30.0)
    R = 20
    o.step(1)                                 # spike at t = 0
    w_prev = o.state(ob.W)[0]
    for t in range(1, R + 2):                 # state at t = 1 .. R+1 is held
        assert o.state(ob.V)[0] == -65.0, t
        o.step(1)
        assert o.state(ob.W)[0] != w_prev     # W keeps evolving
        w_prev = o.state(ob.W)[0]
    assert o.state(ob.V)[0] != -65.0          # released at t = R + 2
    o.step(60)
    rb = o.raster_bool()[:, 0]
    spikes = np.flatnonzero(rb)
    assert spikes[0] == 0 and len(spikes) >= 2 and spikes[1] > 1 + R
    assert np.all(np.diff(spikes) > R + 1)


@pytest.mark.parametrize("mode", MODES)
def test_psc_and_calcium_geometric_decay(mode):
    """PAPER.md:285 eq. 26 / :364 H_c: one event of weight w consumed at step a gives
    r(a+1+k) = w (1 - dt/tau_s)^k; one spike at t gives c(t+1+k) = ca_jump (1 - dt/tau_c)^k."""
    w, delay = 3.25, 7
    net, dl = hand_net(2, [(0, 1, w, delay)])
    cfg = base_cfg(obs_stride=1, ca_jump=0.5)
    o = Oracle(net, cfg, mode, delays=dl)
    o.set_state(ob.V, np.array([30.0, -70.0]))
    o.step(1)                                   # vertex 0 fires at t = 0, event consumed at a = 7
    o.step(delay)                               # now t = 8 = a + 1
    keep_s, keep_c = 1 - float(np.float32(0.1)) / 2.0, 1 - float(np.float32(0.1)) / 500.0
    tol = 1e-12 if mode == "fp64" else 2e-6
    for k in range(50):
        assert abs(o.state(ob.R)[1] - w * keep_s ** k) < tol * w
        assert abs(o.state(ob.CA)[0] - 0.5 * keep_c ** (k + delay)) < tol
        assert o.state(ob.R)[0] == 0.0
        o.step(1)


@pytest.mark.parametrize("mode", MODES)
def test_alpha_function_psc_matrix_power_integral_and_shape(mode):
    """PAPER.md:288-312 eq. 27, 29, 30 with a = 1/tau_s and the arriving weight as an impulse on p.  One event of
    weight w consumed at step a leaves (r, p) = (0, w) at a+1 and then (r, p)(a+1+k) = M^k (0, w) with the Euler map
    M = [[1, dt], [-dt a^2, 1 - 2 a dt]] (numpy matrix power, not the oracle's recurrence); summing the two
    recurrences gives the EXACT discrete integral  dt * sum_k r_k = w / a^2 = w tau^2; and r tracks the paper's
    continuous alpha function (w/a) * (a t e^{-a t}) = w t e^{-a t} to O(dt)."""
    w, delay, tau = 3.25, 7, 2.0
    net, dl = hand_net(2, [(0, 1, w, delay)])
    cfg = base_cfg([rs_class(tau_syn_ms=tau, psc_alpha=1.0)])
    o = Oracle(net, cfg, mode, delays=dl)
    o.set_state(ob.V, np.array([30.0, -70.0]))
    o.step(1 + delay)                           # vertex 0 fires at t = 0; the event is consumed at step a = 7; now t = a + 1
    dt, a = float(np.float32(0.1)), 1.0 / tau
    M = np.array([[1.0, dt], [-dt * a * a, 1.0 - 2.0 * a * dt]])
    tol = 1e-12 if mode == "fp64" else 3e-6
    total, peak_seen = 0.0, 0.0
    for k in range(600):
        y = np.linalg.matrix_power(M, k) @ np.array([0.0, w])
        assert abs(o.state(ob.R)[1] - y[0]) < tol * w and abs(o.state(ob.P)[1] - y[1]) < tol * w, k
        t_ms = k * dt
        assert abs(o.state(ob.R)[1] - w * t_ms * math.exp(-a * t_ms)) < 0.03 * w       # O(dt) from the continuous curve
        total += o.state(ob.R)[1] * dt
        peak_seen = max(peak_seen, o.state(ob.R)[1])
        assert o.state(ob.R)[0] == 0.0 and o.state(ob.P)[0] == 0.0                     # the source received nothing
        o.step(1)
    assert abs(total - w * tau * tau) < (1e-9 if mode == "fp64" else 1e-4) * w * tau * tau
    assert abs(peak_seen - w / (a * math.e)) < 0.03 * w                                # peak w/(a e) at t = 1/a


def test_alpha_function_psc_in_the_pull_definition():
    """The ring simulator and the pure-Python eq.-30 evaluation agree on a small graph with alpha-function classes."""
    rng = np.random.default_rng(4)
    edges = [(i, j, float(rng.uniform(-4, 9)), int(rng.integers(1, 9))) for i in range(7) for j in range(7)
             if i != j and rng.random() < 0.5]
    net, dl = hand_net(7, edges)
    cfg = base_cfg([rs_class(tau_syn_ms=1.5, psc_alpha=1.0, drive_rate_hz=400.0, drive_kick=40.0)], ring_slots=9)
    o = Oracle(net, cfg, "fp64", delays=dl)
    q = pd.PullSimulator(net, cfg, delays=dl)
    o.step(400)
    q.step(400)
    np.testing.assert_array_equal(o.raster_bool(0, 400), np.array(q.raster, dtype=bool))
    assert o.counters()["spikes"] > 0
    np.testing.assert_allclose(o.state(ob.R), q.r, rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(o.state(ob.P), q.p, rtol=1e-9, atol=1e-9)


@pytest.mark.parametrize("direct", (True, False))
@pytest.mark.parametrize("mode", MODES)
def test_chain_arrival_steps(mode, direct):
    """BASELINE invariant 2: on a chain with integer delays and supra-threshold weights hop h consumes
    its event at a_h = f_(h-1) + delay_h and fires at f_h = a_h + L, L = 1 (direct jump) or 2 (PSC)."""
    delays = [3, 1, 15, 7, 2, 9]
    w = 200.0 if direct else 2000.0
    # PSC mode: tau_s = 0.2 ms (keep = 1/2) so the 2000-unit current is gone before the hold ends
    cls = rs_class(tau_syn_ms=0.0 if direct else 0.2)
    net, dl = hand_net(len(delays) + 1, [(h, h + 1, w, d) for h, d in enumerate(delays)])
    o = Oracle(net, base_cfg([cls]), mode, delays=dl)
    v0 = np.full(net.n_vertices, -70.0)
    v0[0] = 30.0
    o.set_state(ob.V, v0)
    consumed_at = {}
    for t in range(80):
        o.step(1)
        for j in np.flatnonzero(o.consumed()):
            consumed_at.setdefault(int(j), []).append(t)
    rb = o.raster_bool()
    L = 1 if direct else 2
    f = 0
    assert rb[0, 0]
    for h, d in enumerate(delays, start=1):
        a = f + d
        assert consumed_at[h] == [a]
        f = a + L
        assert list(np.flatnonzero(rb[:, h])) == [f]
    assert o.counters()["delivered"] == len(delays)


# ---- delivery: conservation and the ring's definition ---------------------------------------------
@pytest.mark.parametrize("k,n,steps", [(1, None, 3000), (2, 1500, 1500)])
def test_event_count_and_mass_conservation(k, n, steps):
    """BASELINE invariant 3: delivered events = sum over fired sources of their out-degree; and in
    fixed point, delivered mass = consumed mass (kicks excluded) + mass resident in the ring."""
    net, cfg = make_config(k, n=n)
    cfg = dict(cfg, obs_stride=0)
    o = Oracle(net, cfg, "fp32")
    deg = np.diff(net.row_offsets.astype(np.int64))
    for _ in range(steps // 100):
        o.step(100)
        c = o.counters()
        assert c["mass_delivered"] == c["mass_consumed"] + int(o.ring().sum())
    rb = o.raster_bool()
    c = o.counters()
    assert c["spikes"] == rb.sum() > 0
    assert c["delivered"] == int((rb.sum(axis=0) * deg).sum())
    row, wfx = net.row_offsets.astype(np.int64), o.w_fx()
    rowsum = np.array([wfx[row[i]:row[i + 1]].sum() for i in range(net.n_vertices)])
    assert c["mass_delivered"] == int((rb.sum(axis=0) * rowsum).sum())


def test_ring_content_definition():
    """After step t, slot s of vertex m holds the sum of w_fx over edges (k->m, delay) and fire steps
    t_s <= t with arrival a = t_s + delay, t < a <= t + D - 1, a = s (mod D); slot t mod D is zero."""
    net, cfg = make_config(2, n=400)
    cfg = dict(cfg, obs_stride=0, classes=[dict(c, drive_rate_hz=60.0) for c in cfg["classes"]])
    o = Oracle(net, cfg, "fp32")
    D, n = cfg["ring_slots"], net.n_vertices
    row, tgt, dl, wfx = net.row_offsets.astype(np.int64), net.targets, o.delays(), o.w_fx()
    T = 700
    o.step(T)
    rb = o.raster_bool()
    assert rb.sum() > 50
    t = T - 1
    expect = np.zeros((D, n), dtype=np.int64)
    for ts in range(max(0, t - D), t + 1):
        for k in np.flatnonzero(rb[ts]):
            for e in range(row[k], row[k + 1]):
                a = ts + int(dl[e])
                if t < a <= t + D - 1:
                    expect[a % D, tgt[e]] += wfx[e]
    assert np.count_nonzero(expect) > 20
    assert np.array_equal(o.ring(), expect)
    assert not o.ring()[t % D].any()


# ---- observation ------------------------------------------------------------------------------------
def test_gauss_statistics():
    """N(0, gamma^2).  Mean, variance, KS distance, lag-1 and cross-vertex correlation."""
    L = lib()
    g = np.array([[L.orc_gauss(9, j, f) for j in range(64)] for f in range(400)])
    assert abs(g.mean()) < 4 / math.sqrt(g.size)
    assert abs(g.var() - 1.0) < 0.05
    assert stats.kstest(g.ravel(), "norm").pvalue > 1e-3
    assert abs(np.corrcoef(g[:-1].ravel(), g[1:].ravel())[0, 1]) < 0.03       # lag-1 in time
    assert abs(np.corrcoef(g[:, 0::2].ravel(), g[:, 1::2].ravel())[0, 1]) < 0.03   # cos/sin partners
    assert abs(np.corrcoef(g[:, 0::4].ravel(), g[:, 2::4].ravel())[0, 1]) < 0.03   # same block


@pytest.mark.parametrize("mode", MODES)
def test_observation_frames(mode):
    """z = n * mean(c over the frame) + b (+ noise).  With gamma = 0 the trace is the
    frame mean of the closed-form calcium decay after one spike."""
    net, _ = hand_net(2, [])
    stride = 10
    cfg = base_cfg(obs_stride=stride, obs_gain=3.0, obs_offset=0.25, obs_sigma=0.0)
    o = Oracle(net, cfg, mode)
    o.set_state(ob.V, np.array([30.0, -70.0]))
    o.step(5 * stride)
    tr = o.trace()
    assert tr.shape == (5, 2)
    keep = 1 - float(np.float32(0.1)) / 500.0
    c = np.array([keep ** k for k in range(5 * stride)])     # c after step t (spike at t = 0)
    expect = 3.0 * c.reshape(5, stride).mean(axis=1) + 0.25
    assert np.abs(tr[:, 0] - expect).max() < (1e-12 if mode == "fp64" else 1e-5)
    assert np.abs(tr[:, 1] - 0.25).max() == 0.0
    # with noise on and no spikes: sample mean -> b, variance -> gamma^2
    net2, _ = hand_net(256, [])
    cfg2 = base_cfg(obs_stride=1, obs_offset=1.0, obs_sigma=0.05, seed=5)
    o2 = Oracle(net2, cfg2, mode)
    o2.step(200)
    z = o2.trace()
    assert abs(z.mean() - 1.0) < 4 * 0.05 / math.sqrt(z.size)
    assert abs(z.std() - 0.05) < 0.002


# ---- fp32-faithful mode against the fp64 definition ----------------------------------------------------
@pytest.mark.parametrize("k,n,nb,steps", [(1, None, None, 4000), (2, 2000, None, 2500), (3, 3001, None, 1500),
                                          (5, 500, 4, 2000)])
def test_fp32_mode_tracks_fp64_until_divergence(k, n, nb, steps):
    """Rasters identical up to the first divergence step t*.  Before t*, every (vertex, checkpoint, variable) sample
    is classed from the rasters and the fp64 state alone (helpers.Fp64Gate): quiet samples
    within 1e-4 rel / 1e-5 abs STRICTLY, recovery samples within 20 x that, upstroke samples (a spike within the next
    3 ms: the quadratic term amplifies any rounding difference) counted and reported; violators < 0.1 % of samples."""
    net, cfg = make_config(k, n=n, n_networks=nb)
    cfg = dict(cfg, obs_stride=0)
    a, b = Oracle(net, cfg, "fp32"), Oracle(net, cfg, "fp64")
    gate, chunk = Fp64Gate(net.n_vertices), 50
    names = (("V", ob.V), ("W", ob.W), ("R", ob.R))
    for done in range(chunk, steps + 1, chunk):
        a.step(chunk)
        b.step(chunk)
        gate.add(done, {w: a.state(i) for w, i in names}, {w: b.state(i) for w, i in names})
    a.step(gate.pre)
    b.step(gate.pre)
    t_star, stats = gate.check(a.raster_bool(), b.raster_bool(), f"oracle fp32 vs fp64, cfg {k}")
    assert b.counters()["spikes"] > 10
    assert t_star is None or t_star > 300
    assert stats["quiet"] > 0.3 * stats["samples"]          # the strict class is not a corner case
