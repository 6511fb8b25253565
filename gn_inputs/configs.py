"""The five BASELINE.json workloads (and, as config 6, the paper's own 80-network test set) as seeded synthetic inputs
(DESIGN.md "Input recipe").

Each entry fixes what BASELINE.json leaves open with the reading listed in DESIGN.md
(SURVEY.md section 8(c) readings #5, #12, #16-#20).  A config can be generated at a reduced vertex
count for tests: the box side is shrunk so the vertex density (and with it the degree and delay
distributions away from the boundary) stays that of the full-size config.

Only inputs are made here; the dictionaries below are data (parameter tables), not arithmetic.
"""
from __future__ import annotations

import math

from .generate import Network, geometric_network

MASTER_SEED = 0x09083934

CONFIG_NAMES = {
    1: "cfg1_n100_2d",
    2: "cfg2_n10k_2d_ei_obs",
    3: "cfg3_n100k_3d_exp",
    4: "cfg4_n1m_3d_rgg",
    5: "cfg5_batch4096x1000_2d_obs",
    6: "paper_table1_80_networks",
}


def _cls(a, d, rate_hz, kick=10.0, tau_syn_ms=2.0):
    """One row of gn_class_params.  b = 0.2, c = -65, k2/k1/k0 = 0.04/5/140, v_peak = 30
    (the (a,b,c,d) form of PAPER.md:216-233 eq. 23-24; reading #1), refractory 2 ms."""
    return dict(a=a, b=0.2, c_reset=-65.0, d=d, k2=0.04, k1=5.0, k0=140.0, v_peak=30.0,
                tau_syn_ms=tau_syn_ms, refractory_ms=2.0, drive_rate_hz=rate_hz, drive_kick=kick)


def hh_class(rate_hz=0.0, kick=10.0, tau_syn_ms=2.0, **over):
    """One row of gn_class_params for a Hodgkin-Huxley vertex (model = 1).  The paper prints no
    values: these are the squid-axon parameters of Hodgkin & Huxley (1952) in the modern convention (rest at -65 mV;
    e_l chosen so that -65 mV is the resting point), C in uF/cm^2, g in mS/cm^2, potentials in mV, rates in 1/ms.
    A spike is V >= v_peak = 0 mV (eq. 31) outside the detection dead time refractory_ms, which is what makes one action
    potential one event (a vertex held above v_peak for longer than that is detected again every dead time).  The Izhikevich-only fields are unused and zero."""
    c = dict(a=0.0, b=0.0, c_reset=0.0, d=0.0, k2=0.0, k1=0.0, k0=0.0, v_peak=0.0, tau_syn_ms=tau_syn_ms,
             refractory_ms=2.0, drive_rate_hz=rate_hz, drive_kick=kick, psc_alpha=0.0,
             model=1.0, hh_c=1.0, hh_g_na=120.0, hh_g_k=36.0, hh_g_l=0.3, hh_e_na=50.0, hh_e_k=-77.0, hh_e_l=-54.387,
             hh_v_rest=-65.0,
             hh_am_a=0.1, hh_am_v=-40.0, hh_am_k=10.0,         # 0.1 (V+40) / (1 - exp(-(V+40)/10))
             hh_bm_a=4.0, hh_bm_v=-65.0, hh_bm_k=18.0,         # 4 exp(-(V+65)/18)
             hh_ah_a=0.07, hh_ah_v=-65.0, hh_ah_k=20.0,        # 0.07 exp(-(V+65)/20)
             hh_bh_a=1.0, hh_bh_v=-35.0, hh_bh_k=10.0,         # 1 / (1 + exp(-(V+35)/10))
             hh_an_a=0.01, hh_an_v=-55.0, hh_an_k=10.0,        # 0.01 (V+55) / (1 - exp(-(V+55)/10))
             hh_bn_a=0.125, hh_bn_v=-65.0, hh_bn_k=80.0)       # 0.125 exp(-(V+65)/80)
    c.update(over)
    return c


def as_hodgkin_huxley(cfg: dict, dt_ms: float = 0.03) -> dict:
    """The same network stepped with Hodgkin-Huxley vertices at the paper's HH time step (0.03 ms, 1 s =
    33,333 steps): every class keeps its drive and PSC and becomes hh_class(); the speed is scaled so that every delay
    keeps its number of STEPS (the ring depth of the config stays valid); steps = one simulated second."""
    classes = [hh_class(c["drive_rate_hz"], c["drive_kick"], c["tau_syn_ms"]) for c in cfg["classes"]]
    return dict(cfg, classes=classes, dt_ms=dt_ms, speed=cfg["speed"] * cfg["dt_ms"] / dt_ms,
                steps=int(round(1000.0 / dt_ms)), name=cfg["name"] + "+hh")


def _rs(rate):  # regular spiking, excitatory
    return _cls(0.02, 8.0, rate)


def _fs(rate):  # fast spiking, inhibitory
    return _cls(0.1, 2.0, rate)


def _p_within_cube(rho):  # P(two uniform points in a unit cube are closer than rho), rho <= 1
    return 4 * math.pi * rho ** 3 / 3 - 3 * math.pi * rho ** 4 / 2 + 8 * rho ** 5 / 5 - rho ** 6 / 6


def _radius_for_degree_cube(n, side, degree):
    lo, hi = 0.0, 1.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if (n - 1) * _p_within_cube(mid) < degree:
            lo = mid
        else:
            hi = mid
    return side * lo


def make_config(k: int, n: int | None = None, n_networks: int | None = None,
                seed: int | None = None) -> tuple[Network, dict]:
    """Return (Network, cfg) for BASELINE config k (1..5).

    `n` overrides the vertex count (per network for config 5) keeping the vertex density;
    `n_networks` overrides config 5's batch size.  cfg carries every scalar gn_create needs
    plus `steps` (the config's nominal run length) and `name`.
    """
    seed = (MASTER_SEED + k) if seed is None else seed
    base = dict(dt_ms=0.1, tau_ca_ms=500.0, ca_jump=1.0, obs_gain=1.0, obs_offset=0.0,
                obs_sigma=0.05, obs_stride=0, seed=seed, name=CONFIG_NAMES[k])
    if k == 1:
        n_full, dim, side = 100, 2, 1.0
        n = n or n_full
        side *= (n / n_full) ** (1 / dim)
        net = geometric_network(seed, n, dim, side, 0.15, p0=0.5, w_exc=(0.0, 8.0))
        cfg = dict(base, ring_slots=16, speed=0.1, classes=[_rs(10.0)], steps=10_000)
    elif k == 2:
        n_full, dim, side = 10_000, 2, 3.0
        n = n or n_full
        side *= (n / n_full) ** (1 / dim)
        # reading #16: radius 0.15 mm, p = 0.665 => mean out-degree 50 away from the boundary
        net = geometric_network(seed, n, dim, side, 0.15, p0=0.665, frac_inh=0.2,
                                w_exc=(0.0, 6.0), w_inh=(-12.0, 0.0))
        cfg = dict(base, ring_slots=16, speed=0.1, classes=[_rs(5.0), _fs(5.0)], steps=10_000,
                   obs_stride=1)
    elif k == 3:
        n_full, dim, side = 100_000, 3, 1.0
        n = n or n_full
        side *= (n / n_full) ** (1 / dim)
        # reading #17: p = 0.3 exp(-d / 0.05 mm), cut off at the delay cap 63 * speed * dt
        net = geometric_network(seed, n, dim, side, 0.315, kind=1, p0=0.3, lam=0.05, frac_inh=0.2,
                                w_exc=(0.0, 6.0), w_inh=(-12.0, 0.0))
        cfg = dict(base, ring_slots=64, speed=0.05, classes=[_rs(5.0), _fs(5.0)], steps=20_000)
    elif k == 4:
        n_full, dim, side = 1_000_000, 3, 2.0
        n = n or n_full
        # reading #18: radius calibrated (closed form) to mean out-degree 200 at FULL size
        radius = _radius_for_degree_cube(n_full, side, 200.0)
        side *= (n / n_full) ** (1 / dim)
        net = geometric_network(seed, n, dim, side, radius, p0=1.0, frac_inh=0.2,
                                w_exc=(0.0, 6.0), w_inh=(-12.0, 0.0))
        cfg = dict(base, ring_slots=128, speed=0.006, classes=[_rs(2.0), _fs(2.0)], steps=10_000)
        net.meta["radius"] = radius
    elif k == 5:
        n_per = n or 1000
        nb = n_networks or 4096
        side = (n_per / 1000) ** 0.5
        # reading #19: 20 % of vertices inhibitory, their out-weights sign-flipped; delays 1..31
        net = geometric_network(seed, n_per, 2, side, 0.08, p0=1.0, frac_inh=0.2,
                                w_exc=(0.0, 8.0), w_inh=(-8.0, 0.0), n_networks=nb)
        cfg = dict(base, ring_slots=32, speed=0.0259, classes=[_rs(10.0), _rs(10.0)], steps=5_000,
                   obs_stride=100)
    elif k == 6:
        # Not a BASELINE config: the paper's own test set (Table 1), regenerated by paper_test_set.py and
        # stepped as ONE batch of 80 independent networks (N = 10 .. 1000, 2D and 3D, four connectivity classes, two
        # densities).  The paper leaves model, weights and speed to the user: config 5's classes and observation; the
        # speed puts the longest possible distance (the cube's diagonal) at 31 steps.  `n` / `n_networks` are ignored.
        from . import paper_test_set as ts
        net = ts.batch(ts.table1(seed))
        side = ts.SPACE
        cfg = dict(base, ring_slots=32, speed=side * math.sqrt(3.0) / 31.0 / base["dt_ms"] * 1.0001,
                   classes=[_rs(10.0), _rs(10.0)], steps=5_000, obs_stride=100)
    else:
        raise ValueError("config must be 1..6")
    net.meta.update(config=k, side=side, seed=seed)
    return net, cfg
