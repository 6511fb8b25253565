"""gn_check_headroom_static (include/gn.h): the overflow check for callers that cannot allocate device memory.

Some users of the library cannot call cudaMalloc when they need this answer: their host program's memory pool owns the
whole GPU and forbids driver allocations, or they sit on a loop that cudaMalloc / cudaFree would stall, or the network's
workspace took the last free memory.  For them this entry point keeps its per-target sums in a fixed 8 MB array inside
libgn.so instead of a caller-supplied workspace.  The array is shared by all calls and keeps what the last call left in
it, so the thing to prove is that a call's answer does not depend on the call before it: every case below is asked
twice in a row, a risky weight set directly in front of a safe one and the other way round, and each answer must equal
the verdict of the existing path -- gn_create, which does the same check in its workspace (GN_E_OVERFLOW_RISK /
GN_E_BAD_GRAPH / success) -- and, for the count of targets at risk, the integer sum written out with numpy (bit-exact:
this is integer work, as in the other GPU tests).

The file is named to be collected last: with `pytest -x` a failure here must not hide the parity tests.  It builds its
own inputs and relies on nothing the other tests leave behind, so it passes alone in a fresh process as well.
"""
import numpy as np
import pytest

import paper_0908_3934_b200 as gn
from gn_inputs import Network
from helpers import base_cfg, rs_class

pytestmark = pytest.mark.gpu

N, D, KICK = 50_000, 16, 10.0
KICK_FX = 655_360                      # rint(10 * 2^16)
LIMIT = 2 ** 31 - 1 - KICK_FX          # the most a target's sum of |w_fx| may reach


def _graph(seed, extra_edges=()):
    """Random digraph of ~8 out-edges per vertex (weights on a 2^-16 grid so that w * 65536 is exact), plus
    extra_edges = [(source, target, w_fx)]; CSR by source."""
    rng = np.random.default_rng(seed)
    src = rng.integers(0, N - 2_000, size=400_000)        # vertices N-2000 .. N-1 get only the edges a case adds
    tgt = rng.integers(0, N - 2_000, size=400_000)
    wfx = rng.integers(-6 * 65536, 8 * 65536, size=400_000)
    if len(extra_edges):
        ex = np.asarray(extra_edges, dtype=np.int64)
        src, tgt, wfx = np.concatenate([src, ex[:, 0]]), np.concatenate([tgt, ex[:, 1]]), np.concatenate([wfx, ex[:, 2]])
    order = np.argsort(src, kind="stable")
    src, tgt, wfx = src[order], tgt[order], wfx[order]
    row = np.zeros(N + 1, dtype=np.uint64)
    np.add.at(row, src + 1, 1)
    row = np.cumsum(row).astype(np.uint64)
    w = (wfx.astype(np.float64) / 65536.0).astype(np.float32)
    assert np.array_equal(np.rint(w.astype(np.float64) * 65536.0).astype(np.int64), wfx)
    return row, tgt.astype(np.uint32), w, wfx


def _exact_sum_edges(target, total):
    """128 edges from distinct sources into `target` whose |w_fx| add up to exactly `total` (each below 2^24)."""
    big = 2 ** 24 - 1
    rest = total - 127 * big
    assert 0 < rest < 2 ** 24
    return [(k, target, big if k % 2 else -big) for k in range(127)] + [(127, target, rest)]


def _existing_path_verdict(row, tgt, w):
    """What gn_create says about this graph: the check as every other caller gets it, in a torch-allocated workspace."""
    net_in = Network(N, 2, 1, np.zeros((N, 2), np.float32), row, tgt, w, np.zeros(N, np.uint8))
    cfg = base_cfg(classes=[rs_class(drive_kick=KICK)], ring_slots=D)
    delays = np.ones(len(tgt), dtype=np.uint8)
    try:
        gn.create_from_inputs(net_in, cfg, delays=delays).destroy()
        return gn.GN_OK
    except gn.GnError as err:
        return err.code


def _static_path(tgt, w, out):
    import torch
    t = torch.from_numpy(tgt.view(np.int32)).cuda()
    x = torch.from_numpy(w).cuda()
    out.fill_(-1)                                         # whatever the caller left in `out` must not matter
    gn.gn_check_headroom_static(N, t, x, KICK, out=out)
    torch.cuda.synchronize()
    return [int(v) for v in out.cpu().numpy().view(np.uint32)]


def _at_risk_by_hand(tgt, wfx):
    s = np.zeros(N, dtype=np.int64)
    np.add.at(s, tgt.astype(np.int64), np.abs(wfx))
    return int(np.count_nonzero(s > LIMIT))


CASES = {
    # nothing near the limit
    "safe": [],
    # one target filled to the limit exactly: still safe (the bound is "exceeds", not "reaches")
    "at_limit": _exact_sum_edges(N - 1, LIMIT),
    # one unit more: at risk
    "one_over": _exact_sum_edges(N - 1, LIMIT + 1),
    # three targets far beyond it (each would wrap an int32 ring slot if all its sources fired together)
    "three_over": [(k, N - 1 - j, 30_000 * 65536) for j in range(3) for k in range(40 + j)],
}
EXPECT = {"safe": 0, "at_limit": 0, "one_over": 1, "three_over": 3}


def test_static_scratch_check_agrees_with_gn_create_on_calls_in_a_row():
    import torch
    out = torch.empty(2, dtype=torch.int32, device="cuda:0")      # the caller's 8 bytes, reused by every call
    graphs = {name: _graph(7, extra) for name, extra in CASES.items()}
    verdict = {name: _existing_path_verdict(*g[:3]) for name, g in graphs.items()}
    assert verdict == {"safe": gn.GN_OK, "at_limit": gn.GN_OK, "one_over": gn.GN_E_OVERFLOW_RISK,
                       "three_over": gn.GN_E_OVERFLOW_RISK}
    # risky right before safe, safe right before risky, and every case twice in a row: the array keeps the sums of the
    # call before, so a missing clear shows up as a target still "at risk" (or counted twice) in the call after
    order = ["three_over", "safe", "safe", "one_over", "one_over", "at_limit", "three_over", "three_over", "at_limit", "safe"]
    for name in order:
        row, tgt, w, wfx = graphs[name]
        at_risk, skipped = _static_path(tgt, w, out)
        assert skipped == 0, name
        assert at_risk == EXPECT[name] == _at_risk_by_hand(tgt, wfx), name
        assert (at_risk > 0) == (verdict[name] == gn.GN_E_OVERFLOW_RISK), name


def test_static_scratch_check_counts_rejected_edges_and_refuses_sizes_beyond_its_array():
    import torch
    out = torch.empty(2, dtype=torch.int32, device="cuda:0")
    row, tgt, w, wfx = _graph(11)
    bad_t, bad_w = tgt.copy(), w.copy()
    bad_t[[5, 77, 300_000]] = [N, N + 9, 2 ** 32 - 1]             # targets outside the network
    bad_w[[1_000, 2_000]] = [np.nan, 40_000.0]                    # not a number; 40000 * 2^16 >= 2^31
    assert _existing_path_verdict(row, bad_t, w) == gn.GN_E_BAD_GRAPH
    assert _existing_path_verdict(row, tgt, bad_w) == gn.GN_E_BAD_GRAPH
    assert _static_path(bad_t, bad_w, out) == [0, 5]
    assert _static_path(tgt, w, out) == [0, 0]                    # and the next call is clean again
    # the limit of the fixed array: refused with a message that names it, nothing launched, nothing truncated
    t = torch.zeros(4, dtype=torch.int32, device="cuda:0")
    x = torch.ones(4, dtype=torch.float32, device="cuda:0")
    out.fill_(-1)
    for n_bad in (gn.GN_STATIC_MAX_VERTICES + 1, 0):
        with pytest.raises(gn.GnError) as ei:
            gn.gn_check_headroom_static(n_bad, t, x, 0.0, out=out)
        assert ei.value.code == gn.GN_E_INVALID_ARG and "GN_STATIC_MAX_VERTICES" in str(ei.value)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [-1, -1]
    # the largest size it accepts: every vertex of a maximum-size network can be a target
    far = torch.tensor([gn.GN_STATIC_MAX_VERTICES - 1, 0, gn.GN_STATIC_MAX_VERTICES - 1, 0], dtype=torch.int32, device="cuda:0")
    big = torch.full((4,), 20_000.0, dtype=torch.float32, device="cuda:0")      # 2 x 20000 x 2^16 > 2^31 - 1 on both targets
    gn.gn_check_headroom_static(gn.GN_STATIC_MAX_VERTICES, far, big, 0.0, out=out)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [2, 0]
