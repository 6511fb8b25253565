"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/gn.h declares; workspace sizing and argument validation; loud failure without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_0908_3934_b200 as gn

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "gn.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gn_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = gn.lib()
    declared = _declared_functions()
    assert set(declared) == set(gn.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name


def test_structs_match_header_layout():
    assert C.sizeof(gn.gn_class_params) == 40 * 4          # 13 + model + 8 Hodgkin-Huxley scalars + 6 rate functions x 3
    # uint32 x2, uint64, uint32 x2, float x2, uint32, float x5, uint32 x3, (pad), uint64, uint32 x2, uint64, float x2
    assert C.sizeof(gn.gn_config) == 104
    assert gn.gn_config.seed.offset == 72 and gn.gn_config.n_edges.offset == 8
    assert gn.gn_config.delivery_mode.offset == 80 and gn.gn_config.queue_capacity.offset == 88


def test_binding_constants_match_the_header():
    """Every GN_* id of include/gn.h (state ids, delivery modes, error codes) has the same value in the binding."""
    text = open(os.path.join(ROOT, "include", "gn.h")).read()
    enum = dict(re.findall(r"\b(GN_[A-Z_]+)\s*=\s*(\d+)", text))
    defs = dict(re.findall(r"#define\s+(GN_[A-Z_]+)\s+\(?(-?\d+)\)?", text))
    assert {"GN_V", "GN_RING", "GN_P", "GN_ACC"} <= set(enum) and {"GN_OK", "GN_E_CUDA", "GN_DELIVER_RESIDENT"} <= set(defs)
    for name, val in {**enum, **defs}.items():
        assert getattr(gn.binding, name) == int(val), name


def test_query_workspace_sizes_and_errors():
    cfg = gn.make_config(1_000_000, 3, 200_000_000, 128, 0.1, 0.006, 2, raster_capacity_steps=0,
                         delivery_mode=gn.GN_DELIVER_RING)
    need = gn.gn_query_workspace(cfg)
    # queue mode (what AUTO picks here: ring 512 MB >> L2), 16 groups of 8 slots: the spike log (128 step slots x 15
    # arrays x N/16 spikes x 4 B) + the 16-bit segment table [N][D] + the raster rows of 3 groups instead of 2 steps
    auto = gn.gn_query_workspace(gn.make_config(1_000_000, 3, 200_000_000, 128, 0.1, 0.006, 2))
    assert auto - need == pytest.approx(128 * 15 * 62_528 * 4 + 1_000_000 * 128 * 2 + 22 * 1_000_064 / 8, rel=1e-3)
    assert auto < 6 * 2 ** 30                                      # config 4 as a whole: under 6 GB
    for bad_q in (dict(delivery_mode=5), dict(queue_group=3), dict(queue_group=32)):
        with pytest.raises(gn.GnError):
            gn.gn_query_workspace(gn.make_config(10, 2, 5, 16, 0.1, 0.1, 1, **bad_q))
    ring, edges = 128 * 1_000_064 * 4, 2 * 200_000_000 * 9   # rows are held twice: caller order and sorted by delay
    assert ring + edges < need < ring + edges + 120_000_000
    bigger = gn.gn_query_workspace(gn.make_config(1_000_000, 3, 200_000_000, 128, 0.1, 0.006, 2, raster_capacity_steps=1000,
                                                      delivery_mode=gn.GN_DELIVER_RING))
    assert bigger - need == pytest.approx((1000 - 2) * 1_000_064 / 8, rel=1e-3)   # two rows are always kept (the spike list)
    for bad in (dict(n_vertices=0), dict(dim=4), dict(ring_slots=1), dict(ring_slots=256), dict(n_classes=0),
                dict(n_classes=9), dict(dt_ms=0.0), dict(n_edges=2 ** 32)):
        kw = dict(n_vertices=10, dim=2, n_edges=5, ring_slots=16, dt_ms=0.1, speed=0.1, n_classes=1)
        kw.update(bad)
        with pytest.raises(gn.GnError) as ei:
            gn.gn_query_workspace(gn.make_config(**kw))
        assert ei.value.code == gn.GN_E_INVALID_ARG
    with pytest.raises(gn.GnError):
        gn.gn_query_workspace(gn.make_config(10, 2, 5, 16, 0.1, 0.1, 1, obs_stride=10, trace_capacity_frames=0))


def test_no_cpu_fallback():
    """Without a CUDA device gn_create must fail loudly (GN_E_CUDA), never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    cfg = gn.make_config(4, 2, 0, 4, 0.1, 0.1, 1)
    with pytest.raises(gn.GnError) as ei:
        gn.gn_create(cfg, [dict.fromkeys(gn.binding.CLASS_FIELDS, 0.0)], None, np.zeros(5, np.uint64), None, None,
                     None, np.zeros(4, np.uint8))
    assert ei.value.code == gn.GN_E_CUDA
    # and the raw C entry point, given a non-device workspace, reports an error instead of running
    L = gn.lib()
    ws = np.zeros(gn.gn_query_workspace(cfg) + 256, dtype=np.uint8)
    base = (ws.ctypes.data + 255) & ~255
    tab = (gn.gn_class_params * 1)()
    h = C.c_void_p(None)
    rc = L.gn_create(C.byref(cfg), tab, None, np.zeros(5, np.uint64).ctypes.data_as(C.c_void_p), None, None, None,
                     np.zeros(4, np.uint8).ctypes.data_as(C.c_void_p), None, None, C.c_void_p(base), ws.nbytes - 256,
                     None, C.byref(h))
    assert rc in (gn.GN_E_CUDA, gn.GN_E_INVALID_ARG) and not h.value
    assert len(L.gn_last_error(None)) > 0


def test_product_never_imports_the_oracle():
    """The product path must not route through oracle/ (and the oracle must not import the product)."""
    for sub, banned in (("paper_0908_3934_b200", ("oracle", "gn_oracle", "pull_definition")),
                        ("oracle", ("paper_0908_3934_b200", "libgn.so", "gn.h")),
                        ("gn_inputs", ("paper_0908_3934_b200", "oracle"))):
        for dirpath, _, files in os.walk(os.path.join(ROOT, sub)):
            for f in files:
                if f.endswith((".py", ".cu", ".h", ".c")):
                    text = open(os.path.join(dirpath, f)).read()
                    for word in banned:
                        hits = [ln for ln in text.splitlines()
                                if re.search(r"^\s*(from|import|#include)\b.*" + re.escape(word), ln)]
                        assert not hits, (f, hits)
