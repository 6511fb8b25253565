"""Thin ctypes binding of include/gn.h -- argument marshalling only.

Every step of the path runs inside libgn.so's CUDA kernels; PyTorch supplies device memory (the
workspace and destination tensors) and the stream.  There is no CPU fallback: if the library is
missing it is built with nvcc, and if that fails the import raises.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build

GN_OK = 0
GN_E_INVALID_ARG, GN_E_BAD_GRAPH, GN_E_OVERFLOW_RISK = -1, -2, -3
GN_E_WORKSPACE_TOO_SMALL, GN_E_RANGE_EVICTED, GN_E_CUDA = -4, -5, -6
(GN_V, GN_W, GN_R, GN_CA, GN_REFR, GN_RING, GN_STEP, GN_COUNTERS, GN_DELAYS, GN_WEIGHTS_FX, GN_BIAS, GN_P, GN_ACC, GN_M,
 GN_H, GN_WEIGHTS, GN_FAULTS, GN_DRIVER) = range(18)
(GN_DRIVER_RING, GN_DRIVER_FUSED, GN_DRIVER_PERSISTENT, GN_DRIVER_QUEUE, GN_DRIVER_RESIDENT, GN_DRIVER_PLASTIC) = range(6)
GN_MODEL_IZHIKEVICH, GN_MODEL_HODGKIN_HUXLEY = 0, 1
GN_MAX_CLASSES = 8
GN_STATIC_MAX_VERTICES = 1048576
GN_DELIVER_AUTO, GN_DELIVER_RING, GN_DELIVER_QUEUE, GN_DELIVER_RESIDENT, GN_DELIVER_RING_STEPWISE = 0, 1, 2, 3, 4

# gn_class_params in declaration order; a class dict may omit psc_alpha, model and the Hodgkin-Huxley fields (0)
CLASS_FIELDS = ("a", "b", "c_reset", "d", "k2", "k1", "k0", "v_peak", "tau_syn_ms",
                "refractory_ms", "drive_rate_hz", "drive_kick", "psc_alpha",
                "model", "hh_c", "hh_g_na", "hh_g_k", "hh_g_l", "hh_e_na", "hh_e_k", "hh_e_l", "hh_v_rest") + \
    tuple(f"hh_{f}_{x}" for f in ("am", "bm", "ah", "bh", "an", "bn") for x in ("a", "v", "k"))
_OPTIONAL_FROM = CLASS_FIELDS.index("psc_alpha")


class gn_class_params(C.Structure):
    _fields_ = [(f, C.c_float) for f in CLASS_FIELDS]        # hh_am[3] ... hh_bn[3] laid out as consecutive floats


class gn_config(C.Structure):
    _fields_ = [("n_vertices", C.c_uint32), ("dim", C.c_uint32), ("n_edges", C.c_uint64),
                ("n_networks", C.c_uint32), ("ring_slots", C.c_uint32), ("dt_ms", C.c_float),
                ("speed", C.c_float), ("n_classes", C.c_uint32), ("tau_ca_ms", C.c_float),
                ("ca_jump", C.c_float), ("obs_gain", C.c_float), ("obs_offset", C.c_float),
                ("obs_sigma", C.c_float), ("obs_stride", C.c_uint32),
                ("raster_capacity_steps", C.c_uint32), ("trace_capacity_frames", C.c_uint32),
                ("seed", C.c_uint64), ("delivery_mode", C.c_uint32), ("queue_group", C.c_uint32),
                ("queue_capacity", C.c_uint64), ("stdp_alpha", C.c_float), ("stdp_beta", C.c_float)]


EXPORTS = ("gn_query_workspace", "gn_create", "gn_step", "gn_read_state", "gn_write_state",
           "gn_read_raster", "gn_observe", "gn_debug_words", "gn_debug_ceilings", "gn_debug_stream_ceilings", "gn_check_headroom_static", "gn_profile", "gn_profile_read", "gn_last_error",
           "gn_destroy")

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, u64, u32, i32, sz = C.c_void_p, C.c_uint64, C.c_uint32, C.c_int, C.c_size_t
        L.gn_query_workspace.argtypes = [C.POINTER(gn_config), C.POINTER(sz)]
        L.gn_create.argtypes = [C.POINTER(gn_config), C.POINTER(gn_class_params), vp, vp, vp, vp, vp, vp, vp, vp,
                                vp, sz, vp, C.POINTER(vp)]
        L.gn_step.argtypes = [vp, u64]
        L.gn_read_state.argtypes = [vp, i32, vp, sz, i32]
        L.gn_write_state.argtypes = [vp, i32, vp, sz, i32]
        L.gn_read_raster.argtypes = [vp, u64, u64, vp, sz, i32]
        L.gn_observe.argtypes = [vp, u64, u64, vp, sz, i32]
        L.gn_debug_words.argtypes = [vp, u64, u32, u64, u32, u32, vp]
        L.gn_debug_ceilings.argtypes = [vp, vp, sz, u32, vp]
        L.gn_debug_stream_ceilings.argtypes = [vp, vp, sz, vp]
        L.gn_check_headroom_static.argtypes = [vp, u32, u64, vp, vp, C.c_float, vp]
        L.gn_profile.argtypes = [vp, i32]
        L.gn_profile_read.argtypes = [vp, vp, vp]
        L.gn_last_error.argtypes = [vp]
        L.gn_last_error.restype = C.c_char_p
        L.gn_destroy.argtypes = [vp]
        for name in EXPORTS:
            if name != "gn_last_error":
                getattr(L, name).restype = i32
        _lib = L
    return _lib


class GnError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gn error {code}: {msg}")
        self.code = code


def _check(rc, handle=None):
    if rc != GN_OK:
        raise GnError(rc, lib().gn_last_error(handle).decode())


def _ptr(a):
    """Host numpy array, torch tensor (host or device) or None -> void pointer."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data_as(C.c_void_p)
    assert a.is_contiguous()
    return C.c_void_p(a.data_ptr())


def make_config(n_vertices, dim, n_edges, ring_slots, dt_ms, speed, n_classes, *, n_networks=1, tau_ca_ms=500.0,
                ca_jump=1.0, obs_gain=1.0, obs_offset=0.0, obs_sigma=0.0, obs_stride=0, raster_capacity_steps=0,
                trace_capacity_frames=0, seed=0, delivery_mode=GN_DELIVER_AUTO, queue_group=0,
                queue_capacity=0, stdp_alpha=0.0, stdp_beta=0.0) -> gn_config:
    return gn_config(n_vertices, dim, n_edges, n_networks, ring_slots, dt_ms, speed, n_classes, tau_ca_ms, ca_jump,
                     obs_gain, obs_offset, obs_sigma, obs_stride, raster_capacity_steps, trace_capacity_frames, seed,
                     delivery_mode, queue_group, queue_capacity, stdp_alpha, stdp_beta)


def gn_query_workspace(cfg: gn_config) -> int:
    n = C.c_size_t(0)
    _check(lib().gn_query_workspace(C.byref(cfg), C.byref(n)))
    return n.value


class GnNet:
    """Owner of one gn_net handle and of the torch workspace tensor behind it."""

    def __init__(self, handle, workspace, cfg, stream):
        self.handle, self.workspace, self.cfg, self.stream = handle, workspace, cfg, stream
        self.n, self.e, self.d = cfg.n_vertices, cfg.n_edges, cfg.ring_slots
        self.words = (self.n + 31) // 32

    def __del__(self):
        self.destroy()

    def destroy(self):
        if getattr(self, "handle", None):
            lib().gn_destroy(self.handle)
            self.handle = None
            self.workspace = None


def gn_create(cfg: gn_config, classes, positions, row_offsets, targets, weights, delays, vertex_class,
              bias=None, net_offsets=None, device="cuda:0", workspace=None) -> GnNet:
    """classes: sequence of dicts with CLASS_FIELDS.  Arrays: numpy (host) or torch tensors."""
    import torch
    if not torch.cuda.is_available():
        raise GnError(GN_E_CUDA, "no CUDA device: this library has no CPU fallback")
    dev = torch.device(device)
    need = gn_query_workspace(cfg)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=dev)
    tab = (gn_class_params * len(classes))(*[gn_class_params(*[c.get(f, 0.0) if i >= _OPTIONAL_FROM else c[f]
                                                               for i, f in enumerate(CLASS_FIELDS)]) for c in classes])
    handle = C.c_void_p(None)
    with torch.cuda.device(dev):
        stream = torch.cuda.current_stream(dev)
        rc = lib().gn_create(C.byref(cfg), tab, _ptr(positions), _ptr(row_offsets), _ptr(targets), _ptr(weights),
                             _ptr(delays), _ptr(vertex_class), _ptr(bias), _ptr(net_offsets),
                             C.c_void_p(workspace.data_ptr()), workspace.numel(), C.c_void_p(stream.cuda_stream),
                             C.byref(handle))
    _check(rc)
    return GnNet(handle, workspace, cfg, stream)


def gn_step(net: GnNet, n_steps: int) -> None:
    _check(lib().gn_step(net.handle, int(n_steps)), net.handle)


_STATE_DTYPE = {GN_V: np.float32, GN_W: np.float32, GN_R: np.float32, GN_CA: np.float32, GN_REFR: np.uint8,
                GN_RING: np.int32, GN_STEP: np.uint64, GN_COUNTERS: np.uint64, GN_DELAYS: np.uint8,
                GN_WEIGHTS_FX: np.int32, GN_BIAS: np.float32, GN_P: np.float32, GN_ACC: np.float32, GN_M: np.float32,
                GN_H: np.float32, GN_WEIGHTS: np.float32, GN_FAULTS: np.uint64,
                GN_DRIVER: np.uint32}


def _state_shape(net, which):
    return {GN_RING: (net.d, net.n), GN_STEP: (1,), GN_COUNTERS: (4,), GN_DELAYS: (net.e,),
            GN_WEIGHTS_FX: (net.e,), GN_WEIGHTS: (net.e,), GN_FAULTS: (2,), GN_DRIVER: (1,)}.get(which, (net.n,))


def gn_read_state(net: GnNet, which: int, out=None):
    """Host numpy result by default; pass a torch CUDA tensor as `out` for a device destination."""
    if out is None:
        out = np.empty(_state_shape(net, which), dtype=_STATE_DTYPE[which])
    is_dev = not isinstance(out, np.ndarray)
    nbytes = out.numel() * out.element_size() if is_dev else out.nbytes
    _check(lib().gn_read_state(net.handle, which, _ptr(out), nbytes, int(is_dev)), net.handle)
    return out


def gn_write_state(net: GnNet, which: int, src) -> None:
    is_dev = not isinstance(src, np.ndarray)
    if not is_dev:
        src = np.ascontiguousarray(src, dtype=_STATE_DTYPE[which])
    nbytes = src.numel() * src.element_size() if is_dev else src.nbytes
    _check(lib().gn_write_state(net.handle, which, _ptr(src), nbytes, int(is_dev)), net.handle)


def gn_read_raster(net: GnNet, t0: int, n_steps: int, out=None):
    if out is None:
        out = np.empty((n_steps, net.words), dtype=np.uint32)
    is_dev = not isinstance(out, np.ndarray)
    nbytes = out.numel() * out.element_size() if is_dev else out.nbytes
    _check(lib().gn_read_raster(net.handle, int(t0), int(n_steps), _ptr(out), nbytes, int(is_dev)), net.handle)
    return out


def gn_observe(net: GnNet, frame0: int, n_frames: int, out=None):
    if out is None:
        out = np.empty((n_frames, net.n), dtype=np.float32)
    is_dev = not isinstance(out, np.ndarray)
    nbytes = out.numel() * out.element_size() if is_dev else out.nbytes
    _check(lib().gn_observe(net.handle, int(frame0), int(n_frames), _ptr(out), nbytes, int(is_dev)), net.handle)
    return out


def gn_debug_words(seed: int, stream_id: int, idx: int, first_vertex: int, n: int, device="cuda:0"):
    import torch
    out = torch.empty(n, dtype=torch.int32, device=device)
    st = torch.cuda.current_stream(out.device)
    _check(lib().gn_debug_words(C.c_void_p(st.cuda_stream), seed, stream_id, idx, first_vertex, n,
                                C.c_void_p(out.data_ptr())))
    return out.cpu().numpy().view(np.uint32)


def gn_debug_ceilings(segment_edges: int, scratch_mb: int = 2048, device="cuda:0"):
    """(scattered reductions / s, gathers of `segment_edges`-edge segments + reductions / s) measured on the device."""
    import torch
    scratch = torch.empty(int(scratch_mb) << 20, dtype=torch.uint8, device=device)
    st = torch.cuda.current_stream(scratch.device)
    out = (C.c_double * 2)()
    with torch.cuda.device(scratch.device):
        _check(lib().gn_debug_ceilings(C.c_void_p(st.cuda_stream), C.c_void_p(scratch.data_ptr()), scratch.numel(),
                                       int(segment_edges), out))
    return float(out[0]), float(out[1])


def gn_debug_stream_ceilings(scratch_mb: int = 2048, device="cuda:0"):
    """(bytes/s read + written by a streaming read-modify-write that stays in L2, the same from HBM), measured on the device."""
    import torch
    scratch = torch.empty(int(scratch_mb) << 20, dtype=torch.uint8, device=device)
    st = torch.cuda.current_stream(scratch.device)
    out = (C.c_double * 2)()
    with torch.cuda.device(scratch.device):
        _check(lib().gn_debug_stream_ceilings(C.c_void_p(st.cuda_stream), C.c_void_p(scratch.data_ptr()), scratch.numel(), out))
    return float(out[0]), float(out[1])


def gn_check_headroom_static(n_vertices: int, targets, weights, largest_kick: float, out=None):
    """gn.h gn_check_headroom_static: torch CUDA tensors in (uint32-as-int32 targets, float32 weights), a 2-word int32
    CUDA tensor out (made here when None -- torch's allocator, not the library's; pass your own where you cannot
    allocate).  Asynchronous on torch's current stream of that device; returns `out`."""
    import torch
    if out is None:
        out = torch.empty(2, dtype=torch.int32, device=targets.device)
    assert targets.is_cuda and weights.is_cuda and out.is_cuda and targets.numel() == weights.numel()
    assert targets.element_size() == 4 and weights.dtype == torch.float32 and out.element_size() == 4 and out.numel() >= 2
    with torch.cuda.device(targets.device):
        st = torch.cuda.current_stream(targets.device)
        _check(lib().gn_check_headroom_static(C.c_void_p(st.cuda_stream), int(n_vertices), int(targets.numel()),
                                              _ptr(targets), _ptr(weights), float(largest_kick), _ptr(out)))
    return out


def gn_profile(net: GnNet, enable: bool) -> None:
    _check(lib().gn_profile(net.handle, int(bool(enable))), net.handle)


def gn_profile_read(net: GnNet):
    """-> (ms[4] summed device time of update / delivery (queue mode: spike logging) / observation / fold, launches[5])."""
    ms = np.zeros(4, dtype=np.float64)
    n = np.zeros(5, dtype=np.uint64)
    _check(lib().gn_profile_read(net.handle, _ptr(ms), _ptr(n)), net.handle)
    return ms, n


def gn_destroy(net: GnNet) -> None:
    net.destroy()


def create_from_inputs(net_in, cfg_in, *, delays=None, bias=None, raster_capacity_steps=0,
                       trace_capacity_frames=0, device="cuda:0", delivery_mode=GN_DELIVER_AUTO, queue_group=0,
                       queue_capacity=0, stdp_alpha=0.0, stdp_beta=0.0) -> GnNet:
    """Convenience: build from a gn_inputs.Network + config dict (marshalling only)."""
    obs = int(cfg_in.get("obs_stride", 0))
    cfg = make_config(net_in.n_vertices, net_in.dim, net_in.n_edges, cfg_in["ring_slots"], cfg_in["dt_ms"],
                      cfg_in["speed"], len(cfg_in["classes"]), n_networks=net_in.n_networks,
                      tau_ca_ms=cfg_in["tau_ca_ms"], ca_jump=cfg_in["ca_jump"], obs_gain=cfg_in["obs_gain"],
                      obs_offset=cfg_in["obs_offset"], obs_sigma=cfg_in["obs_sigma"], obs_stride=obs,
                      raster_capacity_steps=raster_capacity_steps,
                      trace_capacity_frames=trace_capacity_frames if obs else 0, seed=cfg_in["seed"],
                      delivery_mode=delivery_mode, queue_group=queue_group, queue_capacity=queue_capacity,
                      stdp_alpha=stdp_alpha, stdp_beta=stdp_beta)
    return gn_create(cfg, cfg_in["classes"], net_in.positions, net_in.row_offsets, net_in.targets, net_in.weights,
                     None if delays is None else np.ascontiguousarray(delays, dtype=np.uint8),
                     net_in.vertex_class,
                     None if bias is None else np.ascontiguousarray(bias, dtype=np.float32),
                     net_in.net_offsets, device=device)
