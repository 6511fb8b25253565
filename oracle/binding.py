"""ctypes binding of oracle/gn_oracle.c (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gn_oracle.c")
_SO = os.path.join(_HERE, "libgn_oracle.so")
_lib = None

HH_RATES = ("am", "bm", "ah", "bh", "an", "bn")      # alpha_m, beta_m, alpha_h, beta_h, alpha_n, beta_n
CLASS_FIELDS = ("a", "b", "c_reset", "d", "k2", "k1", "k0", "v_peak", "tau_syn_ms",
                "refractory_ms", "drive_rate_hz", "drive_kick", "psc_alpha",
                "model", "hh_c", "hh_g_na", "hh_g_k", "hh_g_l", "hh_e_na", "hh_e_k", "hh_e_l", "hh_v_rest") + \
    tuple(f"hh_{f}_{x}" for f in HH_RATES for x in ("a", "v", "k"))
OPTIONAL_FROM = CLASS_FIELDS.index("psc_alpha")      # psc_alpha and every Hodgkin-Huxley field may be omitted: 0
V, W, R, CA, P, HM, HH = 0, 1, 2, 3, 4, 5, 6


def build_lib(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-o", _SO, _SRC, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build_lib())
        vp, u32, u64, f32, i32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_float, C.c_int
        L.orc_philox4x32_10.argtypes = [vp, vp, vp]
        L.orc_word.restype = u32
        L.orc_word.argtypes = [u64, u32, u32, u64]
        L.orc_gauss.restype = C.c_double
        L.orc_gauss.argtypes = [u64, u32, u64]
        L.orc_delay_steps.restype = u32
        L.orc_delay_steps.argtypes = [vp, vp, u32, f32, f32]
        L.orc_quantise.restype = C.c_int64
        L.orc_quantise.argtypes = [f32]
        L.orc_drive_threshold.restype = u32
        L.orc_drive_threshold.argtypes = [f32, f32]
        L.orc_keep.restype = C.c_double
        L.orc_keep.argtypes = [f32, f32]
        L.orc_refractory_steps.restype = u32
        L.orc_refractory_steps.argtypes = [f32, f32]
        L.orc_hh_rate.restype = C.c_double
        L.orc_hh_rate.argtypes = [i32, C.c_double, C.c_double, C.c_double, C.c_double]
        L.orc_hh_rate32.restype = f32
        L.orc_hh_rate32.argtypes = [i32, f32, f32, f32, f32]
        L.orc_exp32.restype = f32
        L.orc_exp32.argtypes = [f32]
        L.orc_create.restype = vp
        L.orc_create.argtypes = [u32, u32, u64, u32, f32, f32, u32, vp, vp, vp, vp, vp, vp, vp, vp,
                                 f32, f32, f32, f32, f32, u32, u64, u32]
        L.orc_destroy.argtypes = [vp]
        L.orc_step.restype = i32
        L.orc_step.argtypes = [vp, u64, i32]
        for name in ("orc_get_state", "orc_set_state"):
            getattr(L, name).restype = i32
            getattr(L, name).argtypes = [vp, i32, vp]
        for name in ("orc_get_refr", "orc_get_ring", "orc_get_consumed", "orc_get_delays",
                     "orc_get_w_fx", "orc_get_counters"):
            getattr(L, name).restype = None
            getattr(L, name).argtypes = [vp, vp]
        L.orc_enable_stdp.restype = i32
        L.orc_enable_stdp.argtypes = [vp, f32, f32]
        L.orc_get_weights.restype = None
        L.orc_get_weights.argtypes = [vp, vp]
        L.orc_get_raster.restype = i32
        L.orc_get_raster.argtypes = [vp, u64, u64, vp]
        L.orc_get_trace.restype = i32
        L.orc_get_trace.argtypes = [vp, u64, u64, vp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def class_table(classes) -> np.ndarray:
    # psc_alpha (0 = exponential PSC, eq. 26; 1 = alpha-function, eq. 27-30) and the Hodgkin-Huxley fields (model = 1)
    # may be omitted: 0
    return np.array([[c.get(f, 0.0) if i >= OPTIONAL_FROM else c[f] for i, f in enumerate(CLASS_FIELDS)]
                     for c in classes], dtype=np.float32)


class Oracle:
    """One simulated network.  mode: "fp64" (the definition) or "fp32" (fp32-faithful)."""

    def __init__(self, net, cfg, mode="fp64", delays=None, bias=None, threads=1, stdp=None):
        """stdp = (alpha per ms, beta per ms): plastic weights (eq. 32-33), from step 0."""
        L = lib()
        self.n = int(net.n_vertices)
        self.D = int(cfg["ring_slots"])
        self.E = int(net.n_edges)
        self.words = (self.n + 31) // 32
        self.threads = int(threads)
        self._keep = dict(
            cls=class_table(cfg["classes"]),
            pos=np.ascontiguousarray(net.positions, dtype=np.float32),
            row=np.ascontiguousarray(net.row_offsets, dtype=np.uint64),
            tgt=np.ascontiguousarray(net.targets, dtype=np.uint32),
            w=np.ascontiguousarray(net.weights, dtype=np.float32),
            dly=None if delays is None else np.ascontiguousarray(delays, dtype=np.uint8),
            vc=np.ascontiguousarray(net.vertex_class, dtype=np.uint8),
            bias=None if bias is None else np.ascontiguousarray(bias, dtype=np.float32))
        k = self._keep
        self._h = L.orc_create(self.n, int(net.dim), self.E, self.D, cfg["dt_ms"], cfg["speed"],
                               len(cfg["classes"]), _p(k["cls"]), _p(k["pos"]), _p(k["row"]),
                               _p(k["tgt"]), _p(k["w"]), _p(k["dly"]), _p(k["vc"]), _p(k["bias"]),
                               cfg["tau_ca_ms"], cfg["ca_jump"], cfg["obs_gain"], cfg["obs_offset"],
                               cfg["obs_sigma"], int(cfg["obs_stride"]), int(cfg["seed"]),
                               {"fp64": 0, "fp32": 1}[mode])
        if not self._h:
            raise ValueError("orc_create rejected the network (row offsets / target range / delay)")
        if stdp is not None and L.orc_enable_stdp(self._h, float(stdp[0]), float(stdp[1])) != 0:
            raise ValueError("orc_enable_stdp refused (beta < 0, or out of memory)")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def step(self, n_steps=1):
        rc = lib().orc_step(self._h, int(n_steps), self.threads)
        if rc:
            raise OverflowError(f"orc_step failed ({rc}): ring slot outside int32" if rc == -2 else f"orc_step {rc}")

    def state(self, which):
        out = np.empty(self.n, dtype=np.float64)
        assert lib().orc_get_state(self._h, which, _p(out)) == 0
        return out

    def set_state(self, which, values):
        v = np.ascontiguousarray(np.broadcast_to(np.asarray(values, dtype=np.float64), (self.n,)))
        assert lib().orc_set_state(self._h, which, _p(v)) == 0

    def refr(self):
        out = np.empty(self.n, dtype=np.uint32)
        lib().orc_get_refr(self._h, _p(out))
        return out

    def ring(self):
        out = np.empty((self.D, self.n), dtype=np.int64)
        lib().orc_get_ring(self._h, _p(out))
        return out

    def consumed(self):
        out = np.empty(self.n, dtype=np.int64)
        lib().orc_get_consumed(self._h, _p(out))
        return out

    def delays(self):
        out = np.empty(self.E, dtype=np.uint32)
        lib().orc_get_delays(self._h, _p(out))
        return out

    def w_fx(self):
        out = np.empty(self.E, dtype=np.int64)
        lib().orc_get_w_fx(self._h, _p(out))
        return out

    def weights(self):
        """w_ij(t) of every edge in the caller's (CSR) edge order."""
        out = np.empty(self.E, dtype=np.float64)
        lib().orc_get_weights(self._h, _p(out))
        return out

    def counters(self):
        out = np.empty(7, dtype=np.uint64)
        lib().orc_get_counters(self._h, _p(out))
        m = out[5:7].view(np.int64)
        return dict(steps=int(out[0]), spikes=int(out[1]), delivered=int(out[2]), kicks=int(out[3]),
                    frames=int(out[4]), mass_delivered=int(m[0]), mass_consumed=int(m[1]))

    def raster(self, t0=0, n_steps=None):
        n_steps = self.counters()["steps"] - t0 if n_steps is None else n_steps
        out = np.empty((n_steps, self.words), dtype=np.uint32)
        assert lib().orc_get_raster(self._h, int(t0), int(n_steps), _p(out)) == 0
        return out

    def raster_bool(self, t0=0, n_steps=None):
        bits = np.unpackbits(self.raster(t0, n_steps).view(np.uint8), axis=1, bitorder="little")
        return bits[:, :self.n].astype(bool)

    def trace(self, f0=0, n_frames=None):
        n_frames = self.counters()["frames"] - f0 if n_frames is None else n_frames
        out = np.empty((n_frames, self.n), dtype=np.float64)
        assert lib().orc_get_trace(self._h, int(f0), int(n_frames), _p(out)) == 0
        return out
