"""ctypes front end of gn_inputs.c (see that file's header for the recipe)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gn_inputs.c")
_SO = os.path.join(_HERE, "libgn_inputs.so")
_lib = None


def build_lib(force: bool = False) -> str:
    """Compile gn_inputs.c with gcc if the shared object is missing or stale."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build_lib())
        lib.gni_derive_seed.restype = C.c_uint64
        lib.gni_derive_seed.argtypes = [C.c_uint64, C.c_uint64]
        lib.gni_positions.restype = None
        lib.gni_positions.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_double, C.c_void_p]
        lib.gni_classes.restype = None
        lib.gni_classes.argtypes = [C.c_uint64, C.c_uint32, C.c_double, C.c_void_p]
        lib.gni_degrees.restype = C.c_int
        lib.gni_degrees.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, C.c_double, C.c_void_p,
                                    C.c_uint32, C.c_double, C.c_double, C.c_double, C.c_void_p,
                                    C.c_void_p]
        lib.gni_fill.restype = C.c_int
        lib.gni_fill.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, C.c_double, C.c_void_p,
                                 C.c_uint32, C.c_double, C.c_double, C.c_double, C.c_void_p,
                                 C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


@dataclass
class Network:
    """Plain arrays at the C-ABI boundary's types (include/gn.h gn_create)."""
    n_vertices: int
    dim: int
    n_networks: int
    positions: np.ndarray      # float32 [N][dim]
    row_offsets: np.ndarray    # uint64 [N+1], CSR by source
    targets: np.ndarray        # uint32 [E]
    weights: np.ndarray        # float32 [E]
    vertex_class: np.ndarray   # uint8 [N]
    net_offsets: np.ndarray | None = None   # uint32 [n_networks+1]
    meta: dict = field(default_factory=dict)

    @property
    def n_edges(self) -> int:
        return int(self.row_offsets[-1])


def geometric_network(seed: int, n_per: int, dim: int, side: float, radius: float, *,
                      kind: int = 0, p0: float = 1.0, lam: float = 1.0, frac_inh: float = 0.0,
                      w_exc=(0.0, 1.0), w_inh=(-1.0, 0.0), n_networks: int = 1) -> Network:
    """Distance-probability geometric graph(s); `n_networks` > 1 concatenates independent
    networks (block-diagonal CSR, global target ids), each seeded by derive(seed, b)."""
    lib = _load()
    n = n_per * n_networks
    if n_networks == 1:
        seeds = np.array([seed], dtype=np.uint64)
    else:
        seeds = np.array([lib.gni_derive_seed(seed, b) for b in range(n_networks)], dtype=np.uint64)
    pos = np.empty((n, dim), dtype=np.float32)
    cls = np.empty(n, dtype=np.uint8)
    for b in range(n_networks):
        lib.gni_positions(int(seeds[b]), n_per, dim, side, _p(pos[b * n_per:]))
        lib.gni_classes(int(seeds[b]), n_per, frac_inh, _p(cls[b * n_per:]))
    deg = np.empty(n, dtype=np.uint32)
    rc = lib.gni_degrees(n_networks, n_per, dim, side, _p(pos), kind, radius, p0, lam, _p(seeds), _p(deg))
    if rc:
        raise RuntimeError(f"gni_degrees failed ({rc})")
    row = np.zeros(n + 1, dtype=np.uint64)
    np.cumsum(deg, dtype=np.uint64, out=row[1:])
    e = int(row[-1])
    tgt = np.empty(max(e, 1), dtype=np.uint32)[:e]
    w = np.empty(max(e, 1), dtype=np.float32)[:e]
    wr = np.array([w_exc[0], w_exc[1], w_inh[0], w_inh[1]], dtype=np.float64)
    rc = lib.gni_fill(n_networks, n_per, dim, side, _p(pos), kind, radius, p0, lam, _p(seeds),
                      _p(cls), _p(wr), _p(row), _p(tgt), _p(w))
    if rc:
        raise RuntimeError(f"gni_fill failed ({rc})")
    net_off = None
    if n_networks > 1:
        net_off = (np.arange(n_networks + 1, dtype=np.uint64) * n_per).astype(np.uint32)
    return Network(n, dim, n_networks, pos, row, tgt, w, cls, net_off)
