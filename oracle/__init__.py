"""ctypes access to oracle/soc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It holds no arithmetic of its own: every number comes out of the plain C
file next to it (fp64, single-threaded per call).  `simulate(..., threads=k)` only splits the
package-id range over k concurrent calls with private accumulators that are summed at the end
(SURVEY.md 8d.5); the per-package arithmetic is untouched by it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "soc_oracle.c")
_LIB = os.path.join(_HERE, "libsoc_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Sources(C.Structure):
    _fields_ = [("bg_intensity", C.c_double), ("n_point", C.c_int32), ("ps_pos", C.c_void_p),
                ("ps_lum", C.c_void_p), ("n_bg", C.c_int64), ("beam", C.c_void_p)]


class _Result(C.Structure):
    _fields_ = [("emitted", C.c_double), ("escaped", C.c_double), ("absorbed", C.c_double),
                ("cell_steps", C.c_uint64), ("scatterings", C.c_uint64), ("terminated", C.c_uint64)]


REPLAY_DTYPE = np.dtype([("hash", "<u8"), ("steps", "<u4"), ("scatters", "<u4"), ("e_escaped", "<f8")])
TRACE_DTYPE = np.dtype([("pkg", "<i8"), ("gid", "<i8"), ("level", "<i4"), ("kind", "<i4"),
                        ("p0", "<f8", (3,)), ("p1", "<f8", (3,)), ("ds", "<f8"), ("tau_sca", "<f8"),
                        ("tau_drawn", "<f8")])

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.soc_oracle_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.soc_oracle_stream_block.argtypes = [C.c_uint64, C.c_int32, C.c_int64, C.c_uint32, C.c_void_p]
        L.soc_oracle_uniform.argtypes = [C.c_uint32]
        L.soc_oracle_uniform.restype = C.c_double
        L.soc_oracle_hg_cos.argtypes = [C.c_double, C.c_double]
        L.soc_oracle_hg_cos.restype = C.c_double
        L.soc_oracle_rotate.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p]
        L.soc_oracle_grid_create.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p,
                                             C.c_void_p, C.c_void_p]
        L.soc_oracle_grid_create.restype = C.c_void_p
        L.soc_oracle_grid_destroy.argtypes = [C.c_void_p]
        L.soc_oracle_emit_background.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                                                 C.c_void_p, C.c_void_p]
        L.soc_oracle_emit_point.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.soc_oracle_simulate.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_int32,
                                          C.POINTER(_Sources), C.c_int64, C.c_uint64, C.c_double,
                                          C.c_int64, C.c_int64, C.c_void_p, C.POINTER(_Result),
                                          C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
        L.soc_oracle_simulate.restype = C.c_int
        L.soc_oracle_simulate_f32state.argtypes = L.soc_oracle_simulate.argtypes
        L.soc_oracle_simulate_f32state.restype = C.c_int
        L.soc_oracle_trapezoid_weights.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
        L.soc_oracle_update_temperatures.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p,
                                                     C.c_int32, C.c_double, C.c_double, C.c_void_p]
        L.soc_oracle_sizeof_replay.restype = C.c_int64
        L.soc_oracle_sizeof_trace.restype = C.c_int64
        L.soc_oracle_grid_parent.argtypes = [C.c_void_p, C.c_int32]
        L.soc_oracle_grid_parent.restype = C.c_void_p
        assert L.soc_oracle_sizeof_replay() == REPLAY_DTYPE.itemsize
        assert L.soc_oracle_sizeof_trace() == TRACE_DTYPE.itemsize
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().soc_oracle_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def stream_block(seed, ifreq, pkg, block):
    out = np.zeros(4, dtype=np.uint32)
    lib().soc_oracle_stream_block(int(seed), int(ifreq), int(pkg), int(block), _p(out))
    return out


def uniform(word):
    return lib().soc_oracle_uniform(int(word))


def hg_cos(g, u):
    return lib().soc_oracle_hg_cos(float(g), float(u))


def rotate(d, cost, phi):
    d = np.ascontiguousarray(d, dtype=np.float64)
    out = np.zeros(3)
    lib().soc_oracle_rotate(_p(d), float(cost), float(phi), _p(out))
    return out


def emit_background(nx, ny, nz, u):
    u = np.ascontiguousarray(u, dtype=np.float64)
    ijk = np.zeros(3, dtype=np.int32)
    f = np.zeros(3)
    d = np.zeros(3)
    lib().soc_oracle_emit_background(nx, ny, nz, _p(u), _p(ijk), _p(f), _p(d))
    return ijk, f, d


def emit_point(pos, u):
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    u = np.ascontiguousarray(u, dtype=np.float64)
    ijk = np.zeros(3, dtype=np.int32)
    f = np.zeros(3)
    d = np.zeros(3)
    lib().soc_oracle_emit_point(_p(pos), _p(u), _p(ijk), _p(f), _p(d))
    return ijk, f, d


def trapezoid_weights(freq):
    f = np.ascontiguousarray(freq, dtype=np.float64)
    w = np.zeros_like(f)
    lib().soc_oracle_trapezoid_weights(_p(f), len(f), _p(w))
    return w


@dataclass
class Result:
    emitted: float = 0.0
    escaped: float = 0.0
    absorbed: float = 0.0
    cell_steps: int = 0
    scatterings: int = 0
    terminated: int = 0


class Grid:
    """Owns one soc_oracle_grid.  n_cells[l], flattened level-major rho (fp32) and child (int32)."""

    def __init__(self, nx, ny, nz, n_cells, rho, child=None):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.n_cells = np.ascontiguousarray(n_cells, dtype=np.int64)
        self.n_levels = len(self.n_cells)
        self.rho = np.ascontiguousarray(rho, dtype=np.float32)
        self.child = None if child is None else np.ascontiguousarray(child, dtype=np.int32)
        self.n_total = int(self.n_cells.sum())
        assert self.rho.size == self.n_total
        self._h = lib().soc_oracle_grid_create(self.nx, self.ny, self.nz, self.n_levels, _p(self.n_cells),
                                                _p(self.rho), _p(self.child))
        if not self._h:
            raise ValueError("soc_oracle_grid_create: inconsistent hierarchy")

    def __del__(self):
        try:
            if getattr(self, "_h", None):
                lib().soc_oracle_grid_destroy(self._h)
                self._h = None
        except Exception:       # interpreter shutdown
            pass

    def parent(self, level):
        """Reverse links of `level` (1-based, > 1): one entry per octet."""
        n = int(self.n_cells[level - 1]) // 8
        ptr = lib().soc_oracle_grid_parent(self._h, level)
        return np.ctypeslib.as_array(C.cast(ptr, C.POINTER(C.c_int32)), shape=(n,)).copy()


def _sources_struct(src, keep):
    s = _Sources()
    s.bg_intensity = float(src.get("bg_intensity", 0.0))
    pos = src.get("ps_pos")
    lum = src.get("ps_lum")
    s.n_point = 0 if pos is None else len(np.atleast_2d(pos))
    if s.n_point:
        pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
        lum = np.ascontiguousarray(lum, dtype=np.float64).reshape(-1)
        keep += [pos, lum]
        s.ps_pos, s.ps_lum = pos.ctypes.data, lum.ctypes.data
    s.n_bg = int(src.get("n_bg", -1))
    beam = src.get("beam")
    if beam is not None:
        beam = np.ascontiguousarray(beam, dtype=np.float64).reshape(6)
        keep.append(beam)
        s.beam = beam.ctypes.data
    return s


def simulate(grid: Grid, kabs, ksca, g, ifreq, sources: dict, n_packages, seed, weight=1.0,
             pkg_begin=0, pkg_count=None, absorbed=None, want_replay=False, trace_cap=0, threads=1,
             f32state=False):
    """Run packages [pkg_begin, pkg_begin+pkg_count).  Returns (absorbed, Result, replay, trace).

    sources: dict(bg_intensity=, ps_pos=, ps_lum=, n_bg=, beam=).  `absorbed` is accumulated into.
    f32state=False: soc_oracle_simulate, THE oracle (fp64 throughout).  f32state=True: the named variant
    soc_oracle_simulate_f32state (state snapped to fp32 at every store; replay-parity tests only).
    """
    L = lib()
    entry = L.soc_oracle_simulate_f32state if f32state else L.soc_oracle_simulate
    if pkg_count is None:
        pkg_count = n_packages - pkg_begin
    if absorbed is None:
        absorbed = np.zeros(grid.n_total, dtype=np.float64)
    assert absorbed.dtype == np.float64 and absorbed.size == grid.n_total and absorbed.flags.c_contiguous
    replay = np.zeros(pkg_count, dtype=REPLAY_DTYPE) if want_replay else None
    trace = np.zeros(trace_cap, dtype=TRACE_DTYPE) if trace_cap else None
    keep = []
    s = _sources_struct(sources, keep)

    def run(b, n, acc, rep, trc):
        r = _Result()
        nt = C.c_int64(0)
        rc = entry(grid._h, float(kabs), float(ksca), float(g), int(ifreq), C.byref(s),
                   int(n_packages), int(seed), float(weight), int(b), int(n), _p(acc),
                   C.byref(r), _p(rep), _p(trc), 0 if trc is None else len(trc), C.byref(nt))
        if rc != 0:
            raise ValueError("soc_oracle_simulate: bad argument")
        return r, nt.value

    threads = max(1, min(int(threads), max(1, pkg_count)))
    if threads == 1 or trace is not None:
        r, nt = run(pkg_begin, pkg_count, absorbed, replay, trace)
        res = Result(r.emitted, r.escaped, r.absorbed, r.cell_steps, r.scatterings, r.terminated)
        return absorbed, res, replay, (None if trace is None else trace[:nt])

    bounds = np.linspace(0, pkg_count, threads + 1).astype(np.int64)
    accs = [np.zeros(grid.n_total, dtype=np.float64) for _ in range(threads)]

    def job(i):
        b, e = int(bounds[i]), int(bounds[i + 1])
        rep = None if replay is None else replay[b:e]
        return run(pkg_begin + b, e - b, accs[i], rep, None)[0]

    with ThreadPoolExecutor(threads) as ex:
        rs = list(ex.map(job, range(threads)))
    for a in accs:
        absorbed += a
    res = Result(sum(r.emitted for r in rs), sum(r.escaped for r in rs), sum(r.absorbed for r in rs),
                 sum(r.cell_steps for r in rs), sum(r.scatterings for r in rs), sum(r.terminated for r in rs))
    return absorbed, res, replay, None


def update_temperatures(grid: Grid, absorbed, scale, table_T, E_min, E_max):
    absorbed = np.ascontiguousarray(absorbed, dtype=np.float64)
    table_T = np.ascontiguousarray(table_T, dtype=np.float32)
    out = np.zeros(grid.n_total, dtype=np.float32)
    lib().soc_oracle_update_temperatures(grid._h, _p(absorbed), float(scale), _p(table_T), len(table_T),
                                         float(E_min), float(E_max), _p(out))
    return out
