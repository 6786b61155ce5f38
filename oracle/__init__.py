"""ctypes access to oracle/soc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The package walk, the deposits, the temperature lookup and the maps (rows a1-a11,
f2) are computed by the plain C file next to it (fp64, single-threaded per call); `simulate(...,
threads=k)` only splits the package-id range over k concurrent calls with private accumulators that
are summed at the end and leaves the per-package arithmetic untouched.  What is
written here in numpy: the host loop of the iterated run (`iterate`: running-mean reference field,
ALI update, rows f1 / f3) and the stochastic-heating solver (`stochastic_*`, row f4: dense fp64 solve).
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
                ("ps_lum", C.c_void_p), ("n_bg", C.c_int64), ("beam", C.c_void_p),
                ("n_dust", C.c_int64), ("dust_T", C.c_void_p), ("dust_count", C.c_void_p),
                ("dust_freq_hz", C.c_double), ("dust_self", C.c_void_p)]


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
        L.soc_oracle_update_temperatures_ali.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                                         C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_void_p]
        L.soc_oracle_planck.argtypes = [C.c_double, C.c_double]
        L.soc_oracle_planck.restype = C.c_double
        L.soc_oracle_cell_luminosity.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.soc_oracle_emission_counts.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_int32, C.c_int64,
                                                 C.c_int32, C.c_void_p]
        L.soc_oracle_emission_counts.restype = C.c_int64
        L.soc_oracle_emit_cell.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.soc_oracle_make_map.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p,
                                          C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_void_p]
        L.soc_oracle_make_map.restype = None
        L.soc_oracle_dust_stride.argtypes = [C.c_int64]
        L.soc_oracle_dust_stride.restype = C.c_int64
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
    if src.get("dust_count") is not None:             # f1: dust re-emission (the last n_dust package ids)
        T = np.ascontiguousarray(src["dust_T"], dtype=np.float32)
        cnt = np.ascontiguousarray(src["dust_count"], dtype=np.int32)
        keep += [T, cnt]
        s.dust_T, s.dust_count = T.ctypes.data, cnt.ctypes.data
        s.n_dust = int(cnt.sum(dtype=np.int64))
        s.dust_freq_hz = float(src["dust_freq_hz"])
        if src.get("dust_self") is not None:          # f3: in-cell absorption of the cells' own packages, accumulated into
            a = src["dust_self"]
            assert a.dtype == np.float64 and a.flags.c_contiguous
            s.dust_self = a.ctypes.data
    return s


def simulate(grid: Grid, kabs, ksca, g, ifreq, sources: dict, n_packages, seed, weight=1.0,
             pkg_begin=0, pkg_count=None, absorbed=None, want_replay=False, trace_cap=0, threads=1,
             f32state=False):
    """Run packages [pkg_begin, pkg_begin+pkg_count).  Returns (absorbed, Result, replay, trace).

    sources: dict(bg_intensity=, ps_pos=, ps_lum=, n_bg=, beam=, dust_T=, dust_count=, dust_freq_hz=, dust_self=).
    `absorbed` (and `dust_self`, if given) are accumulated into.
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

    def run(b, n, acc, rep, trc, self_acc=None):
        r = _Result()
        nt = C.c_int64(0)
        st = s
        if self_acc is not None:                       # a thread's own in-cell accumulator
            st = _Sources.from_buffer_copy(s)
            st.dust_self = self_acc.ctypes.data
        rc = entry(grid._h, float(kabs), float(ksca), float(g), int(ifreq), C.byref(st),
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
    want_self = sources.get("dust_self") is not None and sources.get("dust_count") is not None
    selfs = [np.zeros(grid.n_total, dtype=np.float64) for _ in range(threads)] if want_self else None

    def job(i):
        b, e = int(bounds[i]), int(bounds[i + 1])
        rep = None if replay is None else replay[b:e]
        return run(pkg_begin + b, e - b, accs[i], rep, None, selfs[i] if want_self else None)[0]

    with ThreadPoolExecutor(threads) as ex:
        rs = list(ex.map(job, range(threads)))
    for a in accs:
        absorbed += a
    if want_self:
        for a in selfs:
            sources["dust_self"] += a
    res = Result(sum(r.emitted for r in rs), sum(r.escaped for r in rs), sum(r.absorbed for r in rs),
                 sum(r.cell_steps for r in rs), sum(r.scatterings for r in rs), sum(r.terminated for r in rs))
    return absorbed, res, replay, None


def planck(nu, T):
    return lib().soc_oracle_planck(float(nu), float(T))


def cell_luminosity(grid: Grid, kabs, freq_hz, T):
    """L_c = 4 pi kabs rho_c h^3 B_nu(T_c) per cell (0 for parents, empty leaves, T <= 0)."""
    T = np.ascontiguousarray(T, dtype=np.float32)
    out = np.zeros(grid.n_total, dtype=np.float64)
    lib().soc_oracle_cell_luminosity(grid._h, float(kabs), float(freq_hz), _p(T), _p(out))
    return out


def emission_counts(grid: Grid, kabs, freq_hz, T, mode, n_request, cap=10000):
    """Packages per cell: mode 'uniform' (same number from every emitting cell) or 'weighted' (in proportion to the
    cell's luminosity, capped).  Returns int32[n_total]."""
    T = np.ascontiguousarray(T, dtype=np.float32)
    out = np.zeros(grid.n_total, dtype=np.int32)
    n = lib().soc_oracle_emission_counts(grid._h, float(kabs), float(freq_hz), _p(T), {"uniform": 0, "weighted": 1}[mode],
                                         int(n_request), int(cap), _p(out))
    if n < 0:
        raise ValueError("soc_oracle_emission_counts: bad argument")
    assert n == int(out.sum(dtype=np.int64))
    return out


def emit_cell(u):
    u = np.ascontiguousarray(u, dtype=np.float64)
    f, d = np.zeros(3), np.zeros(3)
    lib().soc_oracle_emit_cell(_p(u), _p(f), _p(d))
    return f, d


def update_temperatures_ali(grid: Grid, absorbed, self_abs, emitted, scale, table_T, E_min, E_max):
    a, sa, em = (np.ascontiguousarray(x, dtype=np.float64) for x in (absorbed, self_abs, emitted))
    table_T = np.ascontiguousarray(table_T, dtype=np.float32)
    out = np.zeros(grid.n_total, dtype=np.float32)
    lib().soc_oracle_update_temperatures_ali(grid._h, _p(a), _p(sa), _p(em), float(scale), _p(table_T), len(table_T),
                                             float(E_min), float(E_max), _p(out))
    return out


def update_temperatures(grid: Grid, absorbed, scale, table_T, E_min, E_max):
    absorbed = np.ascontiguousarray(absorbed, dtype=np.float64)
    table_T = np.ascontiguousarray(table_T, dtype=np.float32)
    out = np.zeros(grid.n_total, dtype=np.float32)
    lib().soc_oracle_update_temperatures(grid._h, _p(absorbed), float(scale), _p(table_T), len(table_T),
                                         float(E_min), float(E_max), _p(out))
    return out


def make_map(grid: Grid, kabs, ksca, freq_hz, T, ex, ey, direction, centre, npx, npy, pixel):
    """Surface-brightness map (row f2): float64 [npy, npx]."""
    T = np.ascontiguousarray(T, dtype=np.float32)
    v = [np.ascontiguousarray(x, dtype=np.float64).reshape(3) for x in (ex, ey, direction, centre)]
    out = np.zeros((int(npy), int(npx)), dtype=np.float64)
    lib().soc_oracle_make_map(grid._h, float(kabs), float(ksca), float(freq_hz), _p(T), _p(v[0]), _p(v[1]), _p(v[2]), _p(v[3]),
                              int(npx), int(npy), float(pixel), _p(out))
    return out


def dust_stride(n_dust):
    return int(lib().soc_oracle_dust_stride(int(n_dust)))


def iterate(grid: Grid, freq_hz, kabs, ksca, g, const_sources, n_const, n_request, seed, t_scale, table_T, E_min, E_max,
            mode="weighted", cap=10000, reference_field=True, ref_start=1, ali=False, update_T=True, T_start=None,
            threads=1, f32state=False):
    """Iterated run with dust re-emission (rows f1, f3; readings F4-F6 of DESIGN.md), step by step:

      iteration 0   constant sources only (background, point sources), n_const packages per frequency, seed:
                    A_const = sum_f w_f A_f;  T = table(A_const)   (T_start overrides it)
      iteration i   i = 1 .. len(n_request): for every frequency the cells emit n_request[i-1] packages (counts by `mode`
                    from the current T), seed + i:  D_i = sum_f w_f A_dust,f  (and the in-cell part S_i, emission Em_i)
                    reference field: R_i = running mean of D_k, k = ref_start..i, weighted by n_request
                    (R_i = D_i without it, and for i < ref_start)
                    T = table(A_const + R_i)   -- with ALI from (A - S) / (1 - S / Em) (soc_oracle_update_temperatures_ali)
    Returns dict(T=[T_0, T_1, ...], A_const, R, S, Em, emitted=[...], escaped=[...]) (frequency-integrated energies)."""
    freq_hz = np.asarray(freq_hz, dtype=np.float64)
    n_f = len(freq_hz)
    w = trapezoid_weights(freq_hz)
    A_const = np.zeros(grid.n_total)
    esc0 = em0 = 0.0
    for f in range(n_f):
        _, r, _, _ = simulate(grid, kabs[f], ksca[f], g[f], f, const_sources[f], n_const, seed, w[f], absorbed=A_const,
                              threads=threads, f32state=f32state)
        esc0 += w[f] * r.escaped
        em0 += w[f] * r.emitted
    T = update_temperatures(grid, A_const, t_scale, table_T, E_min, E_max) if T_start is None else np.asarray(T_start, np.float32)
    out = dict(T=[T.copy()], A_const=A_const, emitted=[em0], escaped=[esc0], D=[], n_dust=[])
    R, S, Em, W = np.zeros(grid.n_total), np.zeros(grid.n_total), np.zeros(grid.n_total), 0.0
    for i, n_req in enumerate(n_request, start=1):
        D, Si, Emi = np.zeros(grid.n_total), np.zeros(grid.n_total), np.zeros(grid.n_total)
        esc = em = 0.0
        nd = 0
        for f in range(n_f):
            cnt = emission_counts(grid, kabs[f], freq_hz[f], T, mode, n_req, cap)
            n_dust = int(cnt.sum(dtype=np.int64))
            nd += n_dust
            Emi += w[f] * cell_luminosity(grid, kabs[f], freq_hz[f], T)
            if n_dust == 0:
                continue
            src = dict(dust_T=T, dust_count=cnt, dust_freq_hz=freq_hz[f], dust_self=Si, n_bg=0)
            _, r, _, _ = simulate(grid, kabs[f], ksca[f], g[f], f, src, n_dust, seed + i, w[f], absorbed=D, threads=threads,
                                  f32state=f32state)
            esc += w[f] * r.escaped
            em += w[f] * r.emitted
        if reference_field and i >= ref_start:
            R = (W * R + n_req * D) / (W + n_req)
            S = (W * S + n_req * Si) / (W + n_req)
            Em = (W * Em + n_req * Emi) / (W + n_req)
            W += n_req
        else:
            R, S, Em = D, Si, Emi
        A = A_const + R
        if update_T:
            T = (update_temperatures_ali(grid, A, S, Em, t_scale, table_T, E_min, E_max) if ali
                 else update_temperatures(grid, A, t_scale, table_T, E_min, E_max))
        out["T"].append(T.copy()); out["emitted"].append(em); out["escaped"].append(esc); out["D"].append(D)
        out["n_dust"].append(nd)
    out.update(R=R, S=S, Em=Em)
    return out


# ---------------------------------------------------------------------------------------------------------------------
# f4: stochastically heated grains (Appendix A) -- plain numpy, fp64, the definition written out.
# "The calculation reduces to a linear set of equations where the unknowns are the fraction of dust in each enthalpy bin.
#  ... In the transition matrix R, the upward transitions (R_ji, i < j) are obtained by taking a vector product of the
#  intensity with the integration weights.  The pre-calculated cooling rates occupy the elements R_(i-1,i) above the main
#  diagonal.  The diagonal elements R_ii are determined from detailed balance and are equal to the sum of the other column
#  elements multiplied by minus one.  The matrix elements R_ji = 0, i > j + 1 are zeros".
# The paper's programs solve R p = 0 by forward substitution or Gauss-Seidel; the oracle solves the same linear system with
# a general dense solver (LAPACK through numpy), the normalisation sum p = 1 taking the place of the redundant last row.
def stochastic_rate_matrix(W, cool, intensity):
    """R [n_E, n_E] for one grain size and one cell.  W[j, i, f]: integration weights of the upward transition i -> j
    (zero for j <= i); cool[i]: cooling rate i -> i - 1 (cool[0] unused); intensity[f]."""
    W, cool, intensity = (np.asarray(x, dtype=np.float64) for x in (W, cool, intensity))
    n = len(cool)
    R = np.zeros((n, n))
    for i in range(n):
        for j in range(i + 1, n):
            R[j, i] = float(np.dot(W[j, i], intensity))          # "vector product of the intensity with the weights"
    for i in range(1, n):
        R[i - 1, i] = cool[i]
    for i in range(n):
        R[i, i] = -(R[:, i].sum() - R[i, i])                     # detailed balance: every column sums to zero
    return R


def stochastic_solve(R):
    """p >= 0 with R p = 0 and sum p = 1."""
    n = R.shape[0]
    # columns differ by many orders of magnitude (cooling of the hot bins against absorption in the cold ones): scale the
    # unknowns by the cooling time of their bin so that LAPACK sees an O(1) matrix; q_i = p_i * scale_i
    scale = np.array([max(-R[i, i], 1e-300) for i in range(n)])
    A = R / scale[None, :]
    A[-1, :] = 1.0 / scale                                       # sum_i q_i / scale_i = 1 replaces the redundant last row
    rhs = np.zeros(n); rhs[-1] = 1.0
    row = np.abs(A).max(axis=1)
    q = np.linalg.solve(A / row[:, None], rhs / row)
    p = q / scale
    return p / p.sum()


def stochastic_emission(p, emis, abundance):
    """emission[f] = sum_s abundance[s] sum_i p[s, i] emis[s, i, f]."""
    return np.einsum("s,si,sif->f", np.asarray(abundance, np.float64), np.asarray(p, np.float64), np.asarray(emis, np.float64))


def stochastic_cells(model, intensity):
    """All cells and sizes: p[cell, s, i], emission[cell, f].  model: inputs.stochastic_model(); intensity[cell, f]."""
    n_s, n_e, n_f = model["jup"].shape
    W = np.zeros((n_s, n_e, n_e, n_f))
    s_idx, i_idx, f_idx = np.nonzero(model["jup"] >= 0)
    W[s_idx, model["jup"][s_idx, i_idx, f_idx], i_idx, f_idx] = model["wup"][s_idx, i_idx, f_idx]
    intensity = np.asarray(intensity, dtype=np.float64)
    p = np.zeros((len(intensity), n_s, n_e))
    for c in range(len(intensity)):
        for s in range(n_s):
            p[c, s] = stochastic_solve(stochastic_rate_matrix(W[s], model["cool"][s], intensity[c]))
    em = np.stack([stochastic_emission(p[c], model["emis"], model["abundance"]) for c in range(len(intensity))])
    return p, em
