"""Thin ctypes binding over libsoc_b200.so (include/soc.h): argument marshalling only.

Every step of the path (RNG, emission, walk, deposit, scattering, frequency loop, temperature lookup)
runs in the CUDA kernels behind the C ABI.  torch is used for device memory and streams.  There is no
CPU fallback: if the library is not built, or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsoc_b200.so")
if os.environ.get("SOC_B200_LIB"):                      # e.g. the bounds-checked build, libsoc_b200_checked.so (tests)
    LIB_PATH = os.environ["SOC_B200_LIB"]

SOC_GEOM_FP32 = 0
SOC_GEOM_FP64 = 1
MAX_POINT_SOURCES = 64
STATIC_MAX_CELLS = 1 << 21          # soc_update_temperatures_ali_static: cells its built-in scratch array holds

EXPORTS = ["soc_grid_create", "soc_grid_destroy", "soc_grid_n_total", "soc_freq_weights", "soc_simulate_frequency",
           "soc_simulate_packages", "soc_simulate_spectrum", "soc_update_temperatures", "soc_run_host",
           "soc_set_option", "soc_get_timings", "soc_probe_throughput", "soc_launch_count", "soc_last_error", "soc_version",
           "soc_emission_counts", "soc_cell_emission", "soc_update_temperatures_ali", "soc_iterate", "soc_make_map",
           "soc_checked_violations", "soc_stochastic_create", "soc_stochastic_destroy", "soc_stochastic_emission",
           "soc_release_cached_memory", "soc_update_temperatures_ali_static"]


class SocError(RuntimeError):
    pass


class GridDesc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("n_levels", C.c_int32),
                ("n_cells", C.c_void_p), ("density", C.c_void_p), ("child", C.c_void_p),
                ("n_freq", C.c_int32), ("freq_hz", C.c_void_p), ("kabs", C.c_void_p), ("ksca", C.c_void_p),
                ("g", C.c_void_p)]


class Sources(C.Structure):
    _fields_ = [("bg_intensity", C.c_double), ("n_point", C.c_int32), ("ps_pos", C.c_void_p),
                ("ps_lum", C.c_void_p), ("n_bg", C.c_int64), ("beam", C.c_void_p),
                ("n_dust", C.c_int64), ("dust_T", C.c_void_p), ("dust_count", C.c_void_p), ("dust_self", C.c_void_p)]


class MapDesc(C.Structure):
    _fields_ = [("ex", C.c_double * 3), ("ey", C.c_double * 3), ("dir", C.c_double * 3), ("centre", C.c_double * 3),
                ("npx", C.c_int32), ("npy", C.c_int32), ("pixel", C.c_double)]


class StochasticModel(C.Structure):
    _fields_ = [("n_size", C.c_int32), ("n_e", C.c_int32), ("n_freq", C.c_int32), ("jup", C.c_void_p), ("wup", C.c_void_p),
                ("cool", C.c_void_p), ("emis", C.c_void_p), ("abundance", C.c_void_p)]


class IterateOpts(C.Structure):
    _fields_ = [("mode", C.c_int32), ("cap", C.c_int32), ("reference_field", C.c_int32), ("ref_start", C.c_int32),
                ("ali", C.c_int32), ("n_iter", C.c_int32), ("n_request", C.c_void_p)]


class IterateRecord(C.Structure):
    _fields_ = [("emitted", C.c_double), ("escaped", C.c_double), ("absorbed", C.c_double),
                ("n_packages", C.c_int64), ("cell_steps", C.c_uint64)]


class FreqResult(C.Structure):
    _fields_ = [("emitted", C.c_double), ("escaped", C.c_double), ("absorbed", C.c_double),
                ("cell_steps", C.c_uint64), ("scatterings", C.c_uint64), ("terminated", C.c_uint64),
                ("weight_drift", C.c_double), ("gather_requests", C.c_uint64), ("red_requests", C.c_uint64),
                ("suspensions", C.c_uint64), ("queue_refusals", C.c_uint64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


REPLAY_DTYPE = np.dtype([("hash", "<u8"), ("steps", "<u4"), ("scatters", "<u4"), ("e_escaped", "<f8")])

_lib = None


def load():
    """Load the C-ABI library; raises if it has not been built (python -m paper_1812_06632_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise SocError(f"{LIB_PATH} is missing: build it with `python paper_1812_06632_b200/build.py` "
                       "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, u64, u32, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_uint32, C.c_double
    L.soc_grid_create.argtypes = [C.POINTER(GridDesc), C.POINTER(vp)]
    L.soc_grid_destroy.argtypes = [vp]
    L.soc_grid_destroy.restype = None
    L.soc_grid_n_total.argtypes = [vp]
    L.soc_grid_n_total.restype = i64
    L.soc_freq_weights.argtypes = [vp, vp]
    L.soc_simulate_frequency.argtypes = [vp, i32, C.POINTER(Sources), i64, u64, dbl, vp, C.POINTER(FreqResult), u32, vp]
    L.soc_simulate_packages.argtypes = [vp, i32, C.POINTER(Sources), i64, u64, dbl, i64, i64, vp, vp,
                                        C.POINTER(FreqResult), u32, vp]
    L.soc_simulate_spectrum.argtypes = [vp, C.POINTER(Sources), i64, u64, i64, i64, vp, C.POINTER(FreqResult), u32, vp]
    L.soc_update_temperatures.argtypes = [vp, vp, dbl, vp, i32, dbl, dbl, vp, vp]
    L.soc_emission_counts.argtypes = [vp, i32, vp, i32, i64, i32, vp, C.POINTER(i64), C.POINTER(dbl), vp]
    L.soc_cell_emission.argtypes = [vp, vp, vp, vp]
    L.soc_update_temperatures_ali.argtypes = [vp, vp, vp, vp, dbl, vp, i32, dbl, dbl, vp, vp]
    L.soc_update_temperatures_ali_static.argtypes = [vp, vp, vp, vp, dbl, vp, i32, dbl, dbl, vp, vp]
    L.soc_iterate.argtypes = [vp, C.POINTER(Sources), i64, u64, C.POINTER(IterateOpts), dbl, vp, i32, dbl, dbl, vp, vp,
                              C.POINTER(IterateRecord), u32, vp]
    L.soc_make_map.argtypes = [vp, i32, vp, C.POINTER(MapDesc), vp, vp]
    L.soc_stochastic_create.argtypes = [C.POINTER(StochasticModel), C.POINTER(vp)]
    L.soc_stochastic_destroy.argtypes = [vp]
    L.soc_stochastic_destroy.restype = None
    L.soc_stochastic_emission.argtypes = [vp, vp, i64, vp, vp, vp]
    L.soc_run_host.argtypes = [C.POINTER(GridDesc), C.POINTER(Sources), i64, u64, i32, dbl, vp, i32, dbl, dbl, vp, vp,
                               C.POINTER(FreqResult), u32]
    L.soc_set_option.argtypes = [vp, C.c_char_p, i64]
    L.soc_get_timings.argtypes = [vp, i32, vp]
    L.soc_probe_throughput.argtypes = [i32, i64, i64, C.POINTER(C.c_float)]
    L.soc_launch_count.restype = u64
    L.soc_release_cached_memory.restype = i64
    L.soc_checked_violations.restype = i64
    L.soc_last_error.restype = C.c_char_p
    L.soc_version.restype = C.c_char_p
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        raise SocError(f"libsoc_b200 error {rc}: {load().soc_last_error().decode()}")


def _np(a, dtype):
    return None if a is None else np.ascontiguousarray(a, dtype=dtype)


def _ptr(a):
    return None if a is None else a.ctypes.data


def _dev_ptr(t):
    import torch
    if t is None:
        return None
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()
    return t.data_ptr()


def _stream_ptr(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def make_desc(nx, ny, nz, n_cells, density, child, freq_hz, kabs, ksca, g):
    """GridDesc plus the list of host arrays that must stay alive while it is used."""
    keep = [_np(n_cells, np.int64), _np(density, np.float32), _np(child, np.int32), _np(freq_hz, np.float64),
            _np(kabs, np.float64), _np(ksca, np.float64), _np(g, np.float64)]
    d = GridDesc(int(nx), int(ny), int(nz), len(keep[0]), _ptr(keep[0]), _ptr(keep[1]), _ptr(keep[2]),
                 len(keep[3]), _ptr(keep[3]), _ptr(keep[4]), _ptr(keep[5]), _ptr(keep[6]))
    return d, keep


def make_sources(src: dict, keep: list):
    s = Sources()
    s.bg_intensity = float(src.get("bg_intensity", 0.0))
    pos, lum = src.get("ps_pos"), src.get("ps_lum")
    s.n_point = 0 if pos is None else int(np.asarray(pos).reshape(-1, 3).shape[0])
    if s.n_point:
        pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
        lum = np.ascontiguousarray(lum, dtype=np.float64).reshape(-1)
        assert len(lum) == s.n_point
        keep += [pos, lum]
        s.ps_pos, s.ps_lum = pos.ctypes.data, lum.ctypes.data
    s.n_bg = int(src.get("n_bg", -1))
    beam = src.get("beam")
    if beam is not None:
        beam = np.ascontiguousarray(beam, dtype=np.float64).reshape(6)
        keep.append(beam)
        s.beam = beam.ctypes.data
    if src.get("dust_count") is not None:             # f1: DEVICE tensors; n_dust = the sum of dust_count (host int)
        s.n_dust = int(src["n_dust"])
        s.dust_T, s.dust_count = _dev_ptr(src["dust_T"]), _dev_ptr(src["dust_count"])
        s.dust_self = _dev_ptr(src.get("dust_self"))
    return s


def make_sources_array(src_list):
    keep = []
    arr = (Sources * len(src_list))()
    for i, s in enumerate(src_list):
        arr[i] = make_sources(s, keep)
    return arr, keep


class Grid:
    """soc_grid handle."""

    def __init__(self, nx, ny, nz, n_cells, density, child, freq_hz, kabs, ksca, g):
        L = load()
        desc, keep = make_desc(nx, ny, nz, n_cells, density, child, freq_hz, kabs, ksca, g)
        h = C.c_void_p()
        _check(L.soc_grid_create(C.byref(desc), C.byref(h)))
        self._h = h
        self.n_total = int(L.soc_grid_n_total(h))
        self.n_freq = len(keep[3])

    @classmethod
    def from_problem(cls, P):
        return cls(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child, P.freq_hz, P.kabs, P.ksca, P.g)

    def close(self):
        if getattr(self, "_h", None):
            load().soc_grid_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:       # interpreter shutdown
            pass

    def set_option(self, key, value):
        _check(load().soc_set_option(self._h, key.encode(), int(value)))

    def timings_ms(self, n=None):
        """Per-slot photon-kernel device times (needs set_option("timing", 1) before the launches)."""
        ms = np.zeros(self.n_freq if n is None else int(n), dtype=np.float32)
        _check(load().soc_get_timings(self._h, len(ms), _ptr(ms)))
        return ms

    def freq_weights(self):
        w = np.zeros(self.n_freq)
        _check(load().soc_freq_weights(self._h, _ptr(w)))
        return w

    def simulate_frequency(self, ifreq, sources, n_packages, seed, weight, absorbed, want_result=True,
                           flags=SOC_GEOM_FP32, stream=None):
        keep = []
        s = make_sources(sources, keep)
        res = FreqResult()
        _check(load().soc_simulate_frequency(self._h, int(ifreq), C.byref(s), int(n_packages), int(seed), float(weight),
                                             _dev_ptr(absorbed), C.byref(res) if want_result else None, int(flags),
                                             _stream_ptr(stream)))
        return res if want_result else None

    def simulate_packages(self, ifreq, sources, n_packages, seed, weight, pkg_begin, pkg_count, absorbed, replay=None,
                          want_result=True, flags=SOC_GEOM_FP32, stream=None):
        """replay: torch.uint8 CUDA tensor of pkg_count * 24 bytes (see REPLAY_DTYPE) or None."""
        keep = []
        s = make_sources(sources, keep)
        res = FreqResult()
        _check(load().soc_simulate_packages(self._h, int(ifreq), C.byref(s), int(n_packages), int(seed), float(weight),
                                            int(pkg_begin), int(pkg_count), _dev_ptr(absorbed), _dev_ptr(replay),
                                            C.byref(res) if want_result else None, int(flags), _stream_ptr(stream)))
        return res if want_result else None

    def simulate_spectrum(self, sources_list, n_packages, seed, absorbed_int, pkg_begin=0, pkg_count=None,
                          want_results=True, flags=SOC_GEOM_FP32, stream=None):
        assert len(sources_list) == self.n_freq
        arr, keep = make_sources_array(sources_list)
        if pkg_count is None:
            pkg_count = n_packages - pkg_begin
        res = (FreqResult * self.n_freq)() if want_results else None
        _check(load().soc_simulate_spectrum(self._h, arr, int(n_packages), int(seed), int(pkg_begin), int(pkg_count),
                                            _dev_ptr(absorbed_int), res, int(flags), _stream_ptr(stream)))
        return list(res) if want_results else None

    def make_map(self, ifreq, T, ex, ey, direction, centre, npx, npy, pixel, map_out, stream=None):
        """soc_make_map: map_out = DEVICE float32 tensor of npx * npy elements (pixel i fastest)."""
        d = MapDesc()
        for name, v in (("ex", ex), ("ey", ey), ("dir", direction), ("centre", centre)):
            setattr(d, name, (C.c_double * 3)(*[float(x) for x in v]))
        d.npx, d.npy, d.pixel = int(npx), int(npy), float(pixel)
        _check(load().soc_make_map(self._h, int(ifreq), _dev_ptr(T), C.byref(d), _dev_ptr(map_out), _stream_ptr(stream)))

    def emission_counts(self, ifreq, T, mode, n_request, cap, count_out, stream=None):
        """soc_emission_counts: writes count_out (DEVICE int32), returns (n_dust, sum of the luminosities)."""
        n, tot = C.c_int64(0), C.c_double(0.0)
        _check(load().soc_emission_counts(self._h, int(ifreq), _dev_ptr(T), {"uniform": 0, "weighted": 1}[mode], int(n_request),
                                          int(cap), _dev_ptr(count_out), C.byref(n), C.byref(tot), _stream_ptr(stream)))
        return n.value, tot.value

    def cell_emission(self, T, emitted_out, stream=None):
        _check(load().soc_cell_emission(self._h, _dev_ptr(T), _dev_ptr(emitted_out), _stream_ptr(stream)))

    def update_temperatures_ali(self, absorbed, self_abs, emitted, scale, table_T, e_min, e_max, T_out, stream=None):
        tab = _np(table_T, np.float32)
        _check(load().soc_update_temperatures_ali(self._h, _dev_ptr(absorbed), _dev_ptr(self_abs), _dev_ptr(emitted), float(scale),
                                                  _ptr(tab), len(tab), float(e_min), float(e_max), _dev_ptr(T_out),
                                                  _stream_ptr(stream)))

    def update_temperatures_ali_static(self, absorbed, self_abs, emitted, scale, table_T, e_min, e_max, T_out, stream=None):
        """soc_update_temperatures_ali_static: update_temperatures_ali without any allocation inside the library, for host
        programs that own all device memory themselves or cannot afford cudaMalloc's device-wide stall (soc.h).  Grids of
        at most STATIC_MAX_CELLS cells; one scratch array per GPU, so calls that overlap on the device race."""
        tab = _np(table_T, np.float32)
        _check(load().soc_update_temperatures_ali_static(self._h, _dev_ptr(absorbed), _dev_ptr(self_abs), _dev_ptr(emitted),
                                                         float(scale), _ptr(tab), len(tab), float(e_min), float(e_max),
                                                         _dev_ptr(T_out), _stream_ptr(stream)))

    def iterate(self, sources_list, n_const, seed, n_request, t_scale, table_T, e_min, e_max, absorbed_out, T_out,
                mode="weighted", cap=10000, reference_field=True, ref_start=1, ali=False, flags=SOC_GEOM_FP32, stream=None):
        """soc_iterate: constant sources once, then len(n_request) iterations of dust re-emission.  Returns the history."""
        assert len(sources_list) == self.n_freq
        arr, keep = make_sources_array(sources_list)
        req = _np(n_request, np.int64)
        opts = IterateOpts({"uniform": 0, "weighted": 1}[mode], int(cap), int(bool(reference_field)), int(ref_start),
                           int(bool(ali)), len(req), _ptr(req) if len(req) else None)
        hist = (IterateRecord * (len(req) + 1))()
        tab = _np(table_T, np.float32)
        _check(load().soc_iterate(self._h, arr, int(n_const), int(seed), C.byref(opts), float(t_scale), _ptr(tab), len(tab),
                                  float(e_min), float(e_max), _dev_ptr(absorbed_out), _dev_ptr(T_out), hist, int(flags),
                                  _stream_ptr(stream)))
        return [dict(emitted=h.emitted, escaped=h.escaped, absorbed=h.absorbed, n_packages=h.n_packages,
                     cell_steps=h.cell_steps) for h in hist]

    def update_temperatures(self, absorbed, scale, table_T, e_min, e_max, T_out, stream=None):
        tab = _np(table_T, np.float32)
        _check(load().soc_update_temperatures(self._h, _dev_ptr(absorbed), float(scale), _ptr(tab), len(tab),
                                              float(e_min), float(e_max), _dev_ptr(T_out), _stream_ptr(stream)))


def run_host(P, n_packages=None, seed=None, n_iter=None, flags=SOC_GEOM_FP32, want_results=False,
             absorbed_out=None, T_out=None):
    """soc_run_host on an inputs.Problem: HOST buffers in, HOST buffers out."""
    L = load()
    desc, keep = make_desc(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child, P.freq_hz, P.kabs, P.ksca, P.g)
    arr, keep2 = make_sources_array([P.sources(f) for f in range(P.n_freq)])
    n_iter = int(n_iter or P.n_iter)
    if absorbed_out is None:
        absorbed_out = np.zeros(P.n_total, dtype=np.float64)
    has_T = P.table_T is not None
    if T_out is None and has_T:
        T_out = np.zeros(P.n_total, dtype=np.float32)
    tab = _np(P.table_T, np.float32) if has_T else None
    res = (FreqResult * (n_iter * P.n_freq))() if want_results else None
    _check(L.soc_run_host(C.byref(desc), arr, int(n_packages or P.n_packages), int(P.seed if seed is None else seed),
                          n_iter, float(P.t_scale or 0.0), _ptr(tab), 0 if tab is None else len(tab), float(P.e_min),
                          float(P.e_max), _ptr(absorbed_out), _ptr(T_out) if has_T else None, res, int(flags)))
    return absorbed_out, (T_out if has_T else None), (list(res) if want_results else None)


class Stochastic:
    """soc_stochastic handle (row f4): tables of inputs.stochastic_model() on the device."""

    def __init__(self, model):
        jup, wup = _np(model["jup"], np.int32), _np(model["wup"], np.float64)
        cool, emis, ab = _np(model["cool"], np.float64), _np(model["emis"], np.float64), _np(model["abundance"], np.float64)
        self.n_size, self.n_e, self.n_freq = jup.shape
        m = StochasticModel(self.n_size, self.n_e, self.n_freq, _ptr(jup), _ptr(wup), _ptr(cool), _ptr(emis), _ptr(ab))
        h = C.c_void_p()
        _check(load().soc_stochastic_create(C.byref(m), C.byref(h)))
        self._h = h

    def emission(self, intensity, emission_out, p_out=None, stream=None):
        n_cells = intensity.shape[0]
        _check(load().soc_stochastic_emission(self._h, _dev_ptr(intensity), int(n_cells), _dev_ptr(emission_out), _dev_ptr(p_out),
                                              _stream_ptr(stream)))

    def close(self):
        if getattr(self, "_h", None):
            load().soc_stochastic_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def checked_violations():
    """Bounds-checked build: out-of-range kernel indices so far (-1: the product library, checks compiled out)."""
    return int(load().soc_checked_violations())


def probe_throughput(kind, footprint_bytes, n_ops):
    ms = C.c_float(0)
    _check(load().soc_probe_throughput(int(kind), int(footprint_bytes), int(n_ops), C.byref(ms)))
    return ms.value


def launch_count():
    return int(load().soc_launch_count())


def release_cached_memory():
    return int(load().soc_release_cached_memory())
