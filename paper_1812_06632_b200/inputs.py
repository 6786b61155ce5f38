"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic (no RNG stream, no emission/walk/deposit/scatter, no temperature lookup):
it only manufactures the *inputs* of the C-ABI calls -- clouds, dust tables, source spectra and
the T(E) table -- from fixed seeds.  The paper's own workloads (Ramses MHD snapshot PAPER.md:89,
Mathis et al. 1983 field and Compiegne et al. 2011 dust PAPER.md:105) are not available; the
inputs below take their shapes and stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

try:  # threaded FFT when scipy is there; numpy otherwise (same result up to rounding)
    from scipy import fft as _fft

    def _rfftn(a):
        return _fft.rfftn(a, workers=-1)

    def _irfftn(a, s):
        return _fft.irfftn(a, s=s, workers=-1)
except Exception:  # pragma: no cover
    def _rfftn(a):
        return np.fft.rfftn(a)

    def _irfftn(a, s):
        return np.fft.irfftn(a, s=s)

# cgs constants
H_PLANCK = 6.62607015e-27
K_BOLTZ = 1.380649e-16
C_LIGHT = 2.99792458e10
SIGMA_SB = 5.670374419e-5
L_SUN = 3.828e33
PARSEC = 3.0856775814913673e18
LAMBDA_V_UM = 0.55
SIGMA_EXT_V = 5e-22          # cm^2 per H at V


def planck_nu(nu, T):
    """B_nu(T), erg s^-1 cm^-2 Hz^-1 sr^-1 (source spectra and the dust emissivity table)."""
    nu = np.asarray(nu, dtype=np.float64)
    x = H_PLANCK * nu / (K_BOLTZ * T)
    with np.errstate(over="ignore", under="ignore"):
        return 2.0 * H_PLANCK * nu ** 3 / C_LIGHT ** 2 / np.expm1(x)


def gaussian_random_field(n, seed, slope=-3.0):
    """Periodic n^3 Gaussian field with P(k) ~ k^slope, zero mean, unit variance (float64)."""
    rng = np.random.default_rng(seed)
    white = rng.standard_normal((n, n, n))
    fk = _rfftn(white)
    del white
    kx = np.fft.fftfreq(n) * n
    kz = np.fft.rfftfreq(n) * n
    k2 = kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    fk *= k2 ** (slope / 4.0)          # amplitude ~ k^(slope/2)
    fk[0, 0, 0] = 0.0
    del k2
    delta = _irfftn(fk, (n, n, n))
    del fk
    delta -= delta.mean()
    delta /= delta.std()
    return delta


def lognormal_cloud(n, sigma_ln, seed):
    """rho = exp(sigma * delta) / mean, array [z][y][x] (x fastest), float64."""
    rho = np.exp(sigma_ln * gaussian_random_field(n, seed))
    rho /= rho.mean()
    return rho


def max_column(rho3d):
    """Largest line-of-sight column (sum of rho over cells of edge 1) over the three axis projections."""
    return max(float(rho3d.sum(axis=a).max()) for a in range(3))


def wavelength_grid_um(lam_min_um, lam_max_um, n):
    """Log-spaced wavelengths; index 0 = longest wavelength = lowest frequency."""
    if n == 1:
        return np.array([lam_min_um], dtype=np.float64)
    return np.geomspace(lam_max_um, lam_min_um, n)


def dust_model(lam_um, albedo_v=0.6, g_v=0.6):
    """Smooth synthetic power-law dust: q_abs, q_sca (q_abs+q_sca = 1 at V) and g."""
    lam = np.asarray(lam_um, dtype=np.float64)

    def qa(x):
        return (x / LAMBDA_V_UM) ** -1.0 * (1.0 + (x / 50.0) ** 2) ** -0.5

    def qs(x):
        return (x / LAMBDA_V_UM) ** -1.0 * (1.0 + (x / 1.0) ** 2) ** -1.5

    q_abs = (1.0 - albedo_v) * qa(lam) / qa(LAMBDA_V_UM)
    q_sca = albedo_v * qs(lam) / qs(LAMBDA_V_UM)
    g = g_v * (1.0 + (LAMBDA_V_UM / 2.0) ** 2) / (1.0 + (lam / 2.0) ** 2)
    return q_abs, q_sca, g


def background_intensity(nu):
    """Stand-in for the interstellar radiation field: diluted 5000 K blackbody + CMB."""
    return 1e-13 * planck_nu(nu, 5000.0) + planck_nu(nu, 2.73)


def point_source_lnu(nu, lum=100.0 * L_SUN, teff=1.0e4):
    """L_nu (erg s^-1 Hz^-1) of a blackbody of bolometric luminosity lum."""
    return lum * np.pi * planck_nu(nu, teff) / (SIGMA_SB * teff ** 4)


def trapz_weights(x):
    x = np.asarray(x, dtype=np.float64)
    if x.size == 1:
        return np.ones(1)
    w = np.empty_like(x)
    w[0] = 0.5 * abs(x[1] - x[0])
    w[-1] = 0.5 * abs(x[-1] - x[-2])
    w[1:-1] = 0.5 * np.abs(x[2:] - x[:-2])
    return w


def emissivity_per_h(freq_hz, sigma_abs_cm2, T):
    """Lambda(T) = 4 pi sum_f w_f sigma_abs,f B_nu_f(T): power emitted per H atom (erg/s)."""
    w = trapz_weights(freq_hz)
    T = np.atleast_1d(np.asarray(T, dtype=np.float64))
    B = planck_nu(np.asarray(freq_hz)[None, :], T[:, None])
    return 4.0 * np.pi * (B * (w * sigma_abs_cm2)[None, :]).sum(axis=1)


def temperature_table(freq_hz, sigma_abs_cm2, n_table=2048, t_lo=3.0, t_hi=1500.0, n_fine=8192):
    """T_k on the log-uniform grid E_k = E_min (E_max/E_min)^(k/(n-1)) (an INPUT of soc_update_temperatures).

    Lambda is evaluated on a fine log-T grid and inverted by monotone linear interpolation in
    (ln Lambda, ln T).  Returns (table_T float32[n_table], E_min, E_max).
    """
    t_fine = np.geomspace(t_lo, t_hi, n_fine)
    lam = emissivity_per_h(freq_hz, sigma_abs_cm2, t_fine)
    e_min, e_max = float(lam[0]), float(lam[-1])
    ln_e = np.linspace(np.log(e_min), np.log(e_max), n_table)
    ln_t = np.interp(ln_e, np.log(lam), np.log(t_fine))
    return np.exp(ln_t).astype(np.float32), e_min, e_max


# ----------------------------------------------------------------------------- stochastically heated grains (row f4)
def stochastic_model(freq_hz, n_size=25, n_e=64, a_min_um=4e-4, a_max_um=1e-2, t_lo=2.7, t_hi=2500.0):
    """Synthetic stand-in for the grain data of the paper's Appendix A test (DustEM enthalpy tables are not available;
    PAPER.md:359-371: 25 size bins, 128 frequencies).  INPUTS of soc_stochastic_emission, given to both sides:

      per size s (radius a_s, log-spaced) and enthalpy bin i (temperatures T_i log-spaced, enthalpy E = c_V a^3 T^4 / 4,
      a Debye solid):
        jup[s, i, f], wup[s, i, f]   a photon of frequency f takes a grain from bin i to the bin jup that holds E_i + h nu
                                     (the last bin takes everything above); the transition rate is wup * intensity[f]
                                     with wup = 4 pi C_abs(nu) w_f / (h nu), C_abs = pi a^2 Q_abs, Q_abs ~ min(1, 2 pi a /
                                     lambda).  A photon too soft to lift the grain out of its bin heats it continuously:
                                     jup = i + 1 with the rate scaled by h nu / (E_(i+1) - E_i), which conserves the
                                     energy; -1 only in the last bin
        cool[s, i]                   "thermal continuous" cooling to the next lower bin: radiated power / (E_i - E_(i-1))
        emis[s, i, f]                4 pi C_abs(nu_f) B_nu(T_i): emission of one grain in bin i
        abundance[s]                 grains per H, MRN dn/da ~ a^-3.5
    """
    nu = np.asarray(freq_hz, dtype=np.float64)
    w = trapz_weights(nu)
    a = np.geomspace(a_min_um, a_max_um, n_size) * 1e-4                        # cm
    lam = C_LIGHT / nu
    T = np.geomspace(t_lo, t_hi, n_e)
    jup = np.full((n_size, n_e, len(nu)), -1, dtype=np.int32)
    wup = np.zeros((n_size, n_e, len(nu)))
    cool = np.zeros((n_size, n_e))
    emis = np.zeros((n_size, n_e, len(nu)))
    E_all = np.zeros((n_size, n_e))
    for s in range(n_size):
        c_abs = np.pi * a[s] ** 2 * np.minimum(1.0, 2 * np.pi * a[s] / lam)
        E = 2.5e4 * a[s] ** 3 * T ** 4 / 4.0                                    # erg; c_V ~ 2.5e4 T^3 erg cm^-3 K^-1
        E_all[s] = E
        edges = np.concatenate([[0.0], np.sqrt(E[:-1] * E[1:]), [np.inf]])      # bin i = [edges[i], edges[i+1])
        power = np.array([4 * np.pi * float((w * c_abs * planck_nu(nu, t)).sum()) for t in T])
        cool[s, 1:] = power[1:] / (E[1:] - E[:-1])
        emis[s] = 4 * np.pi * c_abs[None, :] * planck_nu(nu[None, :], T[:, None])
        for i in range(n_e):
            j = np.searchsorted(edges, E[i] + H_PLANCK * nu, side="right") - 1
            j = np.minimum(j, n_e - 1)
            rate = 4 * np.pi * c_abs * w / (H_PLANCK * nu)
            up = j > i
            jup[s, i, up] = j[up]
            wup[s, i, up] = rate[up]
            if i + 1 < n_e:
                jup[s, i, ~up] = i + 1
                wup[s, i, ~up] = (rate * H_PLANCK * nu / (E[i + 1] - E[i]))[~up]
    abundance = a ** -3.5
    abundance *= 1e-9 / abundance.sum()
    return dict(jup=jup, wup=wup, cool=cool, emis=emis, abundance=abundance, T=T, E=E_all, a_cm=a, freq_hz=nu)


# ----------------------------------------------------------------------------- hierarchy
def block_average(a):
    n = a.shape[0] // 2
    return a.reshape(n, 2, n, 2, n, 2).mean(axis=(1, 3, 5))


def build_octree(fine_rho, root_n, n_levels, theta):
    """Octree cloud from a fine (root_n * 2^(n_levels-1))^3 field.

    A cell at level l is refined while its block-averaged density exceeds theta x the global mean
    and l < n_levels.  Returns (n_cells[int64], rho[float32, level-major], child[int32]) in the
    paper's cell-vector order: root cells x-fastest, then level 2, ...; the 8 cells of
    an octet are consecutive, slot = bx + 2 by + 4 bz; child = -1 (leaf) or index of the first child
    within the next level.  Parent cells carry rho = 0.
    """
    levels = [np.asarray(fine_rho, dtype=np.float64)]
    while levels[0].shape[0] > root_n:
        levels.insert(0, block_average(levels[0]))
    assert len(levels) == n_levels and levels[0].shape[0] == root_n
    mean = float(levels[-1].mean())
    iz, iy, ix = np.meshgrid(np.arange(root_n), np.arange(root_n), np.arange(root_n), indexing="ij")
    coords = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.int32)   # x fastest
    n_cells, rhos, childs = [], [], []
    for lev in range(n_levels):
        a = levels[lev]
        dens = a[coords[:, 2], coords[:, 1], coords[:, 0]]
        refine = (dens > theta * mean) if lev < n_levels - 1 else np.zeros(len(dens), dtype=bool)
        child = np.full(len(dens), -1, dtype=np.int32)
        child[refine] = 8 * np.arange(int(refine.sum()), dtype=np.int32)
        rho = np.where(refine, 0.0, dens).astype(np.float32)
        n_cells.append(len(dens)); rhos.append(rho); childs.append(child)
        if not refine.any():
            break
        par = coords[refine]
        slots = np.arange(8, dtype=np.int32)
        off = np.stack([slots & 1, (slots >> 1) & 1, (slots >> 2) & 1], axis=1)
        coords = (2 * par[:, None, :] + off[None, :, :]).reshape(-1, 3)
    return np.asarray(n_cells, dtype=np.int64), np.concatenate(rhos), np.concatenate(childs)


# ----------------------------------------------------------------------------- problems
@dataclass
class Problem:
    """Everything the C-ABI calls need for one config (host arrays)."""
    name: str
    nx: int
    ny: int
    nz: int
    n_cells: np.ndarray            # int64 [n_levels]
    rho: np.ndarray                # float32 [n_total], level-major
    child: np.ndarray | None       # int32 [n_total] or None (regular grid)
    freq_hz: np.ndarray            # [n_freq], ascending frequency
    kabs: np.ndarray               # [n_freq] optical depth per unit rho per root-cell edge
    ksca: np.ndarray
    g: np.ndarray
    bg_intensity: np.ndarray       # [n_freq]
    ps_pos: np.ndarray             # [n_point, 3] root-grid units
    ps_lum: np.ndarray             # [n_freq, n_point]
    n_packages: int
    seed: int = 1
    n_iter: int = 1
    # temperature update (None when the config has none)
    t_scale: float | None = None
    table_T: np.ndarray | None = None
    e_min: float = 0.0
    e_max: float = 0.0
    notes: dict = field(default_factory=dict)

    @property
    def n_levels(self):
        return len(self.n_cells)

    @property
    def n_total(self):
        return int(np.sum(self.n_cells))

    @property
    def n_freq(self):
        return len(self.freq_hz)

    @property
    def n_point(self):
        return len(self.ps_pos)

    def sources(self, ifreq):
        d = dict(bg_intensity=float(self.bg_intensity[ifreq]), n_bg=-1)
        if self.n_point:
            d["ps_pos"] = self.ps_pos
            d["ps_lum"] = np.ascontiguousarray(self.ps_lum[ifreq])
        return d


def _single_freq(name, n, rho3d, tau_kind, tau, albedo, g, n_packages, seed=1):
    if tau_kind == "centre_to_edge":
        kext = tau / (0.5 * n)
    else:
        kext = tau / max_column(rho3d)
    z = np.zeros((0, 3))
    return Problem(name, n, n, n, np.array([n ** 3], dtype=np.int64), rho3d.astype(np.float32).ravel(), None,
                   np.array([C_LIGHT / (LAMBDA_V_UM * 1e-4)]), np.array([(1 - albedo) * kext]),
                   np.array([albedo * kext]), np.array([float(g)]), np.array([1.0]), z, np.zeros((1, 0)),
                   int(n_packages), seed)


def _spectral(name, root_n, n_cells, rho, child, kext_v, lam_um, ps_pos, n_packages, n_iter, box_pc=10.0,
              n_table=2048, seed=1):
    nu = C_LIGHT / (lam_um * 1e-4)
    q_abs, q_sca, g = dust_model(lam_um)
    gl_cm = box_pc * PARSEC / root_n
    ps_lum = np.zeros((len(nu), len(ps_pos)))
    for k in range(len(ps_pos)):
        ps_lum[:, k] = point_source_lnu(nu) / gl_cm ** 2      # same energy unit as pi I S (S in root-cell^2)
    table_T, e_min, e_max = temperature_table(nu, SIGMA_EXT_V * q_abs, n_table)
    return Problem(name, root_n, root_n, root_n, np.asarray(n_cells, dtype=np.int64), rho, child, nu,
                   kext_v * q_abs, kext_v * q_sca, g, background_intensity(nu), np.asarray(ps_pos, dtype=np.float64),
                   ps_lum, int(n_packages), seed, n_iter, SIGMA_EXT_V / kext_v, table_T, e_min, e_max,
                   notes=dict(gl_cm=gl_cm, lam_um=lam_um))


def _densest_cell_centres(rho3d, k, pool=None, rng=None):
    n = rho3d.shape[0]
    flat = rho3d.ravel()
    if pool is None:
        idx = np.argsort(flat)[::-1][:k]
    else:
        cand = np.argsort(flat)[::-1][:pool]
        idx = rng.choice(cand, size=k, replace=False)
    iz, iy, ix = np.unravel_index(idx, (n, n, n))
    return np.stack([ix + 0.5, iy + 0.5, iz + 0.5], axis=1)


def make_config(which, n=None, n_packages=None, n_freq=None):
    """Config '1','2','3','4','4p','5' of BASELINE.json.  n / n_packages / n_freq shrink it for tests
    (same recipe, smaller lattice); None = the size as written."""
    which = str(which)
    if which == "1":
        n = n or 32
        return _single_freq("config1", n, np.ones((n, n, n)), "centre_to_edge", 1.0, 0.5, 0.0,
                            n_packages or 100_000)
    if which == "2":
        n = n or 64
        rho = lognormal_cloud(n, 1.0, 1002)
        return _single_freq("config2", n, rho, "peak", 10.0, 0.6, 0.6, n_packages or 1_000_000)
    if which == "3":
        n = n or 128
        rho = lognormal_cloud(n, 1.2, 1003)
        lam = wavelength_grid_um(0.1, 1000.0, n_freq or 64)
        return _spectral("config3", n, [n ** 3], rho.astype(np.float32).ravel(), None, 30.0 / max_column(rho), lam,
                         _densest_cell_centres(rho, 2), n_packages or 4_000_000, 1)
    if which in ("4", "4p"):
        root = n or 64
        n_levels = 4
        fine = lognormal_cloud(root * 2 ** (n_levels - 1), 1.5, 1004)
        theta = 4.0 if which == "4" else 2.0
        n_cells, rho, child = build_octree(fine, root, n_levels, theta)
        lam = wavelength_grid_um(0.1, 1000.0, n_freq or 32)
        # peak tau_V is not stated for config 4: use the config-3 value on the root-resolution cloud
        kext_v = 30.0 / (max_column(fine) / 2 ** (n_levels - 1))
        return _spectral("config" + which, root, n_cells, rho, child, kext_v, lam, np.zeros((0, 3)),
                         n_packages or 1_000_000, 1)
    if which == "5":
        n = n or 256
        rho = lognormal_cloud(n, 1.5, 1005)
        lam = wavelength_grid_um(0.1, 3000.0, n_freq or 128)
        pos = _densest_cell_centres(rho, 10, pool=1000, rng=np.random.default_rng(5))
        return _spectral("config5", n, [n ** 3], rho.astype(np.float32).ravel(), None, 100.0 / max_column(rho), lam,
                         pos, n_packages or 10_000_000, 3)
    raise ValueError(f"unknown config {which!r}")
