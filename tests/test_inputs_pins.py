"""Pins for the input generators that carry physics (paper_1812_06632_b200/inputs.py): the temperature table and the
source spectra feed BOTH the CUDA path and the oracle, so a wrong Lambda(T) would be invisible to parity.  They are
pinned here against closed forms (pin P11; PAPER.md:67 energy balance of equilibrium grains).
"""
import math

import numpy as np
import pytest
from scipy import special

import oracle
from paper_1812_06632_b200 import inputs

H, K, C = inputs.H_PLANCK, inputs.K_BOLTZ, inputs.C_LIGHT


def _power_law(beta, n=6000):
    nu = np.geomspace(1e7, 1e17, n)
    nu0, k0 = 1e12, 3e-25
    return nu, k0 * (nu / nu0) ** beta, nu0, k0


def _lambda_closed(T, beta, nu0, k0):
    """4 pi k0 nu0^-beta (2h/c^2) (kT/h)^(4+beta) Gamma(4+beta) zeta(4+beta)."""
    return 4 * math.pi * k0 * nu0 ** -beta * (2 * H / C ** 2) * (K * T / H) ** (4 + beta) * special.gamma(4 + beta) * special.zeta(4 + beta)


def test_planck_integrates_to_stefan_boltzmann():
    nu = np.geomspace(1e7, 1e17, 6000)
    for T in (2.73, 20.0, 1e4):
        total = float((inputs.trapz_weights(nu) * inputs.planck_nu(nu, T)).sum())
        assert total == pytest.approx(inputs.SIGMA_SB * T ** 4 / math.pi, rel=1e-5)
    # Wien and Rayleigh-Jeans limits
    assert inputs.planck_nu(1e9, 100.0) == pytest.approx(2 * 1e18 * K * 100.0 / C ** 2, rel=1e-3)
    x = H * 1e15 / (K * 300.0)
    assert inputs.planck_nu(1e15, 300.0) == pytest.approx(2 * H * 1e45 / C ** 2 * math.exp(-x), rel=1e-12)


def test_point_source_spectrum_integrates_to_its_luminosity():
    nu = np.geomspace(1e10, 1e17, 5000)
    L = float((inputs.trapz_weights(nu) * inputs.point_source_lnu(nu)).sum())
    assert L == pytest.approx(100.0 * inputs.L_SUN, rel=1e-5)


def test_trapz_weights_match_the_oracle_quadrature():
    nu = np.geomspace(3e11, 3e15, 17)
    assert np.allclose(inputs.trapz_weights(nu), oracle.trapezoid_weights(nu), rtol=1e-14)
    assert inputs.trapz_weights(nu).sum() == pytest.approx(nu[-1] - nu[0], rel=1e-14)
    assert inputs.trapz_weights(nu[::-1].copy()).sum() == pytest.approx(nu[-1] - nu[0], rel=1e-14)   # descending grid


@pytest.mark.parametrize("beta", [0.0, 1.0, 1.7, 2.0])
def test_emissivity_is_the_closed_form_for_power_law_dust(beta):
    """P11: kappa_abs ~ nu^beta on a wide fine grid => Lambda(T) = 4 pi k0 nu0^-beta (2h/c^2)(kT/h)^(4+beta) Gamma zeta."""
    nu, sig, nu0, k0 = _power_law(beta)
    T = np.array([5.0, 20.0, 100.0, 700.0])
    lam = inputs.emissivity_per_h(nu, sig, T)
    assert np.allclose(lam, _lambda_closed(T, beta, nu0, k0), rtol=2e-5)
    # a dropped 4 pi, a wrong weight or a transposed (T, nu) broadcast would fail the line above; the slope too
    assert np.allclose(np.diff(np.log(lam)) / np.diff(np.log(T)), 4 + beta, rtol=1e-4)


@pytest.mark.parametrize("beta", [1.0, 2.0])
def test_temperature_table_round_trip_and_power_law(beta):
    """P11: T(E) is the pure power law (E / prefactor)^(1/(4+beta)); Lambda(T_k) = E_k to interpolation error."""
    nu, sig, nu0, k0 = _power_law(beta)
    table, e_min, e_max = inputs.temperature_table(nu, sig, n_table=2048)
    assert table.dtype == np.float32 and len(table) == 2048
    E = np.exp(np.linspace(math.log(e_min), math.log(e_max), 2048))
    pref = _lambda_closed(1.0, beta, nu0, k0)
    assert np.allclose(table, (E / pref) ** (1 / (4 + beta)), rtol=1e-5)
    assert table[0] == pytest.approx(3.0, rel=1e-6) and table[-1] == pytest.approx(1500.0, rel=1e-6)
    assert (np.diff(table) > 0).all()
    back = inputs.emissivity_per_h(nu, sig, table.astype(np.float64))
    assert np.allclose(back, E, rtol=1e-5 * (4 + beta) + 1e-6)
    # and through the oracle's lookup: a leaf that absorbed E per unit dust sits at T(E) (interpolation error ~ 6e-6)
    g = oracle.Grid(4, 1, 1, [4], np.ones(4, dtype=np.float32))
    Ec = np.array([e_min * 3.3, math.sqrt(e_min * e_max), e_max / 7.7, e_max * 2])
    T = oracle.update_temperatures(g, Ec, 1.0, table, e_min, e_max)
    expect = (np.minimum(Ec, e_max) / pref) ** (1 / (4 + beta))
    assert np.allclose(T, expect, rtol=2e-5)


def test_config_tables_invert_their_own_emissivity():
    """The table of the spectral configs (broken power-law dust, 12 frequencies here): Lambda(T_k) = E_k with the
    config's own quadrature weights -- the balance the oracle and the kernel look up is exact in the discretised sense
    (SURVEY.md 8c.9)."""
    P = inputs.make_config("3", n=8, n_packages=10, n_freq=12)
    q_abs = P.kabs * P.t_scale                                         # kabs = kext_v q_abs, t_scale = sigma_V / kext_v
    E = np.exp(np.linspace(math.log(P.e_min), math.log(P.e_max), len(P.table_T)))
    back = inputs.emissivity_per_h(P.freq_hz, q_abs, P.table_T.astype(np.float64))
    assert np.allclose(back, E, rtol=2e-4)
