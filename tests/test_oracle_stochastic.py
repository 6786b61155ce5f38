"""Pins for the oracle of the stochastic-heating solver (row f4; Appendix A) and for the synthetic grain
model that stands in for the DustEM tables: structure of the rate matrix as the paper states it, closed forms, balance
identities that hold for the exact solution however it is computed, and energy conservation of the model."""
import math

import numpy as np
import pytest

import oracle
from paper_1812_06632_b200 import inputs

NU = inputs.C_LIGHT / (inputs.wavelength_grid_um(0.1, 3000.0, 128) * 1e-4)
W_NU = inputs.trapz_weights(NU)
ISRF = inputs.background_intensity(NU)


def _dense_W(model, s):
    n_s, n_e, n_f = model["jup"].shape
    W = np.zeros((n_e, n_e, n_f))
    i, f = np.nonzero(model["jup"][s] >= 0)
    W[model["jup"][s][i, f], i, f] = model["wup"][s][i, f]
    return W


@pytest.fixture(scope="module")
def model():
    return inputs.stochastic_model(NU, n_size=6, n_e=48)


def test_rate_matrix_has_the_structure_the_paper_states(model):
    for s in (0, 5):
        R = oracle.stochastic_rate_matrix(_dense_W(model, s), model["cool"][s], 30.0 * ISRF)
        n = len(R)
        assert np.allclose(R.sum(axis=0), 0.0, atol=1e-12 * np.abs(R).max())          # detailed balance: columns sum to 0
        assert (np.triu(R, 2) == 0).all()                                             # R_ji = 0 for i > j + 1
        assert np.array_equal(np.diag(R, 1), model["cool"][s][1:]) and (np.diag(R, 1) > 0).all()
        assert (np.tril(R, -1) >= 0).all() and (np.diag(R)[:-1] < 0).all()
        # upward rates are linear in the intensity ("vector product of the intensity with the integration weights")
        R2 = oracle.stochastic_rate_matrix(_dense_W(model, s), model["cool"][s], 60.0 * ISRF)
        assert np.allclose(np.tril(R2, -1), 2 * np.tril(R, -1), rtol=1e-14)


def test_two_level_closed_form():
    W = np.zeros((2, 2, 3)); W[1, 0] = [0.5, 0.25, 2.0]
    R = oracle.stochastic_rate_matrix(W, np.array([0.0, 7.0]), np.array([2.0, 4.0, 1.0]))
    up = 0.5 * 2 + 0.25 * 4 + 2.0 * 1
    assert np.allclose(R, [[-up, 7.0], [up, -7.0]])
    p = oracle.stochastic_solve(R)
    assert p[1] / p[0] == pytest.approx(up / 7.0, rel=1e-14) and p.sum() == pytest.approx(1.0, rel=1e-15)


@pytest.mark.parametrize("scale", [1.0, 1e3, 1e6])
def test_solution_satisfies_the_balance_identities(model, scale):
    """For the exact solution, however obtained: R p = 0, sum p = 1, p >= 0, and the probability flux across every bin
    boundary balances -- sum_{i<j} p_i sum_{k>=j} R_ki = p_j R_(j-1,j) -- which is the forward substitution of the paper's
    explicit solver read as an identity."""
    for s in (0, 3, 5):
        R = oracle.stochastic_rate_matrix(_dense_W(model, s), model["cool"][s], scale * ISRF)
        p = oracle.stochastic_solve(R)
        assert p.sum() == pytest.approx(1.0, rel=1e-13) and p.min() > -1e-14
        assert np.abs(R @ p).max() <= 1e-10 * np.abs(np.diag(R) * p).max()
        n = len(p)
        for j in range(1, n):
            up = sum(p[i] * R[j:, i].sum() for i in range(j))
            down = p[j] * R[j - 1, j]
            if max(up, down) > 1e-12 * np.abs(np.diag(R) * p).max():
                assert up == pytest.approx(down, rel=1e-6)


def test_model_conserves_energy_and_has_the_right_limits(model):
    """The synthetic grain model: what a grain radiates equals what it absorbs (to the enthalpy discretisation); large
    grains in a strong field sit at the equilibrium temperature; the smallest grains in the weak field spend their time far
    below it (that is what "stochastically heated" means)."""
    for scale in (1.0, 1e3, 1e6):
        p, em = oracle.stochastic_cells(model, np.stack([scale * ISRF]))
        for s in range(6):
            a = model["a_cm"][s]
            c_abs = np.pi * a ** 2 * np.minimum(1.0, 2 * np.pi * a / (inputs.C_LIGHT / NU))
            absorbed = float((W_NU * 4 * np.pi * c_abs * scale * ISRF).sum())
            emitted = float((W_NU * (p[0, s][:, None] * model["emis"][s]).sum(axis=0)).sum())
            assert emitted == pytest.approx(absorbed, rel=0.08)
            power = np.array([4 * np.pi * float((W_NU * c_abs * inputs.planck_nu(NU, t)).sum()) for t in model["T"]])
            t_eq = float(np.interp(math.log(absorbed), np.log(power), model["T"]))
            t_mean = float((p[0, s] * model["T"]).sum())
            if s == 5 and scale >= 1e3:
                assert t_mean == pytest.approx(t_eq, rel=0.08)
            if s == 0 and scale == 1.0:
                assert t_mean < 0.4 * t_eq
        assert np.allclose(em[0], oracle.stochastic_emission(p[0], model["emis"], model["abundance"]), rtol=1e-14)
    # the emission is a sum over sizes weighted by the abundances
    p, em = oracle.stochastic_cells(model, np.stack([ISRF]))
    by_hand = sum(model["abundance"][s] * p[0, s] @ model["emis"][s] for s in range(6))
    assert np.allclose(em[0], by_hand, rtol=1e-13)
