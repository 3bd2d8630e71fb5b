"""Pins of the oracle's fluid update (S6) against textbook LBM facts.
P:L117-119 (D2Q9, viscosity set by tau), P:L127 (TRT); pin table SURVEY.md 8(c).3.
"""
import math

import numpy as np
import pytest

from oracle import mco

RNG = np.random.default_rng(777)
W = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)
CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])
CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])


def feq(rho, ux, uy):
    out = np.empty((9,) + rho.shape)
    for q in range(9):
        cu = CX[q] * ux + CY[q] * uy
        out[q] = W[q] * rho * (1 + 3 * cu + 4.5 * cu * cu - 1.5 * (ux * ux + uy * uy))
    return out


def test_lattice_constants():
    # nu_lat = nu dt = (tau+ - 1/2)/3 ; Lambda = (tau+ - 1/2)(tau- - 1/2)
    op, om = mco.lattice_constants(10.0, 1e-2, 0.25)
    assert 1 / op == pytest.approx(0.8, abs=1e-15)
    assert (1 / op - 0.5) * (1 / om - 0.5) == pytest.approx(0.25, abs=1e-15)
    assert 1 / om == pytest.approx(4 / 3, abs=1e-15)
    op, om = mco.lattice_constants(2.0, 0.05, 3 / 16)
    assert (1 / op - 0.5) / 3 == pytest.approx(0.1, abs=1e-15)
    assert (1 / op - 0.5) * (1 / om - 0.5) == pytest.approx(3 / 16, abs=1e-15)


def test_rest_stays_at_rest():
    # BASELINE north_star: "zero forcing keeps the fluid at rest"
    ny, nx = 12, 20
    f0 = feq(np.full((ny, nx), 1.3), np.zeros((ny, nx)), np.zeros((ny, nx)))
    f = f0
    for _ in range(5):
        f, u = mco.lbm_step(f, None, 1 / 0.8, 0.75)
    assert np.abs(f - f0).max() < 1e-15 and np.abs(u).max() < 1e-16


def test_uniform_flow_is_a_fixed_point():
    ny, nx = 8, 8
    ux, uy = 0.05, -0.03
    f0 = feq(np.ones((ny, nx)), np.full((ny, nx), ux), np.full((ny, nx), uy))
    f, u = mco.lbm_step(f0, np.zeros((2, ny, nx)), 1.1, 0.9)
    assert np.abs(f - f0).max() < 1e-15
    assert np.allclose(u[0], ux, atol=1e-15) and np.allclose(u[1], uy, atol=1e-15)


def test_mass_conserved_momentum_grows_by_total_force():
    ny, nx = 16, 24
    rho = 1 + 0.02 * RNG.normal(size=(ny, nx))
    f = feq(rho, 0.02 * RNG.normal(size=(ny, nx)), 0.02 * RNG.normal(size=(ny, nx)))
    f += 1e-3 * RNG.normal(size=f.shape)          # off-equilibrium part too
    G = 1e-3 * RNG.normal(size=(2, ny, nx))
    f2, u = mco.lbm_step(f, G, 1 / 0.8, 0.75)
    assert f2.sum() == pytest.approx(f.sum(), abs=1e-12)
    px = lambda a: np.tensordot(CX, a, 1).sum()
    py = lambda a: np.tensordot(CY, a, 1).sum()
    assert px(f2) - px(f) == pytest.approx(G[0].sum(), abs=1e-13)
    assert py(f2) - py(f) == pytest.approx(G[1].sum(), abs=1e-13)
    # stored u is the Guo velocity (sum c f + G/2)/rho of the PRE-collision state
    r = f.sum(axis=0)
    assert np.allclose(u[0], (np.tensordot(CX, f, 1) + 0.5 * G[0]) / r, atol=1e-15)
    assert np.allclose(u[1], (np.tensordot(CY, f, 1) + 0.5 * G[1]) / r, atol=1e-15)


def test_streaming_direction():
    # a single perturbed population moves by exactly c_q per step (f_q(x+c_q,n+1)=f*_q(x,n)).
    # With omega+ = omega- = 1... collision would erase it; instead use the conserved
    # moments: a density blob advected by its own momentum is hard to read, so test the
    # operator directly with omega = 0 (no relaxation): pure streaming.
    ny, nx = 6, 7
    for q in range(9):
        f = np.zeros((9, ny, nx)) + W[:, None, None]
        f[q, 2, 3] += 0.1
        f2, _ = mco.lbm_step(f, None, 0.0, 0.0)
        j, i = (2 + CY[q]) % ny, (3 + CX[q]) % nx
        d = f2 - W[:, None, None]
        assert d[q, j, i] == pytest.approx(0.1, abs=1e-16)
        d[q, j, i] = 0
        assert np.abs(d).max() < 1e-16
    # periodic wrap of the stream
    f = np.zeros((9, ny, nx)) + W[:, None, None]
    f[5, ny - 1, nx - 1] += 0.2
    f2, _ = mco.lbm_step(f, None, 0.0, 0.0)
    assert f2[5, 0, 0] - W[5] == pytest.approx(0.2, abs=1e-16)


def test_uniform_body_force():
    # uniform G=(g,0): u stays uniform and the stored velocity at step t is g (t + 1/2)/rho0
    ny, nx, g = 8, 8, 1e-4
    f = feq(np.ones((ny, nx)), np.zeros((ny, nx)), np.zeros((ny, nx)))
    G = np.zeros((2, ny, nx))
    G[0] = g
    for t in range(10):
        f, u = mco.lbm_step(f, G, 1 / 0.8, 0.75)
        assert np.allclose(u[0], g * (t + 0.5), rtol=0, atol=1e-17 + 1e-12 * g * (t + 1))
        assert np.abs(u[1]).max() < 1e-18
    assert np.tensordot(CX, f, 1).mean() == pytest.approx(10 * g, rel=1e-12)


@pytest.mark.parametrize("nu_lat,tol", [(0.1, 3e-3), (0.02, 3e-2)])
def test_shear_wave_decays_with_the_viscosity_tau_sets(nu_lat, tol):
    # P:L119 "viscosity is controlled by a single relaxation parameter tau":
    # u_x = U sin(2 pi y/ny) decays as exp(-nu k^2 t), nu = (tau+ - 1/2)/3.
    # Discrete LBM adds an O(k^4) hyper-viscous term (absolute, so relatively larger at
    # small nu): ny = 64 keeps it below 0.3 % at nu = 0.1 and 3 % at nu = 0.02.
    ny, nx, U, T = 64, 4, 1e-3, 200
    op, om = mco.lattice_constants(nu_lat, 1.0, 0.25)
    y = np.arange(ny)[:, None] * np.ones((1, nx))
    k = 2 * math.pi / ny
    f = feq(np.ones((ny, nx)), U * np.sin(k * y), np.zeros((ny, nx)))
    for t in range(T):
        f, u = mco.lbm_step(f, None, op, om)
        if t == 0:
            a0 = 2 * (u[0] * np.sin(k * y)).mean()
    a1 = 2 * (u[0] * np.sin(k * y)).mean()
    rate = -math.log(a1 / a0) / (T - 1)
    assert rate == pytest.approx(nu_lat * k * k, rel=tol)
    assert np.abs(u[1]).max() < 1e-12
    # shear decay is governed by omega+, not omega-: changing Lambda leaves the rate
    op2, om2 = mco.lattice_constants(nu_lat, 1.0, 3 / 16)
    assert op2 == op and om2 != om
