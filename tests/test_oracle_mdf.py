"""Pins of the oracle's Multi-Direct Forcing coupling (
DESIGN.md reading 26): mco_moments, mco_mdf and the MDF branch of the step.

None of these re-types the oracle's loop: they use closed forms (Peskin's sum-of-squares
identity sum_j phi(r - j)^2 = 3/8, which makes the one-bead residual a geometric series), a
dense linear solve of the no-slip condition, and conservation laws.
"""
import numpy as np
import pytest

from oracle import mco
from paper_2607_02954_b200 import worlds

CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])
CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])
WQ = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)
S2 = (3.0 / 8.0) ** 2  # sum over the 4x4 support of delta_h^2 (Peskin 2002: sum phi^2 = 3/8)


def test_peskin_sum_of_squares_identity():
    # the closed form the residual pins rest on, checked on the pinned phi itself
    for r in np.linspace(-0.5, 0.5, 41):
        s = sum(mco.phi(r - j) ** 2 for j in range(-3, 4))
        assert abs(s - 0.375) < 1e-14


def test_moments_of_an_equilibrium():
    # second-order equilibrium at (rho, u): sum f = rho, sum c f = rho u (textbook D2Q9)
    rng = np.random.default_rng(0)
    ny, nx = 5, 7
    rho = 1.0 + 0.05 * rng.standard_normal((ny, nx))
    u = 0.05 * rng.standard_normal((2, ny, nx))
    cu = CX[:, None, None] * u[0] + CY[:, None, None] * u[1]
    f = WQ[:, None, None] * rho * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * (u[0] ** 2 + u[1] ** 2))
    r, us = mco.moments(f)
    assert np.allclose(r, rho, rtol=0, atol=1e-15)
    assert np.allclose(us, u, rtol=0, atol=1e-15)


@pytest.mark.parametrize("rho_f,rho0", [(1.0, 1.0), (1.1, 1.0), (0.9, 1.3)])
def test_single_bead_residual_is_a_geometric_series(rho_f, rho0):
    # One bead in a uniform fluid at rest: U^k = (1 - q^k) V with q = 1 - (rho0/(2 rho)) (3/8)^2,
    # wherever the bead sits; F = rho0 V (1 + q + ... + q^(K-1)).  Catches a wrong factor, a
    # sign, replace-instead-of-accumulate, rho vs rho0, and a wrong kernel.
    nx, ny, K = 16, 12, 6
    V = np.array([[3e-3, -2e-3]])
    q = 1.0 - 0.5 * (rho0 / rho_f) * S2
    for xy in ([[5.0, 6.0]], [[5.37, 6.81]], [[15.9, 0.2]]):  # on a node, generic, across the seam
        r = mco.mdf(xy, V, np.zeros((2, ny, nx)), np.full((ny, nx), rho_f), rho0, K)
        geo = sum(q ** j for j in range(K))
        assert np.allclose(r["F"], rho0 * V * geo, rtol=1e-13, atol=0)
        assert np.allclose(r["resid"], np.abs(V).max() * q ** np.arange(K + 1), rtol=1e-12, atol=0)
        U = mco.interp(r["u"], xy)
        assert np.allclose(U, (1 - q ** K) * V, rtol=1e-12, atol=0)


def test_bead_moving_with_the_fluid_feels_no_force():
    # uniform flow u0 and V = u0: nothing to correct (interpolation reproduces constants)
    nx, ny = 16, 16
    us = np.empty((2, ny, nx)); us[0] = 0.01; us[1] = -0.02
    xy = 16 * worlds.uniform(3, "mdf-x", 10).reshape(5, 2)
    V = np.tile([0.01, -0.02], (5, 1))
    r = mco.mdf(xy, V, us, np.ones((ny, nx)), 1.0, 3)
    assert np.abs(r["F"]).max() < 1e-16 and np.abs(r["G"]).max() < 1e-16
    assert np.allclose(r["u"], us, rtol=0, atol=1e-17)


def _gram(xy, nx, ny):
    # M_ij = sum_g delta_h(g - X_i) delta_h(g - X_j), from deposit/interp of unit beads
    n = len(xy)
    M = np.empty((n, n))
    for j in range(n):
        dj = mco.deposit(nx, ny, xy[j:j + 1])
        M[:, j] = mco.interp(dj[None], xy)[:, 0]
    return M


def test_converges_to_the_no_slip_solution_of_a_dense_solve():
    # fixed point: interp(ustar + spread(F)/(2 rho)) = V  <=>  M F = 2 rho (V - Ustar) for
    # uniform rho.  A short chain with unit spacing: MDF with many iterations reaches it.
    nx, ny, rho = 24, 20, 1.05
    s = np.arange(9.0)
    xy = np.stack([6.3 + s * np.cos(0.4), 7.1 + s * np.sin(0.4)], 1)
    rng = np.random.default_rng(4)
    V = 1e-2 * np.stack([np.cos(0.3 * s), 0.5 + np.sin(0.2 * s)], 1)  # smooth along the chain
    us = 1e-4 * rng.standard_normal((2, ny, nx))
    M = _gram(xy, nx, ny)
    assert np.linalg.eigvalsh(M).max() < 4  # the iteration contracts
    Fex = np.linalg.solve(M, 2 * rho * (V - mco.interp(us, xy)))
    # F^K - Fex = (I - M/2)^K (F^0 - Fex) with rho0 = rho and F^0 = 0: the exact error of the
    # iteration, from the dense matrix (M has small eigenvalues along the chain's high-frequency
    # modes, so F itself converges slowly; the velocity residual M (Fex - F)/(2 rho) does not)
    for K in (1, 3, 32):
        r = mco.mdf(xy, V, us, np.full((ny, nx), rho), rho, K)
        EK = np.linalg.matrix_power(np.eye(9) - 0.5 * M, K) @ (-Fex)
        assert np.allclose(r["F"] - Fex, EK, rtol=1e-9, atol=1e-15)
        slip = V - mco.interp(r["u"], xy)
        assert np.allclose(slip, M @ (Fex - r["F"]) / (2 * rho), rtol=1e-9, atol=1e-16)
    assert np.all(np.diff(r["resid"]) < 0)      # the slip shrinks monotonically (max-norm)
    assert r["resid"][-1] < 0.1 * r["resid"][0]


def test_grid_force_carries_the_bead_force_and_u_is_consistent():
    # sum_g G = sum_i F_i (spread conserves), and u_out = ustar + G/(2 rho) with varying rho
    nx, ny = 20, 24
    rng = np.random.default_rng(7)
    xy = np.stack([20 * worlds.uniform(1, "mdf-a", 30), 24 * worlds.uniform(1, "mdf-b", 30)], 1)
    V = 1e-2 * rng.standard_normal((30, 2))
    us = 1e-3 * rng.standard_normal((2, ny, nx))
    rho = 1 + 0.03 * rng.standard_normal((ny, nx))
    r = mco.mdf(xy, V, us, rho, 1.0, 4)
    assert np.allclose(r["G"].sum(axis=(1, 2)), r["F"].sum(axis=0), rtol=1e-12, atol=1e-18)
    assert np.allclose(r["u"], us + r["G"] / (2 * rho), rtol=0, atol=1e-17)
    # the same result from the separately pinned components, one iteration written out
    r1 = mco.mdf(xy, V, us, rho, 1.0, 1)
    F1 = 1.0 * (V - mco.interp(us, xy))
    assert np.allclose(r1["F"], F1, rtol=1e-14, atol=0)
    assert np.allclose(r1["G"], mco.spread(nx, ny, xy, F1), rtol=1e-14, atol=1e-20)


def _mdf_world(seed=11, iters=3, **kw):
    w = worlds.random_world(48, 32, 5, 12, seed=seed, **kw)
    w["params"]["coupling"] = 1
    w["params"]["mdf_iters"] = iters
    return w


def test_step_glue_mdf():
    # V = D + field displacement (kappa not used), forcing against the moments of the CURRENT
    # populations, fluid advanced with the summed G, beads advected by the stored u
    w = _mdf_world(static_source=True)
    w["xy"] += (0.05 * worlds.normal(5, "pert", w["xy"].size).reshape(-1, 2)).astype(np.float32)
    p = w["params"]
    nx, ny, dt = p["nx"], p["ny"], np.float32(p["dt"]).astype(np.float64)
    W = mco.World(w)
    W.step(2)                       # make the fluid non-trivial
    s0 = W.read_state()
    W.step(1)
    s1, it = W.read_state(), W.read_intermediates()
    X0 = s0["xy"]
    D = mco.elastic(w["offsets"], X0, w["L_rest"], w["theta_rest"], w["k_bend"], w["k_shear"],
                    w["k_stretch"], w["act_amp"], w["act_phase"], w["act_period"], dt, 2)
    assert np.array_equal(it["D"], D)
    V = D.copy()
    for k, fd in enumerate(p["fields"]):
        coup = np.float32(fd["coupling"]).astype(np.float64) * dt * dt
        if fd["kind"] == 0:
            R = mco.radius(fd["sigma"], fd["radius"])
            gx, gy = mco.grad(mco.blur(mco.deposit(nx, ny, X0), np.float32(fd["sigma"]), R))
            V -= coup * mco.interp(np.stack([gx, gy]), X0)
        else:
            gx, gy = mco.grad(mco.static_field(nx, ny, fd["sources"]))
            V += coup * mco.interp(np.stack([gx, gy]), X0)
    f = s0["fdev"] + WQ[:, None, None] * np.float32(p["rho0"]).astype(np.float64)
    rho, us = mco.moments(f)
    r = mco.mdf(X0, V, us, rho, float(np.float32(p["rho0"])), 3)
    assert np.allclose(s1["force"], r["F"], rtol=1e-12, atol=1e-18)
    assert np.allclose(it["G"], r["G"], rtol=1e-12, atol=1e-18)
    assert np.allclose(s1["u"], r["u"], rtol=1e-11, atol=1e-16)   # Guo velocity = u^K
    assert np.allclose(s1["xy"], X0 + mco.interp(s1["u"], X0), rtol=0, atol=1e-14)


def test_no_slip_improves_with_iterations():
    # after the step the beads have moved by interp(u); its distance from V shrinks as the
    # number of forcing iterations grows (what MDF is for, "leaking")
    errs = []
    for K in (1, 2, 4, 8):
        w = _mdf_world(seed=13, iters=K, kappa_rep=None)
        W = mco.World(w)
        W.step(5)
        s0 = W.read_state()
        W.step(1)
        s1, it = W.read_state(), W.read_intermediates()
        errs.append(np.abs((s1["xy"] - s0["xy"]) - it["D"]).max() / np.abs(it["D"]).max())
    assert all(b < a for a, b in zip(errs, errs[1:])), errs
    assert errs[-1] < 0.7 * errs[0]   # slow: D alternates bead to bead, below what delta_h resolves


def test_mdf_step_conserves_mass_and_momentum_budget():
    w = _mdf_world(seed=17)
    W = mco.World(w)
    mom = np.zeros(2)
    for _ in range(6):
        W.step(1)
        mom += W.read_state()["force"].sum(axis=0)
    s = W.read_state()
    assert abs(s["rho"].sum() - 48 * 32) < 1e-10
    got = np.array([np.tensordot(CX, s["fdev"], 1).sum(), np.tensordot(CY, s["fdev"], 1).sum()])
    assert np.allclose(got, mom, rtol=1e-9, atol=1e-15)


def test_mdf_parameters_are_validated():
    w = _mdf_world(iters=0)
    with pytest.raises(ValueError):
        mco.World(w)
    w = _mdf_world(iters=17)
    with pytest.raises(ValueError):
        mco.World(w)
    w = _mdf_world()
    w["params"]["coupling"] = 2
    with pytest.raises(ValueError):
        mco.World(w)


def test_relaxation_factor_of_reading_26_fits_the_configs():
    # The forcing iteration contracts while the row sums of the bead Gram matrix -- rho_b
    # interpolated at the beads -- stay below 4 with the factor rho0 taken here (below 2 with the
    # 2 rho0 that cancels an isolated bead's slip at once).  BASELINE.json config 2 has crossings
    # above 2 and below 4: the reason for the factor (reading 26).  The crowded config
    # 5 is far outside either bound: MDF is not for it.
    w = worlds.make_world("2")
    X = w["xy"].astype(np.float64)
    rows = mco.interp(mco.deposit(256, 256, X)[None], X)[:, 0]
    assert 2.0 < rows.max() < 4.0, rows.max()
    W = mco.World(dict(w, params=dict(w["params"], coupling=1, mdf_iters=3)), threads=4)
    W.step(30)
    s = W.read_state()
    assert np.abs(s["u"]).max() < 0.05 and np.abs(s["rho"] - 1).max() < 0.1
    w5 = worlds.random_world(64, 64, 96, 16, seed=7, kappa=0.25, kappa_rep=2e-4, clustered=3.0)
    X5 = w5["xy"].astype(np.float64)
    assert mco.interp(mco.deposit(64, 64, X5)[None], X5)[:, 0].max() > 8.0
